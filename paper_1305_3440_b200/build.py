"""Build libgf_b200.so (hand-written CUDA for sm_100a + the C ABI of include/gf.h) in-tree.

    python paper_1305_3440_b200/build.py [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so lands next to this file so that it travels to the
GPU box with the source snapshot.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libgf_b200.so")
SOURCES = ["gf_sweep.cu", "gf_aux.cu", "gf_api.cu", "gf_static.cu"]
HEADERS = [os.path.join(CSRC, "gf_device.cuh"), os.path.join(CSRC, "gf_internal.h"),
           os.path.join(INCLUDE, "gf.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]
# kernel-variant experiments (e.g. GF_EXTRA_NVCC_FLAGS="-DGF_LAZY12_F64=22"; see profiles/): rebuild with --force
NVCC_FLAGS += os.environ.get("GF_EXTRA_NVCC_FLAGS", "").split()


def source_hash() -> str:
    """sha256 over the CODE of the kernel sources and headers (comments and white space removed): ties a profile under
    profiles/ to the code it was taken at; rewording a comment does not invalidate a capture."""
    import hashlib
    import re
    h = hashlib.sha256()
    for f in [os.path.join(CSRC, s) for s in SOURCES] + HEADERS:
        text = open(f, encoding="utf-8").read()
        text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)          # block comments
        text = re.sub(r"//[^\n]*", " ", text)                       # line comments (no string literal here holds "//")
        h.update(os.path.basename(f).encode())
        h.update(" ".join(text.split()).encode())
    return h.hexdigest()[:16]


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    objs = []
    jobs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(CSRC, src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + HEADERS):
            cmd = [NVCC, *NVCC_FLAGS, "-c", s, "-o", o]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            jobs.append(cmd)

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n%s\n%s" % (" ".join(cmd), r.stderr))
        return r.stderr

    if jobs:
        with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
            for log in ex.map(run, jobs):
                if verbose and log:
                    print(log)
    if jobs or force or _stale(LIB, objs):
        run([NVCC, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
