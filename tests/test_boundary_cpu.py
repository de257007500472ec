"""CPU-only checks of the C-ABI boundary: the library loads, exports every symbol include/gf.h
declares, and its host-side argument logic answers without a GPU."""
import ctypes
import os
import re

import paper_1305_3440_b200 as gf
from paper_1305_3440_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "gf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gf_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = declared_symbols()
    assert len(names) >= 20
    lib = ctypes.CDLL(gf.lib_path)
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names            # the binding covers the whole header


def test_storage_and_workspace_bytes():
    d = (32, 32, 32, 32)
    V = 32 ** 4
    assert gf.gf_storage_bytes(d, gf.GF_F64, gf.GF_RECON18) == V * 4 * 18 * 8      # 604 MB
    assert gf.gf_storage_bytes(d, gf.GF_F32, gf.GF_RECON12) == V * 4 * 12 * 4
    assert gf.gf_storage_bytes(d, gf.GF_MIXED, gf.GF_RECON18) == 0
    assert gf.gf_storage_bytes(d, gf.GF_F64, 10) == 0
    assert gf.gf_storage_bytes((32, 31, 32, 32), gf.GF_F64, 18) == 0                # odd extent
    assert gf.gf_storage_bytes((0, 4, 4, 4), gf.GF_F64, 18) == 0
    assert gf.gf_workspace_bytes(d) > 0 and gf.gf_workspace_bytes(d) % 8 == 0
    assert gf.gf_workspace_bytes((4, 4, 4, 3)) == 0
    # 64^4 fits the 32-bit site index the kernels use; 2^32 sites do not
    assert gf.gf_storage_bytes((64, 64, 64, 64), gf.GF_F64, 18) == 64 ** 4 * 4 * 18 * 8
    assert gf.gf_storage_bytes((256, 256, 256, 256), gf.GF_F64, 18) == 0


def test_argument_errors_are_reported_before_any_device_work():
    # all of these fail in the host-side checks, so they answer GF_EINVAL even without a GPU
    bad = gf.gf_init_lattice((4, 4, 4, 5), gf.GF_LANDAU, 18, 16, 0, 16, 0, 0, check=False)
    assert bad == gf.GF_EINVAL
    assert gf.gf_init_lattice((4, 4, 4, 4), 7, 18, 16, 0, 16, 0, 0, check=False) == gf.GF_EINVAL
    assert gf.gf_init_lattice((4, 4, 4, 4), gf.GF_LANDAU, 9, 16, 0, 16, 0, 0, check=False) == gf.GF_EINVAL
    assert gf.gf_init_lattice((4, 4, 4, 4), gf.GF_LANDAU, 18, 0, 0, 16, 0, 0, check=False) == gf.GF_EINVAL
    assert gf.gf_init_lattice((4, 4, 4, 4), gf.GF_LANDAU, 18, 24, 0, 16, 0, 0, check=False) == gf.GF_EINVAL  # alignment
    assert gf.gf_init_lattice((4, 4, 4, 4), gf.GF_LANDAU, 18, 16, 0, 0, 0, 0, check=False) == gf.GF_EINVAL   # workspace
    # null context
    assert binding.lib.gf_sweep(None, 0, 0, 1.0, 0.0, gf.GF_F64) == gf.GF_EINVAL
    assert binding.lib.gf_fix_until(None, 0, 1.0, 0.0, gf.GF_F64, 1e-12, 1, 1, None, None) == gf.GF_EINVAL
    assert gf.gf_last_error(None) == "null context"
    gf.gf_destroy(None)


def test_header_is_plain_c_and_a_c_program_links_against_the_library(tmp_path):
    """include/gf.h is a C header (no C++, no torch types): it compiles as strict C99, and a C program that calls
    the host-side entry points links against libgf_b200.so and gets the documented answers without a GPU."""
    import subprocess
    src = tmp_path / "use_gf.c"
    src.write_text(
        '#include <stdio.h>\n#include "gf.h"\n'
        "int main(void) {\n"
        "    const int dims[4] = {32, 32, 32, 32}, odd[4] = {4, 4, 4, 5};\n"
        "    gf_ctx* ctx = (gf_ctx*)0;\n"
        '    printf("%zu %zu %d %d\\n", gf_storage_bytes(dims, GF_F64, GF_RECON18), gf_storage_bytes(odd, GF_F64, GF_RECON18),\n'
        "           gf_init_lattice(&ctx, odd, GF_LANDAU, GF_RECON18, (void*)16, (void*)0, (void*)16, (void*)0, 0),\n"
        "           gf_sweep((gf_ctx*)0, 0, GF_OVERRELAX, 1.7, 0.0, GF_F64));\n"
        "    return ctx != (gf_ctx*)0;\n}\n")
    exe = tmp_path / "use_gf"
    libdir = os.path.dirname(gf.lib_path)
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(ROOT, "include"), str(src),
                    "-o", str(exe), "-L", libdir, "-l:libgf_b200.so", "-Wl,-rpath," + libdir], check=True, capture_output=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()
    assert out == [str(32 ** 4 * 4 * 18 * 8), "0", str(gf.GF_EINVAL), str(gf.GF_EINVAL)]
