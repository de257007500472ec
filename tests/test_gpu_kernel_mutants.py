"""Mutation run of the GPU parity tests (opt-in: GF_KERNEL_MUTANTS=1 python -m pytest tests/test_gpu_kernel_mutants.py -m gpu -s).

The counterpart of tests/test_oracle_mutants.py for the CUDA side: every plausible single-line mistake in the kernels
must make the GPU parity tests fail.  For each mutant a private copy of the package, include/, oracle/, gf_inputs.py
and the GPU test files is made in a temporary directory, ONE source line of csrc/ is replaced, the library is rebuilt
THERE (nvcc, only the translation units that changed) and a subset of the parity tests is run against it with
``pytest -x``; the run must fail.  The unmutated copy must pass (control).  All mutants keep every memory access inside
the buffers (arithmetic, signs, which draw / which neighbour inside the lattice), so a mutant cannot fault the GPU.
Off by default because it rebuilds the library a dozen times (about five minutes on the GPU box); the outcome of a run
is recorded in profiles/r3_kernel_mutants.md.  What needs no rebuild is checked on every run, without a GPU: every
fragment of the list occurs exactly once in the current sources (a list that has gone stale fails at once).
"""
import os
import shutil
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PKG = "paper_1305_3440_b200"
TEST_FILES = ["conftest.py", "test_gpu_parity.py", "test_gpu_checkers.py", "test_gpu_coulomb.py", "test_gpu_transform.py",
              "test_gpu_fix_runahead.py", "curand_philox_ref.cu", "gpu_helpers.py"]
# the subset that is run against every mutant (the whole of these files takes about a minute)
SELECT = ("pack_unpack or unit_links or one_sweep or ten_sweeps or stochastic_counter or philox or config1_fix or random_small or "
          "extreme or unitarity_matches or reunitarize or cast_f32 or deferred_temporal_links_one or slice_mask or "
          "accumulated_transformation or apply_transform or transformation_reproduces or mixed_exact or runahead_equals or "
          "runahead_coulomb or hands_over or reprojection_keeps")

# (name, file under csrc/, exact fragment (must occur exactly once), replacement)
MUTANTS = [
    ("v1 sign", "gf_device.cuh", "T v1 = -(GF_IM(K, I, J) + GF_IM(K, J, I));", "T v1 = (GF_IM(K, I, J) + GF_IM(K, J, I));"),
    ("v3 from the wrong difference", "gf_device.cuh", "T v3 = GF_IM(K, J, J) - GF_IM(K, I, I);", "T v3 = GF_IM(K, I, I) - GF_IM(K, J, J);"),
    ("overrelaxation without |v|", "gf_device.cuh", "v0 = omega * v0 + (T(1) - omega) * n;", "v0 = omega * v0 + (T(1) - omega);"),
    ("a^2: scalar part", "gf_device.cuh", "a[0] = t * a[0] - T(1);", "a[0] = t * a[0];"),
    ("K update: E_JI sign", "gf_device.cuh", "GF_RE(K, J, b) = -a[2] * ir - a[1] * ii + a[0] * jr + a[3] * ji;",
     "GF_RE(K, J, b) = a[2] * ir - a[1] * ii + a[0] * jr + a[3] * ji;"),
    ("g = E3 E2 E1: a sign in E2", "gf_device.cuh", "Rr = -b[2], Ri = b[1], Sr = b[0], Si = -b[3];", "Rr = b[2], Ri = b[1], Sr = b[0], Si = -b[3];"),
    ("U g instead of U g^dagger (one term)", "gf_device.cuh", "im = gf_fma(-GF_RE(U, a, 0), GF_IM(g, b, 0), im);", "im = gf_fma(GF_RE(U, a, 0), GF_IM(g, b, 0), im);"),
    ("third row without the conjugation", "gf_device.cuh", "        GF_RE(m, 2, b) = re;\n        GF_IM(m, 2, b) = -im;", "        GF_RE(m, 2, b) = re;\n        GF_IM(m, 2, b) = im;"),
    ("x-backward neighbour of the wrong parity row", "gf_device.cuh", "        if (s.xodd) return s.h;                                   // x-1 = 2 xh: same xh",
     "        if (!s.xodd) return s.h;                                   // x-1 = 2 xh: same xh"),
    ("site parity ignores t", "gf_device.cuh", "s.xodd = (s.c[2] + s.c[3] + s.c[0] + parity) & 1u;", "s.xodd = (s.c[2] + s.c[3] + parity) & 1u;"),
    ("Philox key schedule", "gf_device.cuh", "k1 += 0xBB67AE85u;", "k1 += 0x9E3779B9u;"),
    ("K without the dagger on the backward link", "gf_sweep.cu", "GF_IM(K, a, b) += (TK)GF_IM(Uf[d], a, b) - (TK)GF_IM(Ub[d], b, a);",
     "GF_IM(K, a, b) += (TK)GF_IM(Uf[d], a, b) + (TK)GF_IM(Ub[d], b, a);"),
    ("second subgroup uses the first draw", "gf_sweep.cu", "sq1 = (double)(w[1] >> 8) * (1.0 / 16777216.0) < P.p;", "sq1 = (double)(w[0] >> 8) * (1.0 / 16777216.0) < P.p;"),
    ("draws keyed by the half-index", "gf_sweep.cu", "philox4x32_10(P.site_offset + 2u * h + s.xodd, 0u, counter, 0u, P.key0, P.key1, w);",
     "philox4x32_10(P.site_offset + 2u * h, 0u, counter, 0u, P.key0, P.key1, w);"),
    ("reverse traversal skips a block", "gf_sweep.cu", "const uint32_t bid = P.reverse ? gridDim.x - 1u - blockIdx.x : blockIdx.x;",
     "const uint32_t bid = P.reverse ? gridDim.x - blockIdx.x : blockIdx.x;"),
    ("theta keeps the trace", "gf_aux.cu", "const double d = GF_IM(M, a, a) - tr3;", "const double d = GF_IM(M, a, a);"),
    ("F from a wrong diagonal entry", "gf_aux.cu", "F += (double)Uf[0] + (double)Uf[8] + (double)Uf[16];", "F += (double)Uf[0] + (double)Uf[8] + (double)Uf[14];"),
    ("unitarity checker returns zero", "gf_aux.cu", "    block_reduce2<OpMax>(dmax, detmax, partials + partial_slot(mg));", "    block_reduce2<OpMax>(0.0 * dmax, 0.0 * detmax, partials + partial_slot(mg));"),
    ("device-side stop decision inverted", "gf_aux.cu", "    bool stop = th < tail.target;", "    bool stop = th > tail.target;"),
    # hand-off when fp32 stalls (gf_set_mixed_stall): the device's decision must be the host's
    ("stall ratio compared the wrong way on the device", "gf_aux.cu", "if (prev > 0.0 && th >= tail.stall * prev) stop = true;", "if (prev > 0.0 && th <= tail.stall * prev) stop = true;"),
    ("stall: previous theta never recorded on the device", "gf_aux.cu", "        *tail.prev = th;\n", "\n"),
    ("stall tested at the first evaluation (no previous theta)", "gf_aux.cu", "if (prev > 0.0 && th >= tail.stall * prev) stop = true;", "if (th >= tail.stall * prev) stop = true;"),
    ("stall ratio compared the wrong way on the host (run-ahead loop)", "gf_api.cu", "prev_theta > 0.0 && *theta_out >= stall * prev_theta;", "prev_theta > 0.0 && *theta_out <= stall * prev_theta;"),
    # re-projection inside the fix loop (gf_set_reunitarize_every)
    ("re-projection skipped by the run-ahead loop", "gf_api.cu", "err = enqueue_reunitarize(ctx, precision, ctx->stop_dev);", "err = GF_OK;"),
    ("re-projection skipped by the waiting loop", "gf_api.cu", "int er = enqueue_reunitarize(ctx, precision, nullptr);", "int er = GF_OK;"),
    ("re-projection in the fix loop copies without projecting", "gf_api.cu", "ctx->links[precision], ctx->links[precision], ctx->G, 1, 8, ctx->stream, stop);",
     "ctx->links[precision], ctx->links[precision], ctx->G, 0, 8, ctx->stream, stop);"),
    # path-specific: the lazy third rows of fp64 / 12-real, the recorded transformation, the fp32 / 18-real tail, deferred
    # temporal links, eq. 3 applied to a field, the re-projection, the plaquette, the Coulomb sums
    ("lazy third row of the forward link enters K with the wrong sign", "gf_sweep.cu",
     "fi = a < 2 ? GF_IM(Uf[d], a, b) : rf[2 * b + 1];", "fi = a < 2 ? GF_IM(Uf[d], a, b) : -rf[2 * b + 1];"),
    ("accumulated transformation: G g^dagger instead of g G", "gf_sweep.cu", "        mul_g_U<ROWS>(g, Gt, out);", "        mul_U_gdag<ROWS>(Gt, g, out);"),
    ("fp32 / 18-real tail loaded with re and im exchanged", "gf_device.cuh", "        m[16] = v.x;\n        m[17] = v.y;", "        m[16] = v.y;\n        m[17] = v.x;"),
    ("deferred temporal links: no lane carries G(x)", "gf_sweep.cu", "const bool gslot = MODE == MODE_DEFER && j == 0;", "const bool gslot = MODE == MODE_DEFER && j == 5;"),
    ("eq. 3 on a field: G(x+mu) without the dagger", "gf_aux.cu", "        mul_full(tmp, Gf, out, true);", "        mul_full(tmp, Gf, out, false);"),
    ("re-projection: row 1 not orthogonalised", "gf_aux.cu", "        GF_RE(m, 1, b) -= pr * GF_RE(m, 0, b) - pi * GF_IM(m, 0, b);", "        GF_RE(m, 1, b) -= pr * GF_RE(m, 0, b) + pi * GF_IM(m, 0, b);"),
    ("plaquette: third link not daggered", "gf_aux.cu", "            mul_full(C, A, D, true);", "            mul_full(C, A, D, false);"),
    ("Coulomb F and theta over all four directions", "gf_aux.cu", "        if (mu < mu0) continue;\n        T Uf[18], Ub[18];", "        T Uf[18], Ub[18];"),
    ("Coulomb F normalisation", "gf_api.cu", "t.scale0 = 1.0 / (3.0 * 3.0 * Vs);", "t.scale0 = 1.0 / (3.0 * 4.0 * Vs);"),
    ("theta normalisation", "gf_api.cu", "t.scale1 = 1.0 / (3.0 * (double)ctx->V * ctx->slab_n);", "t.scale1 = 1.0 / ((double)ctx->V * ctx->slab_n);"),
]


def _prepare(tmp):
    shutil.copytree(os.path.join(ROOT, PKG), os.path.join(tmp, PKG), ignore=shutil.ignore_patterns("__pycache__"))
    shutil.copytree(os.path.join(ROOT, "include"), os.path.join(tmp, "include"))
    shutil.copytree(os.path.join(ROOT, "oracle"), os.path.join(tmp, "oracle"), ignore=shutil.ignore_patterns("__pycache__"))
    shutil.copy(os.path.join(ROOT, "gf_inputs.py"), tmp)
    os.makedirs(os.path.join(tmp, "tests"))
    for f in TEST_FILES:
        shutil.copy(os.path.join(ROOT, "tests", f), os.path.join(tmp, "tests", f))
    shutil.copytree(os.path.join(ROOT, "tests", "golden"), os.path.join(tmp, "tests", "golden"))


def _build(name, fname, old, new):
    """Returns (name, tmp dir) with the mutated library built, or (name, error text)."""
    tmp = tempfile.mkdtemp(prefix="gf_kmut_")
    _prepare(tmp)
    if old is not None:
        path = os.path.join(tmp, PKG, "csrc", fname)
        text = open(path).read()
        if text.count(old) != 1:
            return name, "fragment occurs %d times in %s (the mutant list is stale)" % (text.count(old), fname)
        open(path, "w").write(text.replace(old, new))
    r = subprocess.run([sys.executable, os.path.join(tmp, PKG, "build.py")], capture_output=True, text=True)
    if r.returncode != 0:
        return name, "the mutated source does not compile: %s" % r.stderr[-300:]
    return name, tmp


def _run_tests(tmp):
    env = dict(os.environ, PYTHONPATH=tmp)
    env.pop("GF_KERNEL_MUTANTS", None)
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", "-m", "gpu", "-k", SELECT, "tests"],
                       cwd=tmp, env=env, capture_output=True, text=True, timeout=1200)
    failed = [l for l in r.stdout.splitlines() if l.startswith("FAILED") or l.startswith("ERROR")]
    return r.returncode, (failed[0] if failed else r.stdout.strip().splitlines()[-1] if r.stdout.strip() else r.stderr[-200:])


def test_the_mutant_list_is_current():
    """No GPU, no rebuild: every fragment occurs exactly once in today's sources, and its replacement differs."""
    stale = []
    for name, fname, old, new in MUTANTS:
        n = open(os.path.join(ROOT, PKG, "csrc", fname)).read().count(old)
        if n != 1 or old == new:
            stale.append("%s: fragment occurs %d times in %s" % (name, n, fname))
    assert not stale, stale
    assert len({m[0] for m in MUTANTS}) == len(MUTANTS)


@pytest.mark.gpu
def test_every_kernel_mutant_fails_a_gpu_parity_test():
    if os.environ.get("GF_KERNEL_MUTANTS") != "1":
        pytest.skip("opt-in (GF_KERNEL_MUTANTS=1): rebuilds the library once per mutant; last run: profiles/r3_kernel_mutants.md")
    jobs = [("control (unmutated)", None, None, None)] + MUTANTS
    with ThreadPoolExecutor(max_workers=max(1, min(5, (os.cpu_count() or 4) // 3))) as ex:
        built = list(ex.map(lambda j: _build(*j), jobs))
    report, survivors = [], []
    try:
        for name, tmp in built:
            assert os.path.isdir(tmp), "%s: %s" % (name, tmp)
            rc, first = _run_tests(tmp)
            report.append("%-48s -> rc %d  %s" % (name, rc, first))
            print(report[-1], flush=True)
            if name.startswith("control"):
                assert rc == 0, "the unmutated copy must pass: %s" % first
            elif rc == 0:
                survivors.append(name)
    finally:
        for _, tmp in built:
            if os.path.isdir(tmp):
                shutil.rmtree(tmp, ignore_errors=True)
    assert not survivors, "kernel mutants that pass the GPU parity tests: %s" % survivors
