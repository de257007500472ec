"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json's north_star: links 1e-12 (fp64) / 1e-5 (fp32)
max-abs after one sweep; F and theta 1e-10 / 1e-5 relative after 10 sweeps."""
import numpy as np
import pytest
import torch

import gf_inputs as gi
import oracle
import paper_1305_3440_b200 as gf

pytestmark = pytest.mark.gpu

PREC = {"f64": gf.GF_F64, "f32": gf.GF_F32}
LINK_TOL = {"f64": 1e-12, "f32": 1e-5}
REL_TOL = {"f64": 1e-10, "f32": 1e-5}
CDTYPE = {"f64": torch.complex128, "f32": torch.complex64}
# sizes span several tiles (128-thread blocks, 8..32 sites per warp) and ragged tails:
# 4x6x6x6 -> V/2 = 432 is not a multiple of 32; 6^4 -> 648 is not a multiple of 16
SHAPES = [(4, 4, 4, 4), (4, 6, 6, 6), (6, 6, 6, 6), (4, 6, 8, 10), (8, 8, 8, 8), (2, 2, 2, 2), (6, 2, 4, 2)]


def to_device(U, prec, dev):
    return torch.from_numpy(U).to(dev).to(CDTYPE[prec]).contiguous()


def oracle_input(U, prec):
    """The oracle is fed exactly what the GPU holds: the fp32-rounded field for fp32 runs."""
    if prec == "f32":
        return np.ascontiguousarray(U.astype(np.complex64).astype(np.complex128))
    return U.copy()


def make_field(dims, prec, dev, gauge=gf.GF_LANDAU, recon=18, seed=0):
    return gf.GaugeField(dims, gauge=gauge, recon=recon, precisions=(prec,), seed=seed, device=dev)


def get_links(fld, prec):
    return fld.unpack(PREC[prec], torch.complex128).cpu().numpy()


# ------------------------------------------------------------------------------ layout, reductions

@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("recon", [18, 12])
def test_pack_unpack_roundtrip_and_measure(cuda_device, dims, prec, recon):
    U = gi.smooth_random_gauge(dims, 0.5, 21)
    Uo = oracle_input(U, prec)
    for gauge, og in ((gf.GF_LANDAU, oracle.LANDAU), (gf.GF_COULOMB, oracle.COULOMB)):
        fld = make_field(dims, prec, cuda_device, gauge, recon)
        fld.pack(to_device(U, prec, cuda_device), PREC[prec])
        back = get_links(fld, prec)
        if recon == 18:
            assert np.array_equal(back, Uo)                      # byte-exact layout round trip
        else:
            assert np.array_equal(back[..., :2, :], Uo[..., :2, :])
            assert np.abs(back - Uo).max() < (1e-14 if prec == "f64" else 1e-6)
        F, th = fld.measure(PREC[prec])
        Fo = np.atleast_1d(oracle.functional(Uo, dims, og))
        tho = np.atleast_1d(oracle.theta(Uo, dims, og))
        tol = 1e-12 if (prec == "f64" or recon == 18) else 1e-6   # fp32 recon12 rebuilds row 2 in fp32
        assert np.allclose(F, Fo, rtol=tol, atol=0)
        assert np.allclose(th, tho, rtol=tol * 10, atol=0)
        assert np.allclose(fld.functional(PREC[prec]), F, rtol=0, atol=0)
        assert np.allclose(fld.theta(PREC[prec]), th, rtol=0, atol=0)
        assert abs(fld.plaquette(PREC[prec]) - oracle.plaquette(Uo, dims)) < (1e-13 if prec == "f64" else 1e-6)
        du, dd = fld.unitarity(PREC[prec])
        assert du < (1e-13 if prec == "f64" else 1e-6) and dd < (1e-13 if prec == "f64" else 1e-6)
        fld.close()


def test_unit_links(cuda_device):
    dims = (4, 6, 4, 6)
    fld = make_field(dims, "f64", cuda_device)
    fld.pack(to_device(gi.unit_links(dims), "f64", cuda_device), gf.GF_F64)
    F, th = fld.measure(gf.GF_F64)
    assert F == [1.0] and th == [0.0]
    fld.iterate(2, gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64)
    assert np.array_equal(get_links(fld, "f64"), gi.unit_links(dims))
    assert fld.plaquette(gf.GF_F64) == 1.0


# ------------------------------------------------------------------------------------ the sweep

ALGOS = [("relax", gf.GF_RELAX, oracle.RELAX, 1.0, 0.0), ("overrelax", gf.GF_OVERRELAX, oracle.OVERRELAX, 1.7, 0.0),
         ("stochastic", gf.GF_STOCHASTIC, oracle.STOCHASTIC, 1.0, 0.8)]


@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("lanes", [1, 2, 4])
def test_one_sweep_links_match_oracle(cuda_device, dims, prec, recon, lanes):
    U = gi.smooth_random_gauge(dims, 0.5, 31)
    for gauge, og in ((gf.GF_LANDAU, oracle.LANDAU), (gf.GF_COULOMB, oracle.COULOMB)):
        for name, algo, oalgo, omega, p in ALGOS:
            fld = make_field(dims, prec, cuda_device, gauge, recon, seed=2013)
            fld.set_tuning(PREC[prec], lanes, 128)
            fld.pack(to_device(U, prec, cuda_device), PREC[prec])
            Uo = oracle_input(U, prec)
            for parity in (0, 1):
                fld.sweep(parity, algo, omega, p, PREC[prec])
                oracle.sweep(Uo, dims, parity, og, oalgo, omega, p, seed=2013, half_sweep_counter=parity)
                err = np.abs(get_links(fld, prec) - Uo).max()
                assert err < LINK_TOL[prec], (name, gauge, parity, err)
            assert gf.gf_get_counter(fld.ctx) == 2
            fld.close()


def one_ulp_drift(U, dims, og, oalgo, omega, p, seed, samples=3):
    """How far apart two EXACT (fp64 oracle) runs of 10 sweeps end when their inputs differ by one fp32 ulp in
    every real (random direction; the largest of `samples` independent perturbations): the relative differences
    of F and theta.  Oracle-only; used to derive the fp32 tolerance of the stochastic variant."""
    a32 = np.ascontiguousarray(U.astype(np.complex64)).view(np.float32)
    rng = np.random.default_rng(12345)

    def run(start):
        W = np.ascontiguousarray(start.view(np.complex64).astype(np.complex128))
        for it in range(10):
            for parity in (0, 1):
                oracle.sweep(W, dims, parity, og, oalgo, omega, p, seed=seed, half_sweep_counter=2 * it + parity)
        return np.atleast_1d(oracle.functional(W, dims, og)), np.atleast_1d(oracle.theta(W, dims, og))

    F0, t0 = run(a32)
    dF = dth = 0.0
    for _ in range(samples):
        towards = np.where(rng.random(a32.shape) < 0.5, -np.inf, np.inf).astype(np.float32)
        F1, t1 = run(np.nextafter(a32, towards))
        dF, dth = max(dF, float(np.abs(F1 / F0 - 1).max())), max(dth, float(np.abs(t1 / t0 - 1).max()))
    return dF, dth


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 8, 10), (8, 8, 8, 8)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("recon", [18, 12])
def test_ten_sweeps_F_theta_match_oracle(cuda_device, dims, prec, recon):
    for field, U in (("smooth", gi.smooth_random_gauge(dims, 0.5, 41)), ("hot", gi.hot_links(dims, 42))):
        for gauge, og in ((gf.GF_LANDAU, oracle.LANDAU), (gf.GF_COULOMB, oracle.COULOMB)):
            for name, algo, oalgo, omega, p in ALGOS[1:]:
                # north_star: 1e-10 (fp64) / 1e-5 (fp32) relative after 10 sweeps.  One derived exception (DESIGN.md,
                # "Tolerances"): the stochastic g -> g^2 step is microcanonical, it does not contract differences, and
                # two EXACT runs whose inputs differ by one fp32 ulp already end further apart than 1e-5 (measured
                # right here, by the oracle alone).  An fp32 run rounds every link to fp32 once per half-sweep, 20
                # such perturbations in 10 sweeps, adding in quadrature: the bound for fp32 + stochastic is
                # sqrt(20) x the one-ulp drift, never below north_star's 1e-5.  (A wrong draw or a wrong update
                # changes theta by factors, not by 1e-4.)
                rtol_F = rtol_th = REL_TOL[prec]
                if prec == "f32" and name == "stochastic":
                    dF, dth = one_ulp_drift(U, dims, og, oalgo, omega, p, 7)
                    rtol_F, rtol_th = max(rtol_F, 20 ** 0.5 * dF), max(rtol_th, 20 ** 0.5 * dth)
                    assert rtol_th < 1e-2                   # the exception stays a small tolerance
                fld = make_field(dims, prec, cuda_device, gauge, recon, seed=7)
                fld.pack(to_device(U, prec, cuda_device), PREC[prec])
                Uo = oracle_input(U, prec)
                fld.iterate(10, algo, omega, p, PREC[prec])
                for it in range(10):
                    for parity in (0, 1):
                        oracle.sweep(Uo, dims, parity, og, oalgo, omega, p, seed=7, half_sweep_counter=2 * it + parity)
                F, th = fld.measure(PREC[prec])
                Fo = np.atleast_1d(oracle.functional(Uo, dims, og))
                tho = np.atleast_1d(oracle.theta(Uo, dims, og))
                assert np.allclose(F, Fo, rtol=rtol_F, atol=0), (field, name, gauge, rtol_F, np.abs(np.array(F) / Fo - 1).max())
                assert np.allclose(th, tho, rtol=rtol_th, atol=0), (field, name, gauge, rtol_th, np.abs(np.array(th) / tho - 1).max())
                # the links themselves drift apart as rounding differences are amplified sweep after sweep
                # (strongly on the hot field); only a loose bound is meaningful here
                assert np.abs(get_links(fld, prec) - Uo).max() < (1e-8 if prec == "f64" else 0.1)
                fld.close()


def test_stochastic_counter_and_seed_are_honoured(cuda_device):
    dims = (4, 4, 4, 4)
    U = gi.smooth_random_gauge(dims, 0.5, 51)
    fld = make_field(dims, "f64", cuda_device, seed=1)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    gf.gf_set_rng(fld.ctx, 0xDEADBEEF12345678, 1000)
    fld.sweep(1, gf.GF_STOCHASTIC, 1.0, 0.5, gf.GF_F64)
    Uo = U.copy()
    oracle.sweep(Uo, dims, 1, oracle.LANDAU, oracle.STOCHASTIC, 1.0, 0.5, seed=0xDEADBEEF12345678, half_sweep_counter=1000)
    assert np.abs(get_links(fld, "f64") - Uo).max() < 1e-12
    Uw = U.copy()
    oracle.sweep(Uw, dims, 1, oracle.LANDAU, oracle.STOCHASTIC, 1.0, 0.5, seed=0xDEADBEEF12345678, half_sweep_counter=1001)
    assert np.abs(Uw - Uo).max() > 1e-3               # a different counter is a different sweep


def test_philox_known_answers_on_device(cuda_device):
    import os
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    w = np.array([[int(x, 16) for x in r] for r in rows], dtype=np.uint32)
    rng = np.random.default_rng(3)
    extra_c = rng.integers(0, 2 ** 32, (500, 4), dtype=np.uint32)
    extra_k = rng.integers(0, 2 ** 32, (500, 2), dtype=np.uint32)
    ctr = np.concatenate([w[:, 0:4], extra_c])
    key = np.concatenate([w[:, 4:6], extra_k])
    fld = make_field((4, 4, 4, 4), "f64", cuda_device)
    d_c = torch.from_numpy(ctr.view(np.int32)).to(cuda_device)
    d_k = torch.from_numpy(key.view(np.int32)).to(cuda_device)
    d_o = torch.zeros_like(d_c)
    gf.gf_debug_philox(fld.ctx, len(ctr), d_c.data_ptr(), d_k.data_ptr(), d_o.data_ptr())
    torch.cuda.synchronize()
    out = d_o.cpu().numpy().view(np.uint32)
    assert np.array_equal(out[:3], w[:, 6:10])                         # published vectors
    for i in range(3, len(ctr)):                                        # and the oracle, bit for bit
        assert tuple(out[i]) == oracle.philox4x32_10(ctr[i].tolist(), key[i].tolist())


def test_philox_agrees_with_curand_on_device(cuda_device):
    """Pin 13: a library routine as third opinion.  cuRAND's Philox4_32_10 device
    generator (tests/curand_philox_ref.cu, test-only) initialised with (seed, subsequence = half-sweep
    counter, offset = 4 * site) returns, as its first block, Philox4x32-10 of the counter
    (site lo, site hi, counter, 0) under the key (seed lo, seed hi) -- the sweep kernel's draw.  The
    oracle's and the library's device implementations must both reproduce it bit for bit."""
    import ctypes
    import os
    import subprocess
    here = os.path.dirname(os.path.abspath(__file__))
    so, src = os.path.join(here, "libcurand_philox_ref.so"), os.path.join(here, "curand_philox_ref.cu")
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        subprocess.run(["/usr/local/cuda/bin/nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-shared",
                        "-Xcompiler", "-fPIC", src, "-o", so], check=True)
    ref = ctypes.CDLL(so)
    ref.curand_philox_ref.argtypes = [ctypes.c_int] + [ctypes.c_void_p] * 5
    rng = np.random.default_rng(17)
    n = 2000
    seed = rng.integers(0, 2 ** 63, n, dtype=np.int64)
    site = rng.integers(0, 2 ** 40, n, dtype=np.int64)           # beyond 2^32: exercises the high word
    site[:4] = [0, 1, 2 ** 32 - 1, 2 ** 32]
    counter = rng.integers(0, 2 ** 32, n, dtype=np.int64)
    d_seed, d_sub, d_off = (torch.from_numpy(a).to(cuda_device) for a in (seed, counter, 4 * site))
    d_ref = torch.zeros(n * 4, dtype=torch.int32, device=cuda_device)
    assert ref.curand_philox_ref(n, d_seed.data_ptr(), d_sub.data_ptr(), d_off.data_ptr(), d_ref.data_ptr(),
                                 torch.cuda.current_stream().cuda_stream) == 0
    ctr = np.stack([site & 0xffffffff, site >> 32, counter, np.zeros(n, np.int64)], axis=1).astype(np.uint32)
    key = np.stack([seed & 0xffffffff, seed >> 32], axis=1).astype(np.uint32)
    fld = make_field((4, 4, 4, 4), "f64", cuda_device)
    d_c = torch.from_numpy(ctr.view(np.int32)).to(cuda_device)
    d_k = torch.from_numpy(key.view(np.int32)).to(cuda_device)
    d_o = torch.zeros_like(d_c)
    gf.gf_debug_philox(fld.ctx, n, d_c.data_ptr(), d_k.data_ptr(), d_o.data_ptr())
    torch.cuda.synchronize()
    want = d_ref.cpu().numpy().view(np.uint32).reshape(n, 4)
    assert np.array_equal(d_o.cpu().numpy().view(np.uint32), want)
    for i in range(0, n, 10):
        assert oracle.philox4x32_10(ctr[i].tolist(), key[i].tolist()) == tuple(want[i])
        u = oracle.site_uniforms(int(seed[i]), int(counter[i]), int(site[i]))
        assert all(u[k] == (int(want[i][k]) >> 8) / 2.0 ** 24 for k in range(3))


# ---------------------------------------------------------------------------------- the fix loop

@pytest.mark.parametrize("seed", [0, 1, 2, 3, 4])
def test_config1_fix_until_matches_oracle(cuda_device, seed):
    """configs[0]: 4^4 fp64, omega 1.7, theta < 1e-12, check_every 1."""
    dims = (4, 4, 4, 4)
    U = gi.smooth_random_gauge(dims, 0.3, seed)
    Uo = U.copy()
    it_o, th_o, conv = oracle.fix_until(Uo, dims, oracle.LANDAU, oracle.OVERRELAX, 1.7, theta_target=1e-12, max_iter=2000)
    fld = make_field(dims, "f64", cuda_device)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    P0 = fld.plaquette(gf.GF_F64)
    rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64, 1e-12, 2000, 1)
    assert rc == gf.GF_OK and conv
    assert abs(it - it_o) <= 1 and th < 1e-12
    if it == it_o:
        assert abs(th / th_o - 1) < 1e-3      # theta ~ 1e-12 is a sum of squares of 1e-7-size rounding-limited entries
        assert np.abs(get_links(fld, "f64") - Uo).max() < 1e-11
    assert abs(fld.plaquette(gf.GF_F64) - P0) < 1e-12
    du, dd = fld.unitarity(gf.GF_F64)
    assert du < 1e-12 and dd < 1e-12
    assert abs(fld.functional(gf.GF_F64)[0] - oracle.functional(Uo, dims)) < 1e-10


def test_fix_until_check_every_and_max_iter(cuda_device):
    dims = (4, 4, 4, 4)
    U = gi.smooth_random_gauge(dims, 0.3, 0)
    fld = make_field(dims, "f64", cuda_device)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64, 1e-12, 25, 10)
    assert rc == gf.GF_NOT_CONVERGED and it == 25
    Uo = U.copy()
    it_o, th_o, conv = oracle.fix_until(Uo, dims, oracle.LANDAU, oracle.OVERRELAX, 1.7, theta_target=1e-12, max_iter=25, check_every=10)
    assert it_o == 25 and not conv and abs(th / th_o - 1) < 1e-9
    rc, it2, th2 = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64, 1e-12, 2000, 7)
    assert rc == gf.GF_OK and it2 % 7 == 0 and th2 < 1e-12


def test_coulomb_stochastic_fix_matches_oracle(cuda_device):
    """Small replica of configs[4]: Coulomb, stochastic p = 0.8, Philox seed 2013, per-slice theta."""
    dims = (8, 8, 8, 8)
    U = gi.smooth_random_gauge(dims, 0.6, 1)
    fld = make_field(dims, "f64", cuda_device, gf.GF_COULOMB, seed=2013)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    P0 = fld.plaquette(gf.GF_F64)
    rc, it, th = fld.fix_until(gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64, 1e-12, 50000, 20)
    assert rc == gf.GF_OK and th < 1e-12
    assert max(fld.theta(gf.GF_F64)) == th
    assert abs(fld.plaquette(gf.GF_F64) - P0) < 1e-12
    Uo = U.copy()
    it_o, th_o, conv = oracle.fix_until(Uo, dims, oracle.COULOMB, oracle.STOCHASTIC, 1.0, 0.8, seed=2013,
                                        theta_target=1e-12, max_iter=50000, check_every=20)
    assert conv and abs(it - it_o) <= 20


def test_mixed_precision_fix(cuda_device):
    """configs[2]'s mixed mode on a small lattice: fp32 to 1e-6, cast + re-projection, fp64 to 1e-12."""
    dims = (8, 8, 8, 8)
    U = gi.smooth_random_gauge(dims, 0.5, 1234)
    fld = gf.GaugeField(dims, precisions=("f32", "f64"), device=cuda_device)
    fld.pack(to_device(U, "f32", cuda_device), gf.GF_F32)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    P0 = fld.plaquette(gf.GF_F64)
    rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_MIXED, 1e-12, 20000, 10)
    assert rc == gf.GF_OK and th < 1e-12
    du, dd = fld.unitarity(gf.GF_F64)
    assert du < 1e-12 and dd < 1e-12
    assert abs(fld.plaquette(gf.GF_F64) - P0) < 1e-5       # fp32 phase: gauge orbit kept to fp32 accuracy
    Ug = get_links(fld, "f64")
    assert oracle.theta(np.ascontiguousarray(Ug), dims) < 1.1e-12       # the oracle agrees it is fixed


def test_error_codes_on_device(cuda_device):
    dims = (4, 4, 4, 4)
    fld = make_field(dims, "f64", cuda_device)
    B = gf.binding
    assert B.lib.gf_sweep(fld.ctx, 2, gf.GF_RELAX, 1.0, 0.0, gf.GF_F64) == gf.GF_EINVAL
    assert B.lib.gf_sweep(fld.ctx, 0, 5, 1.0, 0.0, gf.GF_F64) == gf.GF_EINVAL
    assert B.lib.gf_sweep(fld.ctx, 0, gf.GF_OVERRELAX, 2.0, 0.0, gf.GF_F64) == gf.GF_EINVAL
    assert B.lib.gf_sweep(fld.ctx, 0, gf.GF_STOCHASTIC, 1.0, 1.5, gf.GF_F64) == gf.GF_EINVAL
    assert B.lib.gf_sweep(fld.ctx, 0, gf.GF_RELAX, 1.0, 0.0, gf.GF_F32) == gf.GF_ESTATE
    assert "precision" in gf.gf_last_error(fld.ctx)
    assert B.lib.gf_fix_until(fld.ctx, gf.GF_RELAX, 1.0, 0.0, gf.GF_MIXED, 1e-12, 10, 1, None, None) == gf.GF_ESTATE
    assert B.lib.gf_set_tuning(fld.ctx, gf.GF_F64, 3, 128) == gf.GF_EINVAL
    assert gf.gf_get_counter(fld.ctx) == 0


# Full-size parity (32^4 in bench.py's launch configuration, every link, all four storage variants; configs[4]
# at full size; the mixed-precision runs) lives in tests/test_gpu_fullsize.py.


# ------------------------------------------------------------------------- out-of-bounds writes

@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 6, 6, 6), (6, 2, 4, 2), (4, 6, 8, 10)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("recon", [18, 12])
def test_no_writes_outside_the_lent_buffers(cuda_device, dims, prec, recon):
    """compute-sanitizer is closed on this pool: the link, transformation and workspace buffers are
    carved out of larger allocations with 0xA5 guard zones on both sides; every kernel family runs on
    ragged lattices with every lane count and the guards must come back untouched."""
    from paper_1305_3440_b200 import binding as B
    guard = 1 << 16
    nbytes = [B.gf_storage_bytes(dims, PREC[prec], recon), B.gf_transform_bytes(dims, PREC[prec], recon),
              B.gf_workspace_bytes(dims)]
    bufs = [torch.full((n + 2 * guard,), 0xA5, dtype=torch.uint8, device=cuda_device) for n in nbytes]
    ptrs = [b.data_ptr() + guard for b in bufs]
    assert all(p % 16 == 0 for p in ptrs)
    links = (ptrs[0], 0) if prec == "f64" else (0, ptrs[0])
    ctx = B.gf_init_lattice(dims, gf.GF_COULOMB, recon, links[0], links[1], ptrs[2],
                            torch.cuda.current_stream().cuda_stream, 3)
    U = to_device(gi.smooth_random_gauge(dims, 0.5, 2), prec, cuda_device)
    out = torch.empty_like(U)
    B.gf_pack(ctx, U.data_ptr(), prec == "f64", PREC[prec])
    B.gf_set_transform(ctx, ptrs[1] if prec == "f64" else 0, 0 if prec == "f64" else ptrs[1])
    B.gf_transform_identity(ctx, PREC[prec])
    for defer in (0, 1):
        B.gf_set_coulomb_mode(ctx, defer, 0)
        for lanes in (1, 2, 4):
            B.gf_set_tuning(ctx, PREC[prec], lanes, 64)
            for parity in (0, 1):
                B.gf_sweep(ctx, parity, gf.GF_STOCHASTIC, 1.0, 0.5, PREC[prec])
        B.gf_set_slice_mask(ctx, [1, 0] * (dims[0] // 2))
        B.gf_sweep(ctx, 0, gf.GF_OVERRELAX, 1.5, 0.0, PREC[prec])
        B.gf_set_slice_mask(ctx, None)
        B.gf_measure(ctx, PREC[prec], dims[0])
    B.gf_coulomb_finish(ctx, PREC[prec])
    B.gf_apply_transform(ctx, PREC[prec], PREC[prec], PREC[prec])
    B.gf_reunitarize(ctx, PREC[prec])
    B.gf_plaquette(ctx, PREC[prec])
    B.gf_unitarity(ctx, PREC[prec])
    B.gf_unpack(ctx, out.data_ptr(), prec == "f64", PREC[prec])
    torch.cuda.synchronize()
    B.gf_destroy(ctx)
    assert torch.isfinite(torch.view_as_real(out)).all()
    for b, n in zip(bufs, nbytes):
        assert bool((b[:guard] == 0xA5).all()) and bool((b[guard + n:] == 0xA5).all())


# ------------------------------------------------------------------------------------- fuzz

def test_random_small_lattices_against_oracle(cuda_device):
    """40 seeded random combinations of (dims, gauge, algorithm, storage, lanes, block):
    two iterations on the device against the oracle, links within the one-sweep tolerance x 4."""
    rng = np.random.default_rng(2024)
    for case in range(40):
        dims = tuple(int(2 * rng.integers(1, 6)) for _ in range(4))
        prec = ("f64", "f32")[int(rng.integers(0, 2))]
        recon = (18, 12)[int(rng.integers(0, 2))]
        gauge = (gf.GF_LANDAU, gf.GF_COULOMB)[int(rng.integers(0, 2))]
        algo = (gf.GF_RELAX, gf.GF_OVERRELAX, gf.GF_STOCHASTIC)[int(rng.integers(0, 3))]
        lanes, block = (1, 2, 4)[int(rng.integers(0, 3))], (64, 128, 256)[int(rng.integers(0, 3))]
        omega, p, seed = 1.0 + 0.9 * float(rng.random()), float(rng.random()), int(rng.integers(0, 2 ** 40))
        U = gi.smooth_random_gauge(dims, 0.5, 100 + case)
        fld = make_field(dims, prec, cuda_device, gauge=gauge, recon=recon, seed=seed)
        fld.pack(to_device(U, prec, cuda_device), PREC[prec])
        fld.set_tuning(PREC[prec], lanes, block)
        rng.integers(0, 3)                       # (keeps the seeded case list of round 1)
        fld.iterate(2, algo, omega, p, PREC[prec])
        Uo = oracle_input(U, prec)
        og = oracle.LANDAU if gauge == gf.GF_LANDAU else oracle.COULOMB
        for it in range(2):
            for parity in (0, 1):
                oracle.sweep(Uo, dims, parity, og, algo, omega, p, seed=seed, half_sweep_counter=2 * it + parity)
        err = np.abs(get_links(fld, prec) - Uo).max()
        assert err < 4 * LINK_TOL[prec], (case, dims, prec, recon, gauge, algo, lanes, block, err)
        F, th = fld.measure(PREC[prec])
        assert np.allclose(F, oracle.functional(Uo, dims, og), rtol=0, atol=1e-5 if prec == "f32" else 1e-12)
        fld.close()


def test_measure_async_equals_measure(cuda_device):
    """gf_measure_async / gf_measure_collect: several evaluations in flight between sweeps give exactly
    the values the synchronous gf_measure gives at the same points (Landau and Coulomb)."""
    from paper_1305_3440_b200 import binding as B
    dims = (6, 4, 6, 4)
    U = to_device(gi.smooth_random_gauge(dims, 0.5, 9), "f64", cuda_device)
    for gauge in (gf.GF_LANDAU, gf.GF_COULOMB):
        a = make_field(dims, "f64", cuda_device, gauge=gauge)
        b = make_field(dims, "f64", cuda_device, gauge=gauge)
        a.pack(U, gf.GF_F64)
        b.pack(U, gf.GF_F64)
        want = []
        for k in range(5):
            a.iterate(2, gf.GF_OVERRELAX, 1.6, 0.0, gf.GF_F64)
            want.append(a.measure(gf.GF_F64))
            b.iterate(2, gf.GF_OVERRELAX, 1.6, 0.0, gf.GF_F64)
            b.measure_async(gf.GF_F64, k)
        got = [b.measure_collect(k) for k in range(5)]
        assert got == want
        assert B.lib.gf_measure_collect(b.ctx, 0, None, None) == gf.GF_ESTATE          # collected slots are empty again
        assert B.lib.gf_measure_async(b.ctx, gf.GF_F64, 16) == gf.GF_EINVAL
        a.close()
        b.close()


# ------------------------------------------------------------------------------ extreme shapes

@pytest.mark.parametrize("dims", [(4096, 2, 2, 2), (2, 1024, 2, 2), (2, 2, 1022, 2), (2, 2, 2, 1000), (2, 2, 2, 2)])
@pytest.mark.parametrize("prec,recon", [("f64", 18), ("f32", 12)])
def test_extreme_aspect_ratios(cuda_device, dims, prec, recon):
    """The largest time extent the library accepts (4096 slices of 4 sites per parity: per-slice reductions with one
    partial block each, a 4096-entry slice list) and lattices that are one long line in x, y or z (x rows of two sites:
    every x neighbour wraps; strides that are not multiples of the tile): one overrelaxation iteration in Landau gauge and
    one stochastic iteration in Coulomb gauge against the oracle, F / theta per slice, default launch configuration."""
    U = gi.smooth_random_gauge(dims, 0.4, 77)
    for gauge, og, algo, oalgo, omega, p in ((gf.GF_LANDAU, oracle.LANDAU, gf.GF_OVERRELAX, oracle.OVERRELAX, 1.7, 0.0),
                                             (gf.GF_COULOMB, oracle.COULOMB, gf.GF_STOCHASTIC, oracle.STOCHASTIC, 1.0, 0.8)):
        fld = make_field(dims, prec, cuda_device, gauge, recon, seed=11)
        fld.pack(to_device(U, prec, cuda_device), PREC[prec])
        Uo = oracle_input(U, prec)
        if recon == 12:
            Uin = Uo
            Uo = get_links(fld, prec)                             # row 2 as the device rebuilds it ...
            assert np.array_equal(Uo[..., :2, :], Uin[..., :2, :])              # ... from rows it holds bit for bit
            assert np.abs(Uo[..., 2, :] - Uin[..., 2, :]).max() < (1e-14 if prec == "f64" else 1e-6)
        fld.iterate(1, algo, omega, p, PREC[prec])
        for parity in (0, 1):
            oracle.sweep(Uo, dims, parity, og, oalgo, omega, p, seed=11, half_sweep_counter=parity)
        assert np.abs(get_links(fld, prec) - Uo).max() < 2 * LINK_TOL[prec]
        F, th = fld.measure(PREC[prec])
        Fo, tho = np.atleast_1d(oracle.functional(Uo, dims, og)), np.atleast_1d(oracle.theta(Uo, dims, og))
        assert len(F) == (dims[0] if gauge == gf.GF_COULOMB else 1)
        assert np.allclose(F, Fo, rtol=REL_TOL[prec], atol=0)
        assert np.allclose(th, tho, rtol=20 * REL_TOL[prec], atol=1e-30)
        assert abs(fld.plaquette(PREC[prec]) - oracle.plaquette(Uo, dims)) < (1e-12 if prec == "f64" else 1e-5)
        if gauge == gf.GF_COULOMB and dims[0] > 2:               # slice freezing with the longest possible slice list
            mask = np.ones(dims[0], dtype=np.uint8)
            mask[1::3] = 0
            fld.set_slice_mask(mask)
            before = get_links(fld, prec)
            c0 = gf.gf_get_counter(fld.ctx)
            fld.iterate(1, algo, omega, p, PREC[prec])
            Um = before.copy()
            for parity in (0, 1):
                oracle.sweep_masked(Um, dims, parity, mask, algo=oalgo, omega=omega, p=p, seed=11, half_sweep_counter=c0 + parity)
            assert np.abs(get_links(fld, prec) - Um).max() < 2 * LINK_TOL[prec]
        fld.close()


def test_the_link_tolerance_detects_a_relative_error_of_1e_9(cuda_device):
    """Sensitivity of the 1e-12 link comparison: the same half-sweep with omega off by one part in 10^9, or with one real
    of one input link off by 1e-9, lands outside the tolerance -- a kernel mistake of that size cannot hide in it."""
    dims = (4, 6, 4, 6)
    U = gi.smooth_random_gauge(dims, 0.5, 5)
    Uo = U.copy()
    oracle.sweep(Uo, dims, 0, oracle.LANDAU, oracle.OVERRELAX, 1.7)
    fld = make_field(dims, "f64", cuda_device)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    fld.sweep(0, gf.GF_OVERRELAX, 1.7 * (1 + 1e-9), 0.0, gf.GF_F64)
    err = np.abs(get_links(fld, "f64") - Uo).max()
    assert 1e-11 < err < 1e-7, err
    W = U.copy()
    W[1, 2, 3, 0, 2, 1, 1] += 1e-9
    fld.pack(to_device(W, "f64", cuda_device), gf.GF_F64)
    fld.sweep(0, gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64)
    err = np.abs(get_links(fld, "f64") - Uo).max()
    assert 1e-11 < err < 1e-7, err
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)            # control: the unperturbed run is inside
    fld.sweep(0, gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64)
    assert np.abs(get_links(fld, "f64") - Uo).max() < 1e-12
    fld.close()
