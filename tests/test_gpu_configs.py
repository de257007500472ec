"""GPU tests at BASELINE.json's full config sizes (configs[1], [3], [4]) in the default launch
configuration: sampled outputs recomputed one by one by the oracle, properties that hold at any
size (plaquette, unitarity, monotone F, theta falling), and the fix loop against the oracle where the
oracle finishes in seconds (16^4)."""
import numpy as np
import pytest
import torch

import gf_inputs as gi
import oracle
import paper_1305_3440_b200 as gf
from gpu_helpers import assert_pack_round_trip

pytestmark = pytest.mark.gpu

PREC = {"f64": gf.GF_F64, "f32": gf.GF_F32}
CDTYPE = {"f64": torch.complex128, "f32": torch.complex64}
LINK_TOL = {"f64": 1e-12, "f32": 1e-5}


def _site_and_backward(dims, s):
    nt, nx, ny, nz = dims
    x, y, z, t = s % nx, (s // nx) % ny, (s // (nx * ny)) % nz, s // (nx * ny * nz)

    def idx(t, x, y, z):
        return x + nx * (y + ny * (z + nz * t))
    back = [idx((t - 1) % nt, x, y, z), idx(t, (x - 1) % nx, y, z), idx(t, x, (y - 1) % ny, z), idx(t, x, y, (z - 1) % nz)]
    return (x + y + z + t) % 2, back


def sampled_sweep_check(fld, dims, prec, gauge, ogauge, algo, oalgo, omega, p, seed, nsamples, rng):
    """One iteration (parity 0 then 1); after each half-sweep `nsamples` random active sites are
    recomputed by the oracle's single-site update from the pre-sweep links (and the oracle's own
    Philox draws for the stochastic variant)."""
    before = fld.unpack(PREC[prec], torch.complex128).reshape(-1, 4, 3, 3)
    V = before.shape[0]
    for parity in (0, 1):
        counter = gf.gf_get_counter(fld.ctx)
        fld.sweep(parity, algo, omega, p, PREC[prec])
        after = fld.unpack(PREC[prec], torch.complex128).reshape(-1, 4, 3, 3)
        picked = 0
        while picked < nsamples:
            s = int(rng.integers(0, V))
            par, back = _site_and_backward(dims, s)
            if par != parity:
                continue
            picked += 1
            fwd = before[s].cpu().numpy().copy()
            bwd = np.stack([before[back[mu], mu].cpu().numpy() for mu in range(4)])
            u = oracle.site_uniforms(seed, counter, s) if oalgo == oracle.STOCHASTIC else (0.0, 0.0, 0.0)
            oracle.update_links8(fwd, bwd, ogauge, oalgo, omega, p, u)
            got_f = after[s].cpu().numpy()
            got_b = np.stack([after[back[mu], mu].cpu().numpy() for mu in range(4)])
            assert np.abs(got_f - fwd).max() < LINK_TOL[prec], (s, parity)
            assert np.abs(got_b - bwd).max() < LINK_TOL[prec], (s, parity)
        before = after
        del after


# ------------------------------------------------------------------------------ configs[1]: 16^4

def test_config2_16_4_smooth_fix_matches_oracle(cuda_device):
    """16^4, eps 0.5, seed 1234, omega 1.7: fp64 until theta < 1e-12 (check every 10) against the
    oracle's fix loop; fp32 until theta < 1e-6."""
    dims = (16, 16, 16, 16)
    U = gi.smooth_random_gauge(dims, 0.5, 1234)
    oracle.set_threads(0)
    Uo = U.copy()
    it_o, th_o, conv = oracle.fix_until(Uo, dims, oracle.LANDAU, oracle.OVERRELAX, 1.7, theta_target=1e-12,
                                        max_iter=20000, check_every=10)
    oracle.set_threads(1)
    assert conv
    fld = gf.GaugeField(dims, precisions=("f64", "f32"), device=cuda_device)
    Ud = torch.from_numpy(U).to(cuda_device)
    fld.pack(Ud, gf.GF_F64)
    fld.pack(Ud.to(torch.complex64), gf.GF_F32)
    P0 = fld.plaquette(gf.GF_F64)
    assert abs(P0 - oracle.plaquette(U, dims)) < 1e-13
    rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64, 1e-12, 20000, 10)
    assert rc == gf.GF_OK and th < 1e-12
    assert abs(it - it_o) <= 10, (it, it_o)
    assert abs(fld.plaquette(gf.GF_F64) - P0) < 1e-12
    du, dd = fld.unitarity(gf.GF_F64)
    assert du < 1e-12 and dd < 1e-12
    F = fld.functional(gf.GF_F64)[0]
    assert abs(F - oracle.functional(Uo, dims)) < 1e-9          # same maximum of the functional
    got = fld.unpack(gf.GF_F64).cpu().numpy()
    assert oracle.theta(np.ascontiguousarray(got), dims) < 1.01e-12      # the oracle agrees it is fixed
    # fp32 to 1e-6
    rc, it32, th32 = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F32, 1e-6, 20000, 10)
    assert rc == gf.GF_OK and th32 < 1e-6 and it32 < it
    assert abs(fld.plaquette(gf.GF_F32) - P0) < 1e-5
    fld.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_config2_16_4_hot_500_sweeps(cuda_device, prec):
    """16^4 Haar-random links, 500 fixed sweeps: F rises monotonically (checked every 50), theta falls
    overall, gauge invariants hold; after the first 10 sweeps F and theta match the oracle."""
    dims = (16, 16, 16, 16)
    U = gi.hot_links(dims, 1234)
    Uo = np.ascontiguousarray(U.astype(np.complex64).astype(np.complex128)) if prec == "f32" else U.copy()
    fld = gf.GaugeField(dims, precisions=(prec,), device=cuda_device)
    fld.pack(torch.from_numpy(U).to(cuda_device).to(CDTYPE[prec]), PREC[prec])
    P0 = fld.plaquette(PREC[prec])
    F0, th0 = fld.measure(PREC[prec])
    fld.iterate(10, gf.GF_OVERRELAX, 1.7, 0.0, PREC[prec])
    oracle.set_threads(0)
    for it in range(10):
        for parity in (0, 1):
            oracle.sweep(Uo, dims, parity, oracle.LANDAU, oracle.OVERRELAX, 1.7)
    oracle.set_threads(1)
    F, th = fld.measure(PREC[prec])
    rtol = 1e-10 if prec == "f64" else 1e-5
    assert abs(F[0] / oracle.functional(Uo, dims) - 1) < rtol
    assert abs(th[0] / oracle.theta(Uo, dims) - 1) < rtol
    Fs, ths = [F[0]], [th[0]]
    for _ in range(49):
        fld.iterate(10, gf.GF_OVERRELAX, 1.7, 0.0, PREC[prec])
        F, th = fld.measure(PREC[prec])
        Fs.append(F[0])
        ths.append(th[0])
    assert all(b > a for a, b in zip(Fs[4::5], Fs[9::5])) and Fs[-1] > F0[0] + 0.3
    assert ths[-1] < 1e-2 * th0[0]
    assert abs(fld.plaquette(PREC[prec]) - P0) < (1e-12 if prec == "f64" else 1e-5)
    du, dd = fld.unitarity(PREC[prec])
    assert du < (1e-12 if prec == "f64" else 1e-4)
    fld.close()


# ------------------------------------------------------------------------------ configs[3]: 64^4

@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_config4_64_4(cuda_device, prec):
    """64^4 (16.8 M sites; 9.66 GB of fp64 links, byte offsets beyond 2^32), omega 1.8: one iteration
    with sampled sites recomputed by the oracle, then 200 sweeps with F/theta every 10."""
    dims = (64, 64, 64, 64)
    U = gi.torch_smooth_random_gauge(dims, 0.6, 4, device=cuda_device).to(CDTYPE[prec])
    fld = gf.GaugeField(dims, precisions=(prec,), device=cuda_device)
    fld.pack(U, PREC[prec])
    assert_pack_round_trip(fld, PREC[prec], U)      # sampled_sweep_check reads the oracle's input back from the device
    del U
    torch.cuda.empty_cache()
    P0 = fld.plaquette(PREC[prec])
    rng = np.random.default_rng(64)
    sampled_sweep_check(fld, dims, prec, gf.GF_LANDAU, oracle.LANDAU, gf.GF_OVERRELAX, oracle.OVERRELAX, 1.8, 0.0, 0, 24, rng)
    torch.cuda.empty_cache()
    Fs, ths = [], []
    for _ in range(20):
        fld.iterate(10, gf.GF_OVERRELAX, 1.8, 0.0, PREC[prec])
        F, th = fld.measure(PREC[prec])
        Fs.append(F[0])
        ths.append(th[0])
    assert all(b > a for a, b in zip(Fs, Fs[1:]))                  # F keeps rising
    assert ths[-1] < 0.1 * ths[0]
    assert abs(fld.plaquette(PREC[prec]) - P0) < (1e-12 if prec == "f64" else 1e-5)
    du, dd = fld.unitarity(PREC[prec])
    assert du < (1e-12 if prec == "f64" else 1e-4) and dd < (1e-12 if prec == "f64" else 1e-4)
    fld.close()


# ------------------------------------------------------------------------------ configs[4]: Coulomb

def test_config5_coulomb_32_3x64_stochastic(cuda_device):
    """32^3 x 64 Coulomb gauge, fp64, stochastic relaxation p = 0.8, Philox seed 2013: the fix loop until
    theta_t < 1e-12 on every time slice, invariants at the end."""
    dims = (64, 32, 32, 32)
    U = gi.torch_smooth_random_gauge(dims, 0.6, 1, device=cuda_device)
    fld = gf.GaugeField(dims, gauge=gf.GF_COULOMB, precisions=("f64",), seed=2013, device=cuda_device)
    fld.pack(U, gf.GF_F64)
    del U
    P0 = fld.plaquette(gf.GF_F64)
    fld.iterate(1, gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64)          # compared link by link in tests/test_gpu_fullsize.py
    F1 = np.array(fld.functional(gf.GF_F64))
    rc, it, th = fld.fix_until(gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64, 1e-12, 100000, 20)
    assert rc == gf.GF_OK, (it, th)
    thetas = np.array(fld.theta(gf.GF_F64))
    assert thetas.shape == (64,) and thetas.max() < 1e-12 and thetas.max() == th
    assert (np.array(fld.functional(gf.GF_F64)) > F1).all()        # every slice's functional rose
    assert abs(fld.plaquette(gf.GF_F64) - P0) < 1e-12               # incl. temporal plaquettes: a gauge transformation
    du, dd = fld.unitarity(gf.GF_F64)
    assert du < 1e-12 and dd < 1e-12
    print("config5: %d iterations, max theta_t = %.3e" % (it, th))
    fld.close()


# ------------------------------------------- full-size checks of the SURVEY 8(f) features (NEXT-1..3)

def _gauge_transform_torch(U, G):
    """eq. 3 on the device with torch ops (test side only): G(x) U_mu(x) G(x+mu)^dagger."""
    out = torch.empty_like(U)
    for mu, axis in enumerate((0, 3, 2, 1)):          # canonical axes (t, z, y, x); mu = 0,1,2,3 = t,x,y,z
        Gf = torch.roll(G, -1, dims=axis)
        out[..., mu, :, :] = G @ U[..., mu, :, :] @ Gf.conj().transpose(-1, -2)
    return out


@pytest.mark.parametrize("prec,recon", [("f64", 18), ("f32", 12)])
def test_32_4_accumulated_transformation(cuda_device, prec, recon):
    """configs[2] size, default launch configuration with accumulation: U_n = G U_0 G^dagger over the whole
    lattice after 5 iterations (a property that holds at any size; eq. 3 restated with torch ops).  G(x) itself is
    compared with the oracle over the whole lattice in tests/test_gpu_fullsize.py."""
    dims = (32, 32, 32, 32)
    U0 = gi.torch_smooth_random_gauge(dims, 0.6, 1, device=cuda_device).to(CDTYPE[prec])
    fld = gf.GaugeField(dims, recon=recon, precisions=(prec,), device=cuda_device)
    fld.pack(U0, PREC[prec])
    fld.attach_transform((prec,))
    fld.iterate(5, gf.GF_OVERRELAX, 1.7, 0.0, PREC[prec])
    Un = fld.unpack(PREC[prec], torch.complex128)
    G = fld.transform(PREC[prec], torch.complex128)
    replay = _gauge_transform_torch(U0.to(torch.complex128), G)
    assert float((replay - Un).abs().max()) < (1e-12 if prec == "f64" else 2e-5)
    fld.close()


def test_config5_size_deferred_temporal_links_and_freezing(cuda_device):
    """32^3 x 64 Coulomb, fp64, stochastic p = 0.8: ten iterations with deferred temporal links equal
    ten plain iterations link by link (same Philox draws); the plaquette survives; a frozen slice is
    left alone."""
    dims = (64, 32, 32, 32)
    U = gi.torch_smooth_random_gauge(dims, 0.6, 1, device=cuda_device)
    plain = gf.GaugeField(dims, gauge=gf.GF_COULOMB, precisions=("f64",), seed=2013, device=cuda_device)
    plain.pack(U, gf.GF_F64)
    P0 = plain.plaquette(gf.GF_F64)
    plain.iterate(10, gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64)
    want = plain.unpack(gf.GF_F64)
    plain.close()
    fld = gf.GaugeField(dims, gauge=gf.GF_COULOMB, precisions=("f64",), seed=2013, device=cuda_device)
    fld.attach_transform(("f64",))
    fld.pack(U, gf.GF_F64)
    fld.set_coulomb_mode(defer_temporal=True)
    fld.iterate(10, gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64)
    got = fld.unpack(gf.GF_F64)                        # finishes the temporal links
    assert float((got - want).abs().max()) < 1e-11
    assert abs(fld.plaquette(gf.GF_F64) - P0) < 1e-13
    mask = [1] * 64
    mask[5] = mask[40] = 0
    fld.set_slice_mask(mask)
    fld.iterate(2, gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64)
    after = fld.unpack(gf.GF_F64)
    for t in (5, 40):
        assert torch.equal(after[t][..., 1:, :, :], got[t][..., 1:, :, :])
    assert not torch.equal(after[6][..., 1:, :, :], got[6][..., 1:, :, :])
    assert abs(fld.plaquette(gf.GF_F64) - P0) < 1e-13
    fld.close()


def test_32_4_as_two_slabs_equals_the_undivided_lattice(cuda_device):
    from paper_1305_3440_b200.slabs import SlabSet
    dims = (32, 32, 32, 32)
    U = gi.torch_smooth_random_gauge(dims, 0.6, 1, device=cuda_device)
    one = gf.GaugeField(dims, precisions=("f64",), seed=7, device=cuda_device)
    one.pack(U, gf.GF_F64)
    one.iterate(5, gf.GF_STOCHASTIC, 1.0, 0.5, gf.GF_F64)
    want = one.unpack(gf.GF_F64)
    Fw, thw = one.measure(gf.GF_F64)
    one.close()
    lat = SlabSet(dims, 2, seed=7, devices=(str(cuda_device),))
    lat.pack(U, gf.GF_F64)
    lat.iterate(5, gf.GF_STOCHASTIC, 1.0, 0.5, gf.GF_F64)
    F, th = lat.measure(gf.GF_F64)
    got = lat.unpack(gf.GF_F64)
    assert torch.equal(got, want)                     # same kernels, same order of operations per site: bitwise
    assert abs(F[0] - Fw[0]) < 1e-13 and abs(th[0] / thw[0] - 1) < 1e-12
    lat.close()


# ------------------------------------------------------------------------------ the paper's own per-GPU lattices

@pytest.mark.parametrize("dims,prec,recon", [((48, 48, 48, 48), "f64", 18), ((48, 48, 48, 48), "f32", 12),
                                             ((32, 64, 64, 64), "f64", 12), ((32, 64, 64, 64), "f32", 18),
                                             ((4, 128, 128, 128), "f64", 18), ((4, 128, 128, 128), "f32", 12)])
def test_fig3_lattices_sampled_against_oracle(cuda_device, dims, prec, recon):
    """48^4 and 64^3 x 32, the per-GPU lattices of the paper's weak-scaling figure, and 128^3 x 4, the
    largest time slice of its Tab. 1 (a temporal stride of a million sites): extents that are
    not powers of two at a size of several GB, default launch configuration.  One iteration with sampled sites
    recomputed by the oracle, then invariants after 20 more."""
    U = gi.torch_smooth_random_gauge(dims, 0.6, 48, device=cuda_device).to(CDTYPE[prec])
    fld = gf.GaugeField(dims, recon=recon, precisions=(prec,), device=cuda_device)
    fld.pack(U, PREC[prec])
    assert_pack_round_trip(fld, PREC[prec], U)      # sampled_sweep_check reads the oracle's input back from the device
    del U
    torch.cuda.empty_cache()
    P0 = fld.plaquette(PREC[prec])
    F0, th0 = fld.measure(PREC[prec])
    rng = np.random.default_rng(dims[0] + recon)
    sampled_sweep_check(fld, dims, prec, gf.GF_LANDAU, oracle.LANDAU, gf.GF_OVERRELAX, oracle.OVERRELAX, 1.7, 0.0, 0, 24, rng)
    torch.cuda.empty_cache()
    fld.iterate(20, gf.GF_OVERRELAX, 1.7, 0.0, PREC[prec])
    F1, th1 = fld.measure(PREC[prec])
    assert F1[0] > F0[0] and th1[0] < th0[0]
    assert abs(fld.plaquette(PREC[prec]) - P0) < (1e-12 if prec == "f64" else 1e-5)
    du, dd = fld.unitarity(PREC[prec])
    assert du < (1e-12 if prec == "f64" else 1e-4) and dd < (1e-12 if prec == "f64" else 1e-4)
    fld.close()
