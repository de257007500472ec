"""GPU parity of the Coulomb-gauge specialisation: deferred temporal links
(gf_set_coulomb_mode / gf_coulomb_finish) and slice freezing (gf_set_slice_mask, gf_fix_until with
freeze_slices) against the CPU oracle's plain and masked sweeps on the same seeded inputs."""
import numpy as np
import pytest
import torch

import gf_inputs as gi
import oracle
import paper_1305_3440_b200 as gf

pytestmark = pytest.mark.gpu

PREC = {"f64": gf.GF_F64, "f32": gf.GF_F32}
TOL = {"f64": 1e-12, "f32": 1e-5}
CDTYPE = {"f64": torch.complex128, "f32": torch.complex64}


def to_device(U, prec, dev):
    return torch.from_numpy(U).to(dev).to(CDTYPE[prec]).contiguous()


def rounded(U, prec):
    if prec == "f32":
        return np.ascontiguousarray(U.astype(np.complex64).astype(np.complex128))
    return U.copy()


def coulomb_field(dims, prec, dev, recon=18, seed=0, transform=True):
    fld = gf.GaugeField(dims, gauge=gf.GF_COULOMB, recon=recon, precisions=(prec,), seed=seed, device=dev)
    if transform:
        fld.attach_transform((prec,))
    return fld


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 6, 6), (2, 2, 2, 2), (8, 8, 8, 8)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("lanes", [1, 2, 4])
def test_deferred_temporal_links_one_sweep_matches_oracle(cuda_device, dims, prec, recon, lanes):
    """One iteration with the temporal links deferred, then gf_coulomb_finish: the complete field
    equals the oracle's plain Coulomb sweep; before the finish the temporal links are untouched and
    the spatial ones already final."""
    U = gi.smooth_random_gauge(dims, 0.5, 13)
    fld = coulomb_field(dims, prec, cuda_device, recon=recon, seed=4)
    fld.pack(to_device(U, prec, cuda_device), PREC[prec])
    before = fld.unpack(PREC[prec], torch.complex128).cpu().numpy()
    fld.set_coulomb_mode(defer_temporal=True)
    fld.set_tuning(PREC[prec], lanes, 64)
    Uo = rounded(U, prec)
    for parity in (0, 1):
        fld.sweep(parity, gf.GF_STOCHASTIC, 1.0, 0.7, PREC[prec])
        oracle.sweep(Uo, dims, parity, gauge=oracle.COULOMB, algo=oracle.STOCHASTIC, p=0.7, seed=4, half_sweep_counter=parity)
    F, th = fld.measure(PREC[prec])                      # independent of the temporal links
    assert np.allclose(th, oracle.theta(Uo, dims, oracle.COULOMB), rtol=1e-3 if prec == "f32" else 1e-9, atol=1e-14)
    # peek at the raw field without finishing: read the internal buffer through a second context
    raw = gf.GaugeField(dims, gauge=gf.GF_COULOMB, recon=recon, precisions=(prec,), device=cuda_device)
    raw._bufs[PREC[prec]].copy_(fld._bufs[PREC[prec]])
    pending = raw.unpack(PREC[prec], torch.complex128).cpu().numpy()
    assert np.array_equal(pending[..., 0, :, :], before[..., 0, :, :])
    assert np.abs(pending[..., 1:, :, :] - Uo[..., 1:, :, :]).max() < TOL[prec]
    raw.close()
    got = fld.unpack(PREC[prec], torch.complex128).cpu().numpy()          # finishes by itself
    assert np.abs(got - Uo).max() < TOL[prec]
    again = fld.unpack(PREC[prec], torch.complex128).cpu().numpy()        # and only once
    assert np.array_equal(again, got)
    fld.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_deferred_temporal_links_ten_sweeps_and_restart(cuda_device, prec):
    """10 deferred iterations, finish, 5 more, finish: links vs the oracle's 15 plain iterations; the
    plaquette (which sees the temporal links) is the input's."""
    dims = (6, 6, 4, 4)
    U = gi.smooth_random_gauge(dims, 0.5, 14)
    fld = coulomb_field(dims, prec, cuda_device)
    fld.pack(to_device(U, prec, cuda_device), PREC[prec])
    P0 = fld.plaquette(PREC[prec])
    fld.set_coulomb_mode(defer_temporal=True)
    Uo = rounded(U, prec)
    fld.iterate(10, gf.GF_OVERRELAX, 1.6, 0.0, PREC[prec])
    fld.coulomb_finish(PREC[prec])
    fld.iterate(5, gf.GF_OVERRELAX, 1.6, 0.0, PREC[prec])
    for it in range(15):
        for parity in (0, 1):
            oracle.sweep(Uo, dims, parity, gauge=oracle.COULOMB, algo=oracle.OVERRELAX, omega=1.6)
    assert abs(fld.plaquette(PREC[prec]) - P0) < (1e-13 if prec == "f64" else 1e-6)
    got = fld.unpack(PREC[prec], torch.complex128).cpu().numpy()
    assert np.abs(got - Uo).max() < (1e-11 if prec == "f64" else 2e-4)
    F, th = fld.measure(PREC[prec])
    rel = 1e-10 if prec == "f64" else 1e-4
    assert np.allclose(F, oracle.functional(Uo, dims, oracle.COULOMB), rtol=rel)
    assert np.allclose(th, oracle.theta(Uo, dims, oracle.COULOMB), rtol=100 * rel)
    fld.close()


@pytest.mark.parametrize("defer", [False, True])
@pytest.mark.parametrize("lanes", [1, 2, 4])
def test_slice_mask_matches_oracle_masked_sweep(cuda_device, defer, lanes):
    dims = (6, 4, 4, 6)          # Sh = 48 sites per slice and parity: warps straddle slice boundaries
    mask = [1, 0, 1, 1, 0, 0]
    U = gi.smooth_random_gauge(dims, 0.5, 15)
    fld = coulomb_field(dims, "f64", cuda_device, seed=6)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    fld.set_coulomb_mode(defer_temporal=defer)
    fld.set_tuning(gf.GF_F64, lanes, 64)
    fld.set_slice_mask(mask)
    Uo = U.copy()
    for it in range(3):
        for parity in (0, 1):
            fld.sweep(parity, gf.GF_STOCHASTIC, 1.0, 0.5, gf.GF_F64)
            oracle.sweep_masked(Uo, dims, parity, mask, algo=oracle.STOCHASTIC, p=0.5, seed=6, half_sweep_counter=2 * it + parity)
    got = fld.unpack(gf.GF_F64, torch.complex128).cpu().numpy()
    assert np.abs(got - Uo).max() < 1e-12
    for t in (1, 4, 5):
        assert np.array_equal(got[t][..., 1:, :, :], U[t][..., 1:, :, :])
    fld.set_slice_mask(None)
    fld.sweep(0, gf.GF_RELAX, 1.0, 0.0, gf.GF_F64)
    oracle.sweep(Uo, dims, 0, gauge=oracle.COULOMB, algo=oracle.RELAX)
    got = fld.unpack(gf.GF_F64, torch.complex128).cpu().numpy()
    assert np.abs(got - Uo).max() < 1e-12
    fld.close()


@pytest.mark.parametrize("defer", [False, True])
def test_fix_until_with_freezing_matches_oracle(cuda_device, defer):
    dims = (6, 4, 4, 6)
    U = gi.smooth_random_gauge(dims, 0.4, 31)
    fld = coulomb_field(dims, "f64", cuda_device)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    P0 = fld.plaquette(gf.GF_F64)
    fld.set_coulomb_mode(defer_temporal=defer, freeze_slices=True)
    rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.6, 0.0, gf.GF_F64, 1e-12, 3000, 1)
    Uo = U.copy()
    it_o, th_o, frozen_at, conv = oracle.fix_until_freeze(Uo, dims, algo=oracle.OVERRELAX, omega=1.6, theta_target=1e-12,
                                                          max_iter=3000, check_every=1)
    assert rc == gf.GF_OK and conv and abs(it - it_o) <= 1 and th < 1e-12
    got = fld.unpack(gf.GF_F64, torch.complex128).cpu().numpy()
    if it == it_o:
        # spatial links: slice by slice the same trajectory, frozen at the same iteration (unless a
        # theta_t crossed the target within rounding, which the iteration count would show)
        assert np.abs(got[..., 1:, :, :] - Uo[..., 1:, :, :]).max() < 1e-10
    _, tht = fld.measure(gf.GF_F64)
    assert max(tht) < 1e-12 and oracle.theta(np.ascontiguousarray(got), dims, oracle.COULOMB).max() < 1.1e-12
    assert abs(fld.plaquette(gf.GF_F64) - P0) < 1e-13
    du, dd = fld.unitarity(gf.GF_F64)
    assert du < 1e-12 and dd < 1e-12
    fld.close()


def mixed_smoothness_field(dims, seed):
    """Time slices of very different smoothness (eps 0.05 ... 0.6), hence very different convergence times in Coulomb
    gauge: slice t of the input is slice t of one of four seeded smooth fields.  Any SU(3) link field is a valid input."""
    fields = [gi.smooth_random_gauge(dims, eps, seed + k) for k, eps in enumerate((0.05, 0.2, 0.4, 0.6))]
    U = np.empty_like(fields[0])
    for t in range(dims[0]):
        U[t] = fields[(t * 7 + t // 3) % 4][t]
    return U


@pytest.mark.parametrize("defer", [False, True])
@pytest.mark.parametrize("recon", [18, 12])
def test_slices_converging_at_different_times(cuda_device, defer, recon):
    """NEXT-2, "batching slices with different convergence": with freeze_slices the half-sweeps cover the list of
    still-active slices only.  On an input whose slices converge at very different iterations the run stops at the
    oracle's iteration, every slice on the oracle's (frozen) trajectory."""
    dims = (12, 6, 4, 6)
    U = mixed_smoothness_field(dims, 40)
    Uo = U.copy()
    it_o, th_o, frozen_at, conv = oracle.fix_until_freeze(Uo, dims, algo=oracle.OVERRELAX, omega=1.5, theta_target=1e-12,
                                                          max_iter=5000, check_every=5)
    assert conv and frozen_at.max() > 2 * frozen_at.min() and len(set(frozen_at.tolist())) >= 4    # really staggered
    fld = coulomb_field(dims, "f64", cuda_device, recon=recon)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    fld.set_coulomb_mode(defer_temporal=defer, freeze_slices=True)
    launches0 = gf.gf_launch_count(fld.ctx)
    rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.5, 0.0, gf.GF_F64, 1e-12, 5000, 5)
    assert rc == gf.GF_OK and th < 1e-12 and abs(it - it_o) <= 5
    got = fld.unpack(gf.GF_F64, torch.complex128).cpu().numpy()
    if it == it_o:
        assert np.abs(got[..., 1:, :, :] - Uo[..., 1:, :, :]).max() < 1e-10
    assert oracle.theta(np.ascontiguousarray(got), dims, oracle.COULOMB).max() < 1.1e-12
    assert abs(oracle.plaquette(np.ascontiguousarray(got), dims) - oracle.plaquette(U, dims)) < 1e-12
    fld.close()


def test_all_slices_frozen_launches_nothing_and_keeps_the_philox_counter(cuda_device):
    dims = (4, 4, 4, 4)
    U = gi.smooth_random_gauge(dims, 0.5, 3)
    fld = coulomb_field(dims, "f64", cuda_device, seed=9, transform=False)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    fld.set_slice_mask([0, 0, 0, 0])
    n0 = gf.gf_launch_count(fld.ctx)
    fld.iterate(2, gf.GF_STOCHASTIC, 1.0, 0.5, gf.GF_F64)
    assert gf.gf_launch_count(fld.ctx) == n0 and gf.gf_get_counter(fld.ctx) == 4
    assert np.array_equal(fld.unpack(gf.GF_F64, torch.complex128).cpu().numpy(), U)
    fld.set_slice_mask([0, 0, 1, 0])                       # one slice, the last position of a one-entry list
    fld.sweep(0, gf.GF_STOCHASTIC, 1.0, 0.5, gf.GF_F64)
    Uo = U.copy()
    oracle.sweep_masked(Uo, dims, 0, [0, 0, 1, 0], algo=oracle.STOCHASTIC, p=0.5, seed=9, half_sweep_counter=4)
    assert np.abs(fld.unpack(gf.GF_F64, torch.complex128).cpu().numpy() - Uo).max() < 1e-12
    fld.close()


def test_half_sweep_time_follows_the_number_of_active_slices(cuda_device):
    """configs[4] size: with 4 of 64 slices active a half-sweep costs a small fraction of the full one (the launch covers
    the listed slices only; a byte mask consulted by every warp of a full grid took 0.12 of the full time)."""
    dims = (64, 32, 32, 32)
    fld = coulomb_field(dims, "f64", cuda_device, transform=False)
    fld.pack(gi.torch_smooth_random_gauge(dims, 0.6, 1, device=cuda_device), gf.GF_F64)

    def ms(mask, n=20):
        fld.set_slice_mask(mask)
        fld.iterate(3, gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fld.iterate(n, gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64)
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n

    full = ms(None)
    few = ms([1 if t % 16 == 5 else 0 for t in range(64)])
    print("32^3 x 64 fp64: %.4f ms per iteration with 64 active slices, %.4f ms with 4" % (full, few))
    assert few < 0.10 * full                                # 4 / 64 = 0.0625 of the sites; measured 0.065
    fld.close()


def test_coulomb_mode_errors(cuda_device):
    dims = (4, 4, 4, 4)
    B = gf.binding.lib
    lan = gf.GaugeField(dims, precisions=("f64",), device=cuda_device)
    assert B.gf_set_coulomb_mode(lan.ctx, 1, 0) == gf.GF_EINVAL
    assert B.gf_set_coulomb_mode(lan.ctx, 0, 0) == gf.GF_OK
    lan.close()
    cou = gf.GaugeField(dims, gauge=gf.GF_COULOMB, precisions=("f64",), device=cuda_device)
    cou.pack(to_device(gi.smooth_random_gauge(dims, 0.3, 1), "f64", cuda_device), gf.GF_F64)
    assert B.gf_set_coulomb_mode(cou.ctx, 1, 2) == gf.GF_EINVAL
    assert B.gf_set_coulomb_mode(cou.ctx, 1, 0) == gf.GF_OK
    assert B.gf_sweep(cou.ctx, 0, gf.GF_RELAX, 1.0, 0.0, gf.GF_F64) == gf.GF_ESTATE        # no transformation buffer
    assert B.gf_fix_until(cou.ctx, gf.GF_RELAX, 1.0, 0.0, gf.GF_F64, 1e-12, 10, 1, None, None) == gf.GF_ESTATE
    assert gf.gf_get_counter(cou.ctx) == 0
    cou.close()
