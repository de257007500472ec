"""The fused iteration (gf_iterate's t-wavefront launch, include/gf.h) against the two separate
half-sweeps (bitwise) and against the CPU oracle."""
import numpy as np
import pytest
import torch

import gf_inputs as gi
import oracle
import paper_1305_3440_b200 as gf

pytestmark = pytest.mark.gpu

PREC = {"f64": gf.GF_F64, "f32": gf.GF_F32}
CDTYPE = {"f64": torch.complex128, "f32": torch.complex64}


def _field(dims, prec, recon, dev, gauge=gf.GF_LANDAU, seed=0):
    return gf.GaugeField(dims, gauge=gauge, recon=recon, precisions=(prec,), seed=seed, device=dev)


def streamed_ok(dims, prec):
    """include/gf.h: a layout tile (32 sites in fp64, 64 in fp32) is whole x-rows inside one plane."""
    nxh, W = dims[1] // 2, 32 if prec == "f64" else 64
    return W % nxh == 0 and (nxh * dims[2]) % W == 0


# (8,8,8,8): fp64 one tile per plane (fp32: not tileable); (4,16,16,16): several tiles per plane; (6,4,16,4): rows of 2
# sites; (4,64,2,4) / (4,128,2,4): a whole row per tile (the y-neighbours come from one other tile); (8,6,16,16): rows of
# 3 sites, odd; (4,4,4,4), (6,4,8,4), (8,12,8,8): not tileable
SHAPES = [(4, 4, 4, 4), (8, 8, 8, 8), (6, 4, 8, 4), (6, 4, 16, 4), (16, 8, 8, 8), (4, 16, 16, 16), (4, 64, 2, 4), (8, 12, 8, 8),
          (4, 32, 4, 2), (2, 8, 8, 8), (4, 128, 2, 4), (6, 4, 32, 2), (4, 8, 16, 6)]


@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("algo,omega,p", [(gf.GF_STOCHASTIC, 1.0, 0.6), (gf.GF_OVERRELAX, 1.7, 0.0)])
def test_fused_iterations_are_the_half_sweeps(cuda_device, dims, prec, recon, algo, omega, p):
    """gf_iterate with the fused launch against 2n gf_sweep launches of the register kernel with the same lanes per
    site (one in fp32, two in fp64): same arithmetic in the same order, so the links are compared bit for bit."""
    U = torch.from_numpy(gi.smooth_random_gauge(dims, 0.5, 23)).to(cuda_device).to(CDTYPE[prec]).contiguous()
    a = _field(dims, prec, recon, cuda_device, seed=5)
    b = _field(dims, prec, recon, cuda_device, seed=5)
    for f in (a, b):
        f.pack(U, PREC[prec])
        f.set_tuning(PREC[prec], 1 if prec == "f32" else 2, 64)
    a.set_wavefront(2)
    l0 = gf.gf_launch_count(a.ctx)
    a.iterate(7, algo, omega, p, PREC[prec])
    fused = gf.gf_launch_count(a.ctx) - l0 == 7
    assert fused == (streamed_ok(dims, prec) and dims[0] >= 4)              # otherwise it fell back to 14 half-sweeps
    for it in range(7):
        b.sweep(0, algo, omega, p, PREC[prec])
        b.sweep(1, algo, omega, p, PREC[prec])
    assert gf.gf_get_counter(a.ctx) == gf.gf_get_counter(b.ctx) == 14
    assert torch.equal(a.unpack(PREC[prec]), b.unpack(PREC[prec]))
    Fa, tha = a.measure(PREC[prec])                               # also checks that no tile gave up waiting
    Fb, thb = b.measure(PREC[prec])
    assert Fa == Fb and tha == thb
    a.close()
    b.close()


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (4, 16, 16, 16), (2, 8, 16, 8), (4, 64, 2, 4), (4, 128, 2, 2)])
@pytest.mark.parametrize("prec,recon", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
def test_streamed_half_sweeps_are_the_register_kernel(cuda_device, dims, prec, recon):
    """Mode 3: gf_sweep itself through the streamed kernel (one parity per launch, no dependencies)."""
    U = torch.from_numpy(gi.smooth_random_gauge(dims, 0.5, 27)).to(cuda_device).to(CDTYPE[prec]).contiguous()
    a = _field(dims, prec, recon, cuda_device, seed=9)
    b = _field(dims, prec, recon, cuda_device, seed=9)
    for f in (a, b):
        f.pack(U, PREC[prec])
        f.set_tuning(PREC[prec], 1 if prec == "f32" else 2, 64)
    a.set_wavefront(3)
    for k in range(3):
        for parity in (1, 0, 0):                                  # any order of parities, as gf_sweep allows
            a.sweep(parity, gf.GF_STOCHASTIC, 1.0, 0.5, PREC[prec])
            b.sweep(parity, gf.GF_STOCHASTIC, 1.0, 0.5, PREC[prec])
    assert gf.gf_get_counter(a.ctx) == gf.gf_get_counter(b.ctx) == 9
    assert torch.equal(a.unpack(PREC[prec]), b.unpack(PREC[prec]))
    a.close()
    b.close()


@pytest.mark.parametrize("lag,blocks", [(0, 0), (9, 3), (10, 1), (24, 148), (56, 7), (1000, 2)])
def test_fused_iteration_for_any_lag_and_block_count(cuda_device, lag, blocks):
    """The schedule is correct for every lag (clamped to Nz < lag <= (Nt-1) Nz) and any number of persistent blocks:
    the waits, not the order, carry the dependencies."""
    dims = (8, 8, 8, 8)
    U = torch.from_numpy(gi.smooth_random_gauge(dims, 0.5, 33)).to(cuda_device)
    a = _field(dims, "f64", 18, cuda_device, seed=4)
    b = _field(dims, "f64", 18, cuda_device, seed=4)
    for f in (a, b):
        f.pack(U, gf.GF_F64)
        f.set_tuning(gf.GF_F64, 2, 64)
    a.set_wavefront(2)
    a.set_wave_tuning(lag, blocks)
    a.iterate(4, gf.GF_STOCHASTIC, 1.0, 0.5, gf.GF_F64)
    b.iterate(4, gf.GF_STOCHASTIC, 1.0, 0.5, gf.GF_F64)
    assert torch.equal(a.unpack(gf.GF_F64), b.unpack(gf.GF_F64))
    a.close()
    b.close()


@pytest.mark.parametrize("gauge", [gf.GF_LANDAU, gf.GF_COULOMB])
def test_fused_iterations_match_oracle(cuda_device, gauge):
    dims = (8, 8, 8, 8)
    og = oracle.LANDAU if gauge == gf.GF_LANDAU else oracle.COULOMB
    U = gi.smooth_random_gauge(dims, 0.5, 29)
    fld = _field(dims, "f64", 18, cuda_device, gauge=gauge, seed=3)
    fld.pack(torch.from_numpy(U).to(cuda_device), gf.GF_F64)
    fld.set_wavefront(2)
    fld.iterate(1, gf.GF_STOCHASTIC, 1.0, 0.7, gf.GF_F64)
    Uo = U.copy()
    for parity in (0, 1):
        oracle.sweep(Uo, dims, parity, gauge=og, algo=oracle.STOCHASTIC, p=0.7, seed=3, half_sweep_counter=parity)
    assert np.abs(fld.unpack(gf.GF_F64).cpu().numpy() - Uo).max() < 1e-12
    fld.iterate(9, gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64)
    for _ in range(9):
        for parity in (0, 1):
            oracle.sweep(Uo, dims, parity, gauge=og, algo=oracle.OVERRELAX, omega=1.7)
    F, th = fld.measure(gf.GF_F64)
    assert np.allclose(F, oracle.functional(Uo, dims, og), rtol=1e-10)
    assert np.allclose(th, oracle.theta(Uo, dims, og), rtol=1e-10)
    fld.close()


def test_fused_iteration_eligibility_and_modes(cuda_device):
    """Contexts that are not eligible (slice mask, transformation buffer attached) fall back to two half-sweeps per
    iteration, silently and with the same links; the default is off."""
    dims = (8, 8, 8, 8)
    U = torch.from_numpy(gi.smooth_random_gauge(dims, 0.5, 31)).to(cuda_device)
    mask = [1, 1, 0, 1, 0, 0, 1, 1]
    a = _field(dims, "f64", 18, cuda_device, gauge=gf.GF_COULOMB)
    b = _field(dims, "f64", 18, cuda_device, gauge=gf.GF_COULOMB)
    for f in (a, b):
        f.pack(U, gf.GF_F64)
        f.set_tuning(gf.GF_F64, 2, 64)
    a.set_wavefront(2)
    b.set_wavefront(0)
    l0, l1 = gf.gf_launch_count(a.ctx), gf.gf_launch_count(b.ctx)
    a.iterate(5, gf.GF_OVERRELAX, 1.5, 0.0, gf.GF_F64)
    b.iterate(5, gf.GF_OVERRELAX, 1.5, 0.0, gf.GF_F64)
    assert gf.gf_launch_count(a.ctx) - l0 == 5 and gf.gf_launch_count(b.ctx) - l1 == 10
    assert torch.equal(a.unpack(gf.GF_F64), b.unpack(gf.GF_F64))
    for f in (a, b):
        f.set_slice_mask(mask)
    l0 = gf.gf_launch_count(a.ctx)
    a.iterate(3, gf.GF_OVERRELAX, 1.5, 0.0, gf.GF_F64)            # masked: not fused
    b.iterate(3, gf.GF_OVERRELAX, 1.5, 0.0, gf.GF_F64)
    assert gf.gf_launch_count(a.ctx) - l0 == 6
    assert torch.equal(a.unpack(gf.GF_F64), b.unpack(gf.GF_F64))
    a.set_slice_mask(None)
    c = _field(dims, "f64", 18, cuda_device)                      # default: off
    c.pack(U, gf.GF_F64)
    l0 = gf.gf_launch_count(c.ctx)
    c.iterate(3, gf.GF_RELAX, 1.0, 0.0, gf.GF_F64)
    assert gf.gf_launch_count(c.ctx) - l0 == 6
    c.close()
    a.attach_transform(("f64",))                                  # accumulation: not fused
    l0 = gf.gf_launch_count(a.ctx)
    a.iterate(2, gf.GF_OVERRELAX, 1.5, 0.0, gf.GF_F64)
    assert gf.gf_launch_count(a.ctx) - l0 == 4
    assert gf.binding.lib.gf_set_wavefront(a.ctx, 4) == gf.GF_EINVAL
    assert gf.binding.lib.gf_set_wave_tuning(a.ctx, -1, 0) == gf.GF_EINVAL
    a.close()
    b.close()
