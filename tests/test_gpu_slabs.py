"""GPU parity of the slab decomposition along t (gf_set_slab): several slabs of one
lattice, each with its own context and stream, sharing the boundary temporal links in place, driven
from one process on one GPU, against the CPU oracle's sweeps of the undivided lattice."""
import numpy as np
import pytest
import torch

import gf_inputs as gi
import oracle
import paper_1305_3440_b200 as gf
from paper_1305_3440_b200.slabs import SlabSet, local_dims, neighbours

pytestmark = pytest.mark.gpu

PREC = {"f64": gf.GF_F64, "f32": gf.GF_F32}
CDTYPE = {"f64": torch.complex128, "f32": torch.complex64}


def rounded(U, prec):
    if prec == "f32":
        return np.ascontiguousarray(U.astype(np.complex64).astype(np.complex128))
    return U.copy()


@pytest.mark.parametrize("dims,nslabs", [((8, 4, 4, 4), 2), ((8, 4, 6, 6), 4), ((12, 6, 6, 6), 3), ((4, 4, 4, 4), 2)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("recon", [18, 12])
def test_slabs_one_sweep_links_match_oracle(cuda_device, dims, nslabs, prec, recon):
    U = gi.smooth_random_gauge(dims, 0.5, 41)
    lat = SlabSet(dims, nslabs, recon=recon, precisions=(prec,), seed=12, devices=(str(cuda_device),))
    lat.pack(torch.from_numpy(U).to(cuda_device).to(CDTYPE[prec]), PREC[prec])
    Uo = rounded(U, prec)
    P0 = oracle.plaquette(Uo, dims)
    assert abs(lat.plaquette(PREC[prec]) - P0) < (1e-13 if prec == "f64" else 1e-6)      # crosses the slab boundaries
    F, th = lat.measure(PREC[prec])
    # (fp32 fields stored as 12 reals rebuild the third row in fp32)
    assert abs(F[0] - oracle.functional(Uo, dims)) < (1e-12 if prec == "f64" else 1e-6)
    assert abs(th[0] / oracle.theta(Uo, dims) - 1) < (1e-9 if prec == "f64" else 1e-4)
    for parity in (0, 1):
        lat.sweep(parity, gf.GF_STOCHASTIC, 1.0, 0.6, PREC[prec])
        oracle.sweep(Uo, dims, parity, algo=oracle.STOCHASTIC, p=0.6, seed=12, half_sweep_counter=parity)
    got = lat.unpack(PREC[prec]).cpu().numpy()
    assert np.abs(got - Uo).max() < (1e-12 if prec == "f64" else 1e-5)
    lat.close()


@pytest.mark.parametrize("gauge", [gf.GF_LANDAU, gf.GF_COULOMB])
def test_slabs_ten_sweeps_F_theta_match_oracle(cuda_device, gauge):
    dims, nslabs = (8, 6, 4, 6), 2
    og = oracle.LANDAU if gauge == gf.GF_LANDAU else oracle.COULOMB
    U = gi.smooth_random_gauge(dims, 0.5, 42)
    lat = SlabSet(dims, nslabs, gauge=gauge, devices=(str(cuda_device),))
    lat.pack(torch.from_numpy(U).to(cuda_device), gf.GF_F64)
    lat.iterate(10, gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64)
    Uo = U.copy()
    for _ in range(10):
        for parity in (0, 1):
            oracle.sweep(Uo, dims, parity, gauge=og, algo=oracle.OVERRELAX, omega=1.7)
    F, th = lat.measure(gf.GF_F64)
    assert np.allclose(F, oracle.functional(Uo, dims, og), rtol=1e-10)
    assert np.allclose(th, oracle.theta(Uo, dims, og), rtol=1e-10)
    assert abs(lat.plaquette(gf.GF_F64) - oracle.plaquette(U, dims)) < 1e-13
    got = lat.unpack(gf.GF_F64).cpu().numpy()
    assert np.abs(got - Uo).max() < 1e-11
    lat.close()


def test_slabs_fix_until_matches_the_undivided_run(cuda_device):
    dims = (8, 4, 4, 4)
    U = gi.smooth_random_gauge(dims, 0.3, 3)
    lat = SlabSet(dims, 2, devices=(str(cuda_device),))
    lat.pack(torch.from_numpy(U).to(cuda_device), gf.GF_F64)
    rc, it, th = lat.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64, 1e-12, 2000, 1)
    Uo = U.copy()
    it_o, th_o, conv = oracle.fix_until(Uo, dims, algo=oracle.OVERRELAX, omega=1.7, theta_target=1e-12, max_iter=2000)
    assert rc == gf.GF_OK and conv and abs(it - it_o) <= 1 and th < 1e-12
    got = lat.unpack(gf.GF_F64).cpu().numpy()
    assert oracle.theta(np.ascontiguousarray(got), dims) < 1.1e-12
    du, dd = lat.unitarity(gf.GF_F64)
    assert du < 1e-12 and dd < 1e-12
    lat.close()


def test_slab_argument_errors(cuda_device):
    B = gf.binding.lib
    f = gf.GaugeField((4, 4, 4, 4), precisions=("f64",), device=cuda_device)
    flag = torch.zeros(4, dtype=torch.int32, device=cuda_device)
    assert B.gf_set_slab(f.ctx, 2, 2, None, None, None, None, None, None, None) == gf.GF_EINVAL          # rank out of range
    assert B.gf_set_slab(f.ctx, 0, 2, None, None, None, None, flag.data_ptr(), flag.data_ptr(), flag.data_ptr()) == gf.GF_EINVAL
    p = f._bufs[gf.GF_F64].data_ptr()
    assert B.gf_set_slab(f.ctx, 0, 2, p, None, p, None, flag.data_ptr(), flag.data_ptr(), flag.data_ptr()) == gf.GF_OK
    assert B.gf_fix_until(f.ctx, gf.GF_RELAX, 1.0, 0.0, gf.GF_F64, 1e-12, 10, 1, None, None) == gf.GF_ESTATE
    assert B.gf_set_slab(f.ctx, 0, 1, None, None, None, None, None, None, None) == gf.GF_OK               # back to one lattice
    f.close()
    with pytest.raises(ValueError):
        local_dims((6, 4, 4, 4), 2)          # slabs of odd length would break the checkerboard
    assert neighbours(0, 4) == (3, 1) and neighbours(3, 4) == (2, 0)
