"""GPU parity of the accumulated gauge transformation G(x) (eq. 3):
gf_set_transform / gf_sweep accumulation, gf_apply_transform and gf_fix_until(GF_MIXED_EXACT) against
the CPU oracle's sweep_accumulate / apply_transform on the same seeded inputs."""
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
GAUGE = {gf.GF_LANDAU: oracle.LANDAU, gf.GF_COULOMB: oracle.COULOMB}


def to_device(U, prec, dev):
    return torch.from_numpy(U).to(dev).to(CDTYPE[prec]).contiguous()


def rounded(U, prec):
    if prec == "f32":
        return np.ascontiguousarray(U.astype(np.complex64).astype(np.complex128))
    return U.copy()


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 6, 6), (6, 2, 4, 2), (8, 8, 8, 8)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("lanes", [1, 2, 4])
def test_accumulated_transformation_matches_oracle_after_one_sweep(cuda_device, dims, prec, recon, lanes):
    U = gi.smooth_random_gauge(dims, 0.5, 77)
    fld = gf.GaugeField(dims, recon=recon, precisions=(prec,), device=cuda_device)
    fld.pack(to_device(U, prec, cuda_device), PREC[prec])
    fld.attach_transform((prec,))
    fld.set_tuning(PREC[prec], lanes, 64)
    Uo, Go = rounded(U, prec), oracle.identity_transform(dims)
    for parity in (0, 1):
        fld.sweep(parity, gf.GF_OVERRELAX, 1.7, 0.0, PREC[prec])
        oracle.sweep_accumulate(Uo, Go, dims, parity, algo=oracle.OVERRELAX, omega=1.7)
        if parity == 0:      # the other parity has not been touched yet
            G = fld.transform(PREC[prec]).cpu().numpy()
            par = np.indices(G.shape[:4]).sum(axis=0) % 2
            assert np.all(G[par == 1] == np.eye(3))
    G = fld.transform(PREC[prec]).cpu().numpy()
    assert np.abs(G - Go).max() < TOL[prec]
    got = fld.unpack(PREC[prec], torch.complex128).cpu().numpy()
    assert np.abs(got - Uo).max() < TOL[prec]
    fld.close()


@pytest.mark.parametrize("gauge,algo", [(gf.GF_LANDAU, gf.GF_OVERRELAX), (gf.GF_COULOMB, gf.GF_STOCHASTIC)])
def test_transformation_reproduces_the_swept_links_after_ten_sweeps(cuda_device, gauge, algo):
    """The identity U_n = G U_0 G^dagger (eq. 3) on the device, through gf_apply_transform, and
    G against the oracle's after 10 iterations (fp64)."""
    dims = (8, 4, 6, 4)
    U = gi.smooth_random_gauge(dims, 0.5, 5)
    fld = gf.GaugeField(dims, gauge=gauge, precisions=("f64", "f32"), seed=9, device=cuda_device)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    fld.attach_transform(("f64",))
    fld.iterate(10, algo, 1.7, 0.8, gf.GF_F64)
    Uo, Go = U.copy(), oracle.identity_transform(dims)
    oalgo = oracle.OVERRELAX if algo == gf.GF_OVERRELAX else oracle.STOCHASTIC
    for it in range(10):
        for parity in (0, 1):
            oracle.sweep_accumulate(Uo, Go, dims, parity, gauge=GAUGE[gauge], algo=oalgo, omega=1.7, p=0.8, seed=9,
                                    half_sweep_counter=2 * it + parity)
    G = fld.transform(gf.GF_F64).cpu().numpy()
    assert np.abs(G - Go).max() < 1e-11
    swept = fld.unpack(gf.GF_F64, torch.complex128).cpu().numpy()
    # replay on the input: f64 input -> f32 slot of the context is not used; write into the f64 field itself
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    fld.apply_transform(gf.GF_F64, gf.GF_F64, gf.GF_F64)
    replay = fld.unpack(gf.GF_F64, torch.complex128).cpu().numpy()
    assert np.abs(replay - swept).max() < 1e-12
    assert np.abs(replay - oracle.apply_transform(U, Go, dims)).max() < 1e-11
    fld.close()


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("gprec,src,dst", [("f64", "f64", "f64"), ("f64", "f64", "f32"), ("f32", "f64", "f64"),
                                           ("f32", "f32", "f32"), ("f64", "f32", "f64")])
def test_apply_transform_matches_oracle(cuda_device, recon, gprec, src, dst):
    """gf_apply_transform for a Haar-random G against oracle.apply_transform; an fp32 G is compared
    with the oracle fed the fp32-rounded, re-projected G (Gram-Schmidt in numpy, fp64)."""
    dims = (4, 6, 4, 8)
    U = gi.smooth_random_gauge(dims, 0.4, 3)
    G = gi.random_gauge(dims, 11)
    fld = gf.GaugeField(dims, recon=recon, precisions=("f64", "f32"), device=cuda_device)
    fld.pack(to_device(U, src, cuda_device), PREC[src])
    fld.attach_transform(("f64", "f32"))
    fld.set_transform(to_device(G, gprec, cuda_device), PREC[gprec])
    fld.apply_transform(PREC[gprec], PREC[src], PREC[dst])
    got = fld.unpack(PREC[dst], torch.complex128).cpu().numpy()
    Gr = rounded(G, gprec)
    if gprec == "f32":
        Gr = _gram_schmidt(Gr)
    want = oracle.apply_transform(rounded(U, src), np.ascontiguousarray(Gr), dims)
    # an fp32 source stored as 12 reals has its third row rebuilt from fp32 rows: fp32-level agreement
    exact = dst == "f64" and (src == "f64" or recon == 18)
    assert np.abs(got - want).max() < (1e-12 if exact else 1e-6)
    if dst == "f64":
        du, dd = fld.unitarity(gf.GF_F64)
        assert du < (1e-12 if src == "f64" else 1e-6)
    fld.close()


def _gram_schmidt(G):
    r0 = G[..., 0, :] / np.linalg.norm(G[..., 0, :], axis=-1, keepdims=True)
    r1 = G[..., 1, :] - np.sum(r0.conj() * G[..., 1, :], axis=-1, keepdims=True) * r0
    r1 = r1 / np.linalg.norm(r1, axis=-1, keepdims=True)
    r2 = np.conj(np.cross(r0, r1))
    return np.stack([r0, r1, r2], axis=-2)


def test_transform_cast_and_identity(cuda_device):
    dims = (4, 4, 4, 4)
    G = gi.random_gauge(dims, 2)
    fld = gf.GaugeField(dims, precisions=("f64", "f32"), device=cuda_device)
    fld.attach_transform(("f64", "f32"))
    assert np.all(fld.transform(gf.GF_F64).cpu().numpy() == np.eye(3))
    fld.set_transform(to_device(G, "f32", cuda_device), gf.GF_F32)
    fld.transform_cast(gf.GF_F32, gf.GF_F64)
    G64 = fld.transform(gf.GF_F64).cpu().numpy()
    assert np.abs(G64 - G).max() < 1e-6
    GG = np.einsum("...ab,...cb->...ac", G64, G64.conj())
    assert np.abs(GG - np.eye(3)).max() < 1e-14 and np.abs(np.linalg.det(G64) - 1).max() < 1e-14
    fld.transform_identity(gf.GF_F64)
    assert np.all(fld.transform(gf.GF_F64).cpu().numpy() == np.eye(3))
    # errors: no buffer for that precision
    fld.attach_transform(("f64",))
    assert gf.binding.lib.gf_transform_identity(fld.ctx, gf.GF_F32) == gf.GF_ESTATE
    assert gf.binding.lib.gf_fix_until(fld.ctx, gf.GF_RELAX, 1.0, 0.0, gf.GF_MIXED_EXACT, 1e-12, 10, 1, None, None) == gf.GF_ESTATE
    fld.close()


@pytest.mark.parametrize("recon", [18, 12])
def test_mixed_exact_fix_is_gauge_equivalent_to_the_input_at_fp64_accuracy(cuda_device, recon):
    """GF_MIXED_EXACT: fp32 sweeps record G, the fp64 input is transformed by the re-projected G, fp64
    sweeps finish.  Unlike GF_MIXED the plaquette is kept to 1e-13, and the returned G maps the input
    onto the result (checked with the oracle's eq. 3)."""
    dims = (8, 8, 8, 8)
    U = gi.smooth_random_gauge(dims, 0.5, 1234)
    fld = gf.GaugeField(dims, recon=recon, precisions=("f32", "f64"), device=cuda_device)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    fld.attach_transform(("f64", "f32"))
    P0 = fld.plaquette(gf.GF_F64)
    rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_MIXED_EXACT, 1e-12, 20000, 10)
    assert rc == gf.GF_OK and th < 1e-12
    du, dd = fld.unitarity(gf.GF_F64)
    assert du < 1e-12 and dd < 1e-12
    assert abs(fld.plaquette(gf.GF_F64) - P0) < 1e-13
    Ug = fld.unpack(gf.GF_F64, torch.complex128).cpu().numpy()
    G = fld.transform(gf.GF_F64).cpu().numpy()
    assert np.abs(oracle.apply_transform(U, np.ascontiguousarray(G), dims) - Ug).max() < 1e-11
    assert oracle.theta(np.ascontiguousarray(Ug), dims) < 1.1e-12
    # the fp64-only run needs about the same number of iterations: the fp32 phase did real work
    fld2 = gf.GaugeField(dims, recon=recon, precisions=("f64",), device=cuda_device)
    fld2.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    rc2, it2, _ = fld2.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64, 1e-12, 20000, 10)
    assert rc2 == gf.GF_OK and abs(it - it2) <= 0.2 * it2 + 20
    fld.close()
    fld2.close()


def test_mixed_handoff_knob(cuda_device):
    """gf_set_mixed_handoff: a later hand-off moves iterations into the fp32 phase; GF_MIXED_EXACT still
    returns a field gauge equivalent to the input at fp64 accuracy."""
    dims = (8, 8, 8, 8)
    U = gi.smooth_random_gauge(dims, 0.5, 1234)
    fld = gf.GaugeField(dims, precisions=("f32", "f64"), device=cuda_device)
    fld.attach_transform(("f64", "f32"))
    assert gf.binding.lib.gf_set_mixed_handoff(fld.ctx, 0.0) == gf.GF_EINVAL
    fld.set_mixed_handoff(1e-10)
    fld.pack(to_device(U, "f64", cuda_device), gf.GF_F64)
    P0 = fld.plaquette(gf.GF_F64)
    c0 = gf.gf_launch_count(fld.ctx)
    rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_MIXED_EXACT, 1e-12, 20000, 10)
    assert rc == gf.GF_OK and th < 1e-12
    assert abs(fld.plaquette(gf.GF_F64) - P0) < 1e-13
    Ug = fld.unpack(gf.GF_F64, torch.complex128).cpu().numpy()
    G = fld.transform(gf.GF_F64).cpu().numpy()
    assert np.abs(oracle.apply_transform(U, np.ascontiguousarray(G), dims) - Ug).max() < 1e-11
    assert oracle.theta(np.ascontiguousarray(Ug), dims) < 1.1e-12
    fld.close()
