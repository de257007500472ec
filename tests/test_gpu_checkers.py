"""The GPU-side checkers and projections are themselves checked: gf_unitarity against the oracle's
unitarity_defect on fields that are NOT unitary (both outputs), gf_reunitarize and the fp32 -> fp64 cast against
the definition of the projection (Gram-Schmidt on rows 0 and 1, row 2 = conj(row 0 x row 1), restated in numpy
here) with the result judged by the oracle.  A unitarity kernel that returned zeros, or a projection that left the
links alone, fails here."""
import numpy as np
import pytest
import torch

import gf_inputs as gi
import oracle
import paper_1305_3440_b200 as gf

pytestmark = pytest.mark.gpu

PREC = {"f64": gf.GF_F64, "f32": gf.GF_F32}
CDTYPE = {"f64": torch.complex128, "f32": torch.complex64}
DIMS = (4, 6, 8, 10)          # V/2 = 960 sites per parity: several blocks and a ragged tail


def perturbed_field(dims, seed, noise):
    U = gi.hot_links(dims, seed)
    rng = np.random.default_rng(seed + 1)
    return np.ascontiguousarray(U + noise * (rng.standard_normal(U.shape) + 1j * rng.standard_normal(U.shape)))


def gram_schmidt_su3(U):
    """Definition of the projection (reading A15/A18): row 0 normalised; row 1 minus its component along
    row 0, normalised; row 2 = conj(row 0 x row 1)."""
    r0 = U[..., 0, :] / np.linalg.norm(U[..., 0, :], axis=-1, keepdims=True)
    r1 = U[..., 1, :] - np.sum(r0.conj() * U[..., 1, :], axis=-1, keepdims=True) * r0
    r1 = r1 / np.linalg.norm(r1, axis=-1, keepdims=True)
    r2 = np.conj(np.cross(r0, r1))
    return np.stack([r0, r1, r2], axis=-2)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("recon", [18, 12])
def test_unitarity_matches_the_oracle_on_a_non_unitary_field(cuda_device, prec, recon):
    U = perturbed_field(DIMS, 3, 1e-3)
    flat = U.reshape(-1, 4, 3, 3)
    flat[11, 2] *= 1.05                                   # one link far off: |U U^dagger - 1| = 0.1025, det = 1.157..
    flat[-1, 3][[0, 1]] = flat[-1, 3][[1, 0]]             # last link of the field: rows swapped, det ~ -1
    fld = gf.GaugeField(DIMS, recon=recon, precisions=(prec,), device=cuda_device)
    fld.pack(torch.from_numpy(U).to(cuda_device).to(CDTYPE[prec]), PREC[prec])
    held = fld.unpack(PREC[prec], torch.complex128).cpu().numpy()      # what the device holds (12-real: row 2 rebuilt)
    want = oracle.unitarity_defect(np.ascontiguousarray(held), DIMS)
    got = fld.unitarity(PREC[prec])
    tol = 1e-12 if (prec == "f64" or recon == 18) else 1e-6            # fp32 12-real: row 2 is rebuilt in fp32 twice
    assert want[0] > 0.05 and want[1] > 0.1                            # the defects are really there
    assert abs(got[0] - want[0]) < tol * max(1.0, want[0]), (got, want)
    assert abs(got[1] - want[1]) < tol * max(1.0, want[1]), (got, want)
    if recon == 18:
        assert abs(want[1] - 2.0) < 0.02                               # the swapped rows dominate the determinant defect
    # the two outputs separately: a field whose only defect is in the determinant, and one that is fine
    V = gi.hot_links(DIMS, 5)
    if recon == 18:
        V.reshape(-1, 4, 3, 3)[500, 1] *= np.exp(0.3j)
        fld.pack(torch.from_numpy(V).to(cuda_device).to(CDTYPE[prec]), PREC[prec])
        du, dd = fld.unitarity(PREC[prec])
        eps = 1e-13 if prec == "f64" else 1e-6
        assert du < eps and abs(dd - 2 * np.sin(0.45)) < eps
    fld.pack(torch.from_numpy(gi.hot_links(DIMS, 5)).to(cuda_device).to(CDTYPE[prec]), PREC[prec])
    du, dd = fld.unitarity(PREC[prec])
    assert du < (1e-13 if prec == "f64" else 1e-6) and dd < (1e-13 if prec == "f64" else 1e-6)
    fld.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("recon", [18, 12])
def test_reunitarize_is_gram_schmidt_and_lands_in_SU3(cuda_device, prec, recon):
    U = perturbed_field(DIMS, 7, 1e-3)
    fld = gf.GaugeField(DIMS, recon=recon, precisions=(prec,), device=cuda_device)
    fld.pack(torch.from_numpy(U).to(cuda_device).to(CDTYPE[prec]), PREC[prec])
    held = fld.unpack(PREC[prec], torch.complex128).cpu().numpy()
    assert oracle.unitarity_defect(np.ascontiguousarray(held), DIMS)[0] > (1e-3 if recon == 18 else 1e-4)
    gf.gf_reunitarize(fld.ctx, PREC[prec])
    got = fld.unpack(PREC[prec], torch.complex128).cpu().numpy()
    want = gram_schmidt_su3(held)                                      # from rows 0, 1 of what the device held
    tol = 1e-13 if prec == "f64" else 5e-7                             # the projection runs in fp64, the store rounds
    assert np.abs(got - want).max() < tol
    du, dd = oracle.unitarity_defect(np.ascontiguousarray(got), DIMS)  # judged by the oracle
    assert du < (1e-14 if prec == "f64" else 1e-6) and dd < (1e-14 if prec == "f64" else 1e-6)
    # row 0 keeps its direction, row 2 is the conjugate cross product of the new rows 0 and 1
    cosang = np.abs(np.sum(got[..., 0, :].conj() * held[..., 0, :], axis=-1)) / np.linalg.norm(held[..., 0, :], axis=-1)
    assert np.abs(cosang - 1).max() < (1e-14 if prec == "f64" else 1e-6)
    assert np.abs(got[..., 2, :] - np.conj(np.cross(got[..., 0, :], got[..., 1, :]))).max() < (1e-14 if prec == "f64" else 1e-6)
    # the device checker agrees with the oracle on the projected field too
    gdu, gdd = fld.unitarity(PREC[prec])
    assert abs(gdu - du) < (1e-14 if prec == "f64" else 1e-6) and abs(gdd - dd) < (1e-14 if prec == "f64" else 1e-6)
    fld.close()


@pytest.mark.parametrize("recon", [18, 12])
def test_cast_f32_to_f64_reprojects_and_f64_to_f32_rounds(cuda_device, recon):
    """gf_cast fp32 -> fp64 is the mixed-precision hand-off (reading A15): every link is re-projected in fp64."""
    U = perturbed_field(DIMS, 9, 1e-3)
    fld = gf.GaugeField(DIMS, recon=recon, precisions=("f32", "f64"), device=cuda_device)
    fld.pack(torch.from_numpy(U).to(cuda_device).to(torch.complex64), gf.GF_F32)
    held = fld.unpack(gf.GF_F32, torch.complex128).cpu().numpy()
    fld.cast(gf.GF_F32, gf.GF_F64)
    got = fld.unpack(gf.GF_F64, torch.complex128).cpu().numpy()
    assert np.abs(got - gram_schmidt_su3(held)).max() < 1e-13        # only rows 0 and 1 of what was held enter
    du, dd = oracle.unitarity_defect(np.ascontiguousarray(got), DIMS)
    assert du < 1e-14 and dd < 1e-14
    # fp64 -> fp32 is a plain rounding of every stored real (no projection)
    V = perturbed_field(DIMS, 10, 1e-3)
    fld.pack(torch.from_numpy(V).to(cuda_device), gf.GF_F64)
    fld.cast(gf.GF_F64, gf.GF_F32)
    got32 = fld.unpack(gf.GF_F32, torch.complex64).cpu().numpy()
    rows = slice(0, 3) if recon == 18 else slice(0, 2)
    assert np.array_equal(got32[..., rows, :], V.astype(np.complex64)[..., rows, :])
    fld.close()
