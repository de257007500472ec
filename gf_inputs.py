"""Seeded synthetic link fields (the input recipe of DESIGN.md, "Inputs").

This module serves BOTH the CPU oracle's tests and the CUDA path's tests/bench.  It holds
none of the method's arithmetic (no K, no SU(2) solve, no F or theta): only random SU(3)
matrices and the textbook gauge transformation used to *construct* inputs.  It imports neither
``oracle`` nor ``paper_1305_3440_b200``.

Canonical layout everywhere: complex array of shape ``(Nt, Nz, Ny, Nx, 4, 3, 3)``; the link
index mu = 0 is time, 1,2,3 = x,y,z; ``dims = (Nt, Nx, Ny, Nz)``.

The paper's thermalised gauge configurations are not available; these
fields stand in for them (BASELINE.json ``configs``): a smooth field U = exp(i eps H) with H
traceless Hermitian and Gaussian, then a Haar-random gauge transformation
g(x) U_mu(x) g(x+mu)^dagger (eq. 3); or a "hot" field of independent Haar links.
"""
import numpy as np

# lattice axis of the canonical array that direction mu runs along: (t,z,y,x) are axes 0..3
AXIS_OF_MU = (0, 3, 2, 1)


def field_shape(dims):
    nt, nx, ny, nz = dims
    return (nt, nz, ny, nx)


# ------------------------------------------------------------------ numpy (host) generators

def _complex_gaussian(rng, shape):
    ri = rng.standard_normal(shape + (2,))
    return ri[..., 0] + 1j * ri[..., 1]


def traceless_hermitian(rng, shape):
    """H = (M + M^dagger)/2 - (tr/3) 1 with Re M, Im M ~ N(0,1) i.i.d.; shape + (3,3)."""
    M = _complex_gaussian(rng, shape + (3, 3))
    H = 0.5 * (M + np.conj(np.swapaxes(M, -1, -2)))
    tr = np.trace(H, axis1=-2, axis2=-1) / 3.0
    H[..., 0, 0] -= tr
    H[..., 1, 1] -= tr
    H[..., 2, 2] -= tr
    return H


def exp_i_hermitian(H, eps):
    """exp(i eps H) through the Hermitian eigendecomposition."""
    w, V = np.linalg.eigh(H)
    return np.einsum("...ab,...b,...cb->...ac", V, np.exp(1j * eps * w), np.conj(V))


def haar_su3(rng, shape):
    """Haar-random SU(3): QR of a complex Gaussian 3x3, phases of diag(R) moved into Q,
    det normalised to 1 with the principal cube root."""
    Z = _complex_gaussian(rng, shape + (3, 3))
    Q, R = np.linalg.qr(Z)
    d = np.diagonal(R, axis1=-2, axis2=-1)
    Q = Q * (d / np.abs(d))[..., None, :]
    det = np.linalg.det(Q)
    return Q / (det ** (1.0 / 3.0))[..., None, None]


def gauge_transform(U, g):
    """U_mu(x) -> g(x) U_mu(x) g(x + mu_hat)^dagger (eq. 3); periodic."""
    out = np.empty_like(U)
    for mu in range(4):
        g_fwd = np.roll(g, -1, axis=AXIS_OF_MU[mu])
        out[..., mu, :, :] = np.einsum("...ab,...bc,...dc->...ad", g, U[..., mu, :, :], np.conj(g_fwd))
    return out


def unit_links(dims):
    U = np.zeros(field_shape(dims) + (4, 3, 3), np.complex128)
    U[..., 0, 0] = U[..., 1, 1] = U[..., 2, 2] = 1.0
    return U


def smooth_links(dims, eps, seed):
    """U_mu(x) = exp(i eps H_mu(x)); also returns H (for closed-form small-field checks)."""
    rng = np.random.default_rng(seed)
    H = traceless_hermitian(rng, field_shape(dims) + (4,))
    return np.ascontiguousarray(exp_i_hermitian(H, eps)), H


def smooth_random_gauge(dims, eps, seed):
    """The configs' standard input: smooth field, then a Haar-random gauge transformation.
    Draw order is fixed: all H (canonical order) first, then all g."""
    rng = np.random.default_rng(seed)
    H = traceless_hermitian(rng, field_shape(dims) + (4,))
    U = exp_i_hermitian(H, eps)
    g = haar_su3(rng, field_shape(dims))
    return np.ascontiguousarray(gauge_transform(U, g))


def hot_links(dims, seed):
    """Independent Haar-random link on every (x, mu) (strong-coupling-like)."""
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(haar_su3(rng, field_shape(dims) + (4,)))


def random_gauge(dims, seed):
    return haar_su3(np.random.default_rng(seed), field_shape(dims))


# ---------------------------------------------------------------- torch (device) generators
# Same recipe, torch generator: statistically, not bitwise, the same fields.  Used where the
# host generators would take too long (32^4 bench inputs, 64^4).  Works slab by slab in t to
# bound temporary memory.

def _torch_complex_gaussian(torch, gen, shape, device):
    ri = torch.randn(shape + (2,), generator=gen, device=device, dtype=torch.float64)
    return torch.view_as_complex(ri)


def _torch_haar_su3(torch, gen, shape, device):
    # Gram-Schmidt on the columns of a complex Gaussian = its QR with diag(R) > 0, i.e. the
    # phase-fixed Q of haar_su3 above.
    Z = _torch_complex_gaussian(torch, gen, shape + (3, 3), device)
    c0, c1, c2 = Z[..., :, 0], Z[..., :, 1], Z[..., :, 2]
    q0 = c0 / torch.linalg.vector_norm(c0, dim=-1, keepdim=True)
    c1 = c1 - q0 * (q0.conj() * c1).sum(-1, keepdim=True)
    q1 = c1 / torch.linalg.vector_norm(c1, dim=-1, keepdim=True)
    c2 = c2 - q0 * (q0.conj() * c2).sum(-1, keepdim=True) - q1 * (q1.conj() * c2).sum(-1, keepdim=True)
    q2 = c2 / torch.linalg.vector_norm(c2, dim=-1, keepdim=True)
    Q = torch.stack((q0, q1, q2), dim=-1)
    det = torch.linalg.det(Q)
    phase = torch.polar(torch.ones_like(det.real), torch.angle(det) / 3.0)
    return Q / phase[..., None, None]


def _torch_polish_unitary(torch, U, slab=4):
    """Two Newton-Schulz steps U <- U (3 - U^dagger U)/2, in place, slab by slab.  Classical
    Gram-Schmidt on an ill-conditioned Gaussian draw leaves |UU^dagger - 1| ~ 1e-12 on the worst of
    10^7 matrices; each step squares the defect, so the field ends at rounding level."""
    eye3 = 3.0 * torch.eye(3, dtype=U.dtype, device=U.device)
    for t0 in range(0, U.shape[0], slab):
        W = U[t0:t0 + slab]
        for _ in range(2):
            W = 0.5 * (W @ (eye3 - W.mH @ W))
        U[t0:t0 + slab] = W
    return U


def torch_smooth_random_gauge(dims, eps, seed, device="cuda", slab=4):
    import torch
    nt, nx, ny, nz = dims
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    U = torch.empty(field_shape(dims) + (4, 3, 3), dtype=torch.complex128, device=device)
    g = torch.empty(field_shape(dims) + (3, 3), dtype=torch.complex128, device=device)
    for t0 in range(0, nt, slab):
        t1 = min(nt, t0 + slab)
        shp = (t1 - t0, nz, ny, nx)
        M = _torch_complex_gaussian(torch, gen, shp + (4, 3, 3), device)
        H = 0.5 * (M + M.mH)
        tr = torch.diagonal(H, dim1=-2, dim2=-1).sum(-1) / 3.0
        H = H - tr[..., None, None] * torch.eye(3, dtype=H.dtype, device=device)
        U[t0:t1] = torch.linalg.matrix_exp(1j * eps * H)
        g[t0:t1] = _torch_haar_su3(torch, gen, shp, device)
        del M, H
    for mu in range(4):
        g_fwd = torch.roll(g, -1, dims=AXIS_OF_MU[mu])
        U[..., mu, :, :] = g @ U[..., mu, :, :] @ g_fwd.mH
        del g_fwd
    del g
    return _torch_polish_unitary(torch, U, slab)


def torch_hot_links(dims, seed, device="cuda"):
    import torch
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    return _torch_polish_unitary(torch, _torch_haar_su3(torch, gen, field_shape(dims) + (4,), device).contiguous())
