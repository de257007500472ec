"""ctypes binding of the CPU oracle (oracle/gf_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.  It
shares no code with ``paper_1305_3440_b200`` and neither imports the other.

All link fields are numpy ``complex128`` arrays in the canonical layout
``(Nt, Nz, Ny, Nx, 4, 3, 3)`` (site s = x + Nx (y + Ny (z + Nz t)); mu = 0 is time,
1,2,3 = x,y,z); ``dims = (Nt, Nx, Ny, Nz)``.  Functions that update links do so IN PLACE.
Citations are in gf_oracle.c next to the code that implements each passage.
"""
import ctypes as C

import numpy as np

from . import build as _build

LANDAU, COULOMB = 0, 1
RELAX, OVERRELAX, STOCHASTIC = 0, 1, 2

_lib = None


def load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(_build.build())
    cd_p = C.c_void_p
    i4 = C.POINTER(C.c_int)
    dbl_p = C.POINTER(C.c_double)
    lib.oracle_set_threads.argtypes = [C.c_int]
    lib.oracle_set_threads.restype = C.c_int
    lib.oracle_get_threads.restype = C.c_int
    lib.oracle_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
    lib.oracle_site_uniforms.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, dbl_p]
    lib.oracle_functional.argtypes = [cd_p, i4, C.c_int, dbl_p]
    lib.oracle_theta.argtypes = [cd_p, i4, C.c_int, dbl_p]
    lib.oracle_site_delta.argtypes = [cd_p, i4, C.c_int, C.c_size_t, cd_p]
    lib.oracle_site_K.argtypes = [cd_p, i4, C.c_int, C.c_size_t, cd_p]
    lib.oracle_su2_vector.argtypes = [cd_p, C.c_int, C.c_int, dbl_p]
    lib.oracle_su2_update.argtypes = [dbl_p, C.c_int, C.c_double, C.c_double, C.c_double, dbl_p]
    lib.oracle_site_g.argtypes = [cd_p, C.c_int, C.c_double, C.c_double, dbl_p, cd_p]
    lib.oracle_update_links8.argtypes = [cd_p, cd_p, C.c_int, C.c_int, C.c_double, C.c_double,
                                         dbl_p, cd_p]
    lib.oracle_sweep_ordered.argtypes = [cd_p, i4, C.c_int, C.c_int, C.c_int, C.c_double,
                                         C.c_double, C.c_uint64, C.c_uint32, C.c_int]
    lib.oracle_sweep.argtypes = lib.oracle_sweep_ordered.argtypes[:-1]
    lib.oracle_sweep_accumulate.argtypes = [cd_p, cd_p, i4, C.c_int, C.c_int, C.c_int, C.c_double,
                                            C.c_double, C.c_uint64, C.c_uint32]
    lib.oracle_apply_transform.argtypes = [cd_p, cd_p, i4, cd_p]
    lib.oracle_sweep_masked.argtypes = [cd_p, cd_p, i4, i4, C.c_int, C.c_int, C.c_int, C.c_double,
                                        C.c_double, C.c_uint64, C.c_uint32]
    lib.oracle_fix_until_freeze.argtypes = [cd_p, i4, C.c_int, C.c_double, C.c_double, C.c_uint64, C.c_uint32,
                                            C.c_double, C.c_int, C.c_int, dbl_p, i4, C.POINTER(C.c_int)]
    lib.oracle_fix_until_freeze.restype = C.c_int
    lib.oracle_fix_until.argtypes = [cd_p, i4, C.c_int, C.c_int, C.c_double, C.c_double,
                                     C.c_uint64, C.c_uint32, C.c_double, C.c_int, C.c_int,
                                     dbl_p, C.POINTER(C.c_int)]
    lib.oracle_fix_until.restype = C.c_int
    lib.oracle_plaquette.argtypes = [cd_p, i4]
    lib.oracle_plaquette.restype = C.c_double
    lib.oracle_unitarity_defect.argtypes = [cd_p, i4, dbl_p]
    _lib = lib
    return lib


def _dims(dims):
    assert len(dims) == 4
    return (C.c_int * 4)(*[int(d) for d in dims])


def _field(U, dims):
    nt, nx, ny, nz = dims
    assert isinstance(U, np.ndarray) and U.dtype == np.complex128 and U.flags.c_contiguous
    assert U.shape == (nt, nz, ny, nx, 4, 3, 3), (U.shape, dims)
    return U.ctypes.data_as(C.c_void_p)


def _mat(M):
    assert M.dtype == np.complex128 and M.flags.c_contiguous
    return M.ctypes.data_as(C.c_void_p)


def _dbl(a):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_double))


def nslices(dims, gauge):
    return dims[0] if gauge == COULOMB else 1


def set_threads(n):
    """n < 1: all cores.  Returns the thread count in effect."""
    return load().oracle_set_threads(int(n))


def get_threads():
    return load().oracle_get_threads()


def philox4x32_10(counter, key):
    ctr = (C.c_uint32 * 4)(*counter)
    k = (C.c_uint32 * 2)(*key)
    out = (C.c_uint32 * 4)()
    load().oracle_philox4x32_10(ctr, k, out)
    return tuple(int(w) for w in out)


def site_uniforms(seed, half_sweep_counter, s):
    u = np.zeros(3)
    load().oracle_site_uniforms(int(seed), int(half_sweep_counter), int(s), _dbl(u))
    return u


def functional(U, dims, gauge=LANDAU):
    out = np.zeros(nslices(dims, gauge))
    load().oracle_functional(_field(U, dims), _dims(dims), gauge, _dbl(out))
    return out if gauge == COULOMB else float(out[0])


def theta(U, dims, gauge=LANDAU):
    out = np.zeros(nslices(dims, gauge))
    load().oracle_theta(_field(U, dims), _dims(dims), gauge, _dbl(out))
    return out if gauge == COULOMB else float(out[0])


def site_delta(U, dims, s, gauge=LANDAU):
    D = np.zeros((3, 3), np.complex128)
    load().oracle_site_delta(_field(U, dims), _dims(dims), gauge, int(s), _mat(D))
    return D


def site_K(U, dims, s, gauge=LANDAU):
    K = np.zeros((3, 3), np.complex128)
    load().oracle_site_K(_field(U, dims), _dims(dims), gauge, int(s), _mat(K))
    return K


def su2_vector(K, i, j):
    K = np.ascontiguousarray(K, np.complex128)
    v = np.zeros(4)
    load().oracle_su2_vector(_mat(K), i, j, _dbl(v))
    return v


def su2_update(v, algo, omega=1.0, p=0.0, u=0.0):
    v = np.ascontiguousarray(v, np.float64)
    a = np.zeros(4)
    load().oracle_su2_update(_dbl(v), algo, omega, p, u, _dbl(a))
    return a


def site_g(K, algo, omega=1.0, p=0.0, u=(0.0, 0.0, 0.0)):
    K = np.ascontiguousarray(K, np.complex128)
    u = np.ascontiguousarray(u, np.float64)
    g = np.zeros((3, 3), np.complex128)
    load().oracle_site_g(_mat(K), algo, omega, p, _dbl(u), _mat(g))
    return g


def update_links8(fwd, bwd, gauge, algo, omega=1.0, p=0.0, u=(0.0, 0.0, 0.0)):
    """fwd[mu] = U_mu(x), bwd[mu] = U_mu(x - mu_hat), shape (4,3,3) each; updated in place.
    Returns g(x)."""
    assert fwd.shape == (4, 3, 3) and bwd.shape == (4, 3, 3)
    u = np.ascontiguousarray(u, np.float64)
    g = np.zeros((3, 3), np.complex128)
    load().oracle_update_links8(_mat(fwd), _mat(bwd), gauge, algo, omega, p, _dbl(u), _mat(g))
    return g


def sweep(U, dims, parity, gauge=LANDAU, algo=OVERRELAX, omega=1.0, p=0.0, seed=0,
          half_sweep_counter=0, reverse_order=False):
    load().oracle_sweep_ordered(_field(U, dims), _dims(dims), gauge, parity, algo, omega, p,
                                int(seed), int(half_sweep_counter), int(bool(reverse_order)))


def _transform(G, dims):
    nt, nx, ny, nz = dims
    assert isinstance(G, np.ndarray) and G.dtype == np.complex128 and G.flags.c_contiguous
    assert G.shape == (nt, nz, ny, nx, 3, 3), (G.shape, dims)
    return G.ctypes.data_as(C.c_void_p)


def identity_transform(dims):
    nt, nx, ny, nz = dims
    G = np.zeros((nt, nz, ny, nx, 3, 3), np.complex128)
    G[..., 0, 0] = G[..., 1, 1] = G[..., 2, 2] = 1.0
    return G


def sweep_accumulate(U, G, dims, parity, gauge=LANDAU, algo=OVERRELAX, omega=1.0, p=0.0, seed=0,
                     half_sweep_counter=0):
    """The half-sweep of ``sweep`` that also records Gtot(x) <- g(x) Gtot(x); U and G in place."""
    load().oracle_sweep_accumulate(_field(U, dims), _transform(G, dims), _dims(dims), gauge, parity,
                                   algo, omega, p, int(seed), int(half_sweep_counter))


def apply_transform(U, G, dims):
    """Returns G(x) U_mu(x) G(x+mu)^dagger (eq. 3) as a new array."""
    out = np.empty_like(U)
    load().oracle_apply_transform(_field(U, dims), _transform(G, dims), _dims(dims), _field(out, dims))
    return out


def sweep_masked(U, dims, parity, slice_active, G=None, gauge=COULOMB, algo=OVERRELAX, omega=1.0, p=0.0, seed=0,
                 half_sweep_counter=0):
    """Half-sweep that skips the sites of time slices with slice_active[t] == 0 (reading A17b)."""
    act = (C.c_int * dims[0])(*[int(bool(a)) for a in slice_active])
    load().oracle_sweep_masked(_field(U, dims), _transform(G, dims) if G is not None else None, act, _dims(dims),
                               gauge, parity, algo, omega, p, int(seed), int(half_sweep_counter))


def fix_until_freeze(U, dims, algo=OVERRELAX, omega=1.0, p=0.0, seed=0, first_counter=0, theta_target=1e-12,
                     max_iter=2000, check_every=1):
    """Coulomb gauge with slice freezing.  Returns (iterations, theta_t array, frozen_at array, converged)."""
    th = np.zeros(dims[0])
    fr = (C.c_int * dims[0])()
    conv = C.c_int()
    it = load().oracle_fix_until_freeze(_field(U, dims), _dims(dims), algo, omega, p, int(seed), int(first_counter),
                                        theta_target, max_iter, check_every, _dbl(th), fr, C.byref(conv))
    if it < 0:
        raise ValueError("oracle fix loops hold per-slice state for at most 4096 time slices, got %d" % dims[0])
    return it, th, np.array(list(fr)), bool(conv.value)


def fix_until(U, dims, gauge=LANDAU, algo=OVERRELAX, omega=1.0, p=0.0, seed=0, first_counter=0,
              theta_target=1e-12, max_iter=2000, check_every=1):
    """Returns (iterations, theta at the last evaluation, converged)."""
    th = C.c_double()
    conv = C.c_int()
    it = load().oracle_fix_until(_field(U, dims), _dims(dims), gauge, algo, omega, p, int(seed),
                                 int(first_counter), theta_target, max_iter, check_every,
                                 C.byref(th), C.byref(conv))
    if it < 0:
        raise ValueError("oracle fix loops hold per-slice state for at most 4096 time slices, got %d" % dims[0])
    return it, th.value, bool(conv.value)


def plaquette(U, dims):
    return load().oracle_plaquette(_field(U, dims), _dims(dims))


def unitarity_defect(U, dims):
    out = np.zeros(2)
    load().oracle_unitarity_defect(_field(U, dims), _dims(dims), _dbl(out))
    return float(out[0]), float(out[1])
