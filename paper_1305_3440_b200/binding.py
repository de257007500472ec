"""ctypes marshalling for libgf_b200.so -- one Python function per C entry point of include/gf.h.

Device pointers are plain integers (``tensor.data_ptr()``), the stream is
``torch.cuda.current_stream().cuda_stream``.  Calls return the C return code; negative codes
raise ``GFError`` carrying ``gf_last_error``'s text unless ``check=False`` is passed.
"""
import ctypes as C
import os

GF_OK, GF_NOT_CONVERGED = 0, 1
GF_EINVAL, GF_ENOMEM, GF_ECUDA, GF_ESTATE = -1, -2, -3, -4
GF_LANDAU, GF_COULOMB = 0, 1
GF_F32, GF_F64, GF_MIXED, GF_MIXED_EXACT = 0, 1, 2, 3
GF_RELAX, GF_OVERRELAX, GF_STOCHASTIC = 0, 1, 2
GF_RECON18, GF_RECON12 = 18, 12
GF_SOLVER_AUTO = -1

_HERE = os.path.dirname(os.path.abspath(__file__))
lib_path = os.path.join(_HERE, "libgf_b200.so")


class GFError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("libgf_b200 error %d: %s" % (code, text))
        self.code = code


def _load():
    if not os.path.exists(lib_path):
        raise ImportError(
            "%s is missing: build it with `python paper_1305_3440_b200/build.py` "
            "(there is no CPU or PyTorch fallback)" % lib_path)
    L = C.CDLL(lib_path)
    vp, i32, u32, u64, dbl = C.c_void_p, C.c_int, C.c_uint32, C.c_uint64, C.c_double
    ip, dp = C.POINTER(C.c_int), C.POINTER(C.c_double)
    sig = {
        "gf_storage_bytes": (C.c_size_t, [ip, i32, i32]),
        "gf_workspace_bytes": (C.c_size_t, [ip]),
        "gf_init_lattice": (i32, [C.POINTER(vp), ip, i32, i32, vp, vp, vp, vp, u64]),
        "gf_pack": (i32, [vp, vp, i32, i32]),
        "gf_unpack": (i32, [vp, vp, i32, i32]),
        "gf_load_host": (i32, [vp, vp, i32, i32, vp]),
        "gf_store_host": (i32, [vp, vp, i32, i32, vp]),
        "gf_sweep": (i32, [vp, i32, i32, dbl, dbl, i32]),
        "gf_iterate": (i32, [vp, i32, i32, dbl, dbl, i32]),
        "gf_functional": (i32, [vp, i32, dp]),
        "gf_theta": (i32, [vp, i32, dp]),
        "gf_measure": (i32, [vp, i32, dp, dp]),
        "gf_measure_async": (i32, [vp, i32, i32]),
        "gf_measure_collect": (i32, [vp, i32, dp, dp]),
        "gf_measure_static": (i32, [ip, i32, i32, i32, vp, vp, vp, C.c_char_p, C.c_size_t]),
        "gf_fix_until": (i32, [vp, i32, dbl, dbl, i32, dbl, i32, i32, ip, dp]),
        "gf_transform_bytes": (C.c_size_t, [ip, i32, i32]),
        "gf_set_transform": (i32, [vp, vp, vp]),
        "gf_transform_identity": (i32, [vp, i32]),
        "gf_transform_pack": (i32, [vp, vp, i32, i32]),
        "gf_transform_unpack": (i32, [vp, vp, i32, i32]),
        "gf_transform_cast": (i32, [vp, i32, i32]),
        "gf_apply_transform": (i32, [vp, i32, i32, i32]),
        "gf_set_coulomb_mode": (i32, [vp, i32, i32]),
        "gf_coulomb_finish": (i32, [vp, i32]),
        "gf_set_slice_mask": (i32, [vp, C.c_char_p]),
        "gf_set_slab": (i32, [vp, i32, i32, vp, vp, vp, vp, vp, vp, vp]),
        "gf_enable_peer": (i32, [vp, i32]),
        "gf_get_device": (i32, [vp, ip]),
        "gf_set_rng": (i32, [vp, u64, u32]),
        "gf_get_counter": (i32, [vp, C.POINTER(u32)]),
        "gf_reunitarize": (i32, [vp, i32]),
        "gf_cast": (i32, [vp, i32, i32]),
        "gf_plaquette": (i32, [vp, i32, dp]),
        "gf_unitarity": (i32, [vp, i32, dp]),
        "gf_set_tuning": (i32, [vp, i32, i32, i32]),
        "gf_set_solver_precision": (i32, [vp, i32]),
        "gf_set_traversal": (i32, [vp, i32]),
        "gf_set_fix_runahead": (i32, [vp, i32]),
        "gf_set_mixed_stall": (i32, [vp, dbl]),
        "gf_set_reunitarize_every": (i32, [vp, i32]),
        "gf_set_mixed_handoff": (i32, [vp, dbl]),
        "gf_debug_philox": (i32, [vp, i32, vp, vp, vp]),
        "gf_launch_count": (i32, [vp, C.POINTER(u64)]),
        "gf_last_error": (C.c_char_p, [vp]),
        "gf_destroy": (None, [vp]),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    return L


lib = _load()
EXPORTS = ("gf_storage_bytes gf_workspace_bytes gf_init_lattice gf_pack gf_unpack gf_load_host gf_store_host "
           "gf_sweep gf_iterate gf_functional gf_theta gf_measure gf_measure_async gf_measure_collect gf_measure_static gf_fix_until gf_set_rng gf_get_counter gf_reunitarize "
           "gf_cast gf_transform_bytes gf_set_transform gf_transform_identity gf_transform_pack gf_transform_unpack "
           "gf_transform_cast gf_apply_transform gf_set_coulomb_mode gf_coulomb_finish gf_set_slice_mask gf_set_slab gf_enable_peer gf_get_device gf_plaquette gf_unitarity gf_set_tuning gf_set_solver_precision gf_set_traversal gf_set_fix_runahead gf_set_mixed_stall gf_set_reunitarize_every gf_set_mixed_handoff gf_debug_philox gf_launch_count gf_last_error "
           "gf_destroy").split()


def _dims(dims):
    return (C.c_int * 4)(*[int(d) for d in dims])


def _rc(ctx, rc, check=True):
    if rc < 0 and check:
        raise GFError(rc, gf_last_error(ctx))
    return rc


def gf_storage_bytes(dims, precision, recon):
    return lib.gf_storage_bytes(_dims(dims), precision, recon)


def gf_workspace_bytes(dims):
    return lib.gf_workspace_bytes(_dims(dims))


def gf_init_lattice(dims, gauge, recon, dev_links_f64, dev_links_f32, dev_workspace, cuda_stream, seed,
                    check=True):
    """Returns the opaque context handle (an int), or the negative code if check=False."""
    ctx = C.c_void_p()
    rc = lib.gf_init_lattice(C.byref(ctx), _dims(dims), gauge, recon, dev_links_f64 or None,
                             dev_links_f32 or None, dev_workspace or None, cuda_stream or None, int(seed))
    if rc < 0:
        if check:
            raise GFError(rc, "gf_init_lattice failed")
        return rc
    return ctx.value


def gf_destroy(ctx):
    lib.gf_destroy(ctx)


def gf_last_error(ctx):
    s = lib.gf_last_error(ctx)
    return s.decode() if s else ""


def gf_pack(ctx, dev_canonical, canonical_is_f64, precision, check=True):
    return _rc(ctx, lib.gf_pack(ctx, dev_canonical, int(canonical_is_f64), precision), check)


def gf_unpack(ctx, dev_canonical, canonical_is_f64, precision, check=True):
    return _rc(ctx, lib.gf_unpack(ctx, dev_canonical, int(canonical_is_f64), precision), check)


def gf_load_host(ctx, host_canonical, canonical_is_f64, precision, dev_staging, check=True):
    return _rc(ctx, lib.gf_load_host(ctx, host_canonical, int(canonical_is_f64), precision, dev_staging), check)


def gf_store_host(ctx, host_canonical, canonical_is_f64, precision, dev_staging, check=True):
    return _rc(ctx, lib.gf_store_host(ctx, host_canonical, int(canonical_is_f64), precision, dev_staging), check)


def gf_sweep(ctx, parity, algo, omega, p, precision, check=True):
    return _rc(ctx, lib.gf_sweep(ctx, parity, algo, omega, p, precision), check)


def gf_iterate(ctx, n, algo, omega, p, precision, check=True):
    return _rc(ctx, lib.gf_iterate(ctx, int(n), algo, omega, p, precision), check)


def _nout(ctx_dims, gauge):
    return ctx_dims[0] if gauge == GF_COULOMB else 1


def gf_functional(ctx, precision, n_out=1, check=True):
    """n_out: 1 (Landau) or Nt (Coulomb).  Returns a list of floats."""
    out = (C.c_double * n_out)()
    _rc(ctx, lib.gf_functional(ctx, precision, out), check)
    return list(out)


def gf_theta(ctx, precision, n_out=1, check=True):
    out = (C.c_double * n_out)()
    _rc(ctx, lib.gf_theta(ctx, precision, out), check)
    return list(out)


def gf_measure(ctx, precision, n_out=1, check=True):
    """Returns (F list, theta list) from one pass over the field."""
    f = (C.c_double * n_out)()
    t = (C.c_double * n_out)()
    _rc(ctx, lib.gf_measure(ctx, precision, f, t), check)
    return list(f), list(t)


def gf_measure_async(ctx, precision, slot, check=True):
    return _rc(ctx, lib.gf_measure_async(ctx, precision, int(slot)), check)


def gf_measure_collect(ctx, slot, n_out=1, check=True):
    """Returns (F list, theta list) of what gf_measure_async put into the slot."""
    f = (C.c_double * n_out)()
    t = (C.c_double * n_out)()
    _rc(ctx, lib.gf_measure_collect(ctx, int(slot), f, t), check)
    return list(f), list(t)


GF_STATIC_MAX_BLOCKS = 65536


def gf_measure_static(dims, gauge, precision, recon, dev_links, dev_out, cuda_stream, check=True):
    """F and theta of an internal link field without a context and without any allocation (include/gf.h): for callers
    that must not call cudaMalloc / cudaMallocHost where they need theta.  dev_links: the storage a context of the same
    dims / precision / recon packs and sweeps; dev_out: device pointer to 2 doubles (Landau: F, theta) or 2 * Nt
    (Coulomb: F_t, theta_t interleaved).  Asynchronous on cuda_stream; calls that overlap on the GPU race on the
    library's static scratch.  Returns the C return code; a negative one raises GFError with the call's own text."""
    err = C.create_string_buffer(512)
    rc = lib.gf_measure_static(_dims(dims), gauge, precision, recon, dev_links or None, dev_out or None,
                               cuda_stream or None, err, len(err))
    if rc < 0 and check:
        raise GFError(rc, err.value.decode())
    return rc


def gf_fix_until(ctx, algo, omega, p, precision, theta_target, max_iter, check_every, check=True):
    """Returns (return code, iterations, theta)."""
    it = C.c_int(0)
    th = C.c_double(0.0)
    rc = _rc(ctx, lib.gf_fix_until(ctx, algo, omega, p, precision, theta_target, max_iter, check_every,
                                   C.byref(it), C.byref(th)), check)
    return rc, it.value, th.value


def gf_set_rng(ctx, seed, half_sweep_counter, check=True):
    return _rc(ctx, lib.gf_set_rng(ctx, int(seed), int(half_sweep_counter)), check)


def gf_get_counter(ctx):
    c = C.c_uint32(0)
    _rc(ctx, lib.gf_get_counter(ctx, C.byref(c)))
    return c.value


def gf_reunitarize(ctx, precision, check=True):
    return _rc(ctx, lib.gf_reunitarize(ctx, precision), check)


def gf_cast(ctx, from_precision, to_precision, check=True):
    return _rc(ctx, lib.gf_cast(ctx, from_precision, to_precision), check)


def gf_transform_bytes(dims, precision, recon):
    return lib.gf_transform_bytes(_dims(dims), precision, recon)


def gf_set_transform(ctx, dev_g_f64, dev_g_f32, check=True):
    return _rc(ctx, lib.gf_set_transform(ctx, dev_g_f64 or None, dev_g_f32 or None), check)


def gf_transform_identity(ctx, precision, check=True):
    return _rc(ctx, lib.gf_transform_identity(ctx, precision), check)


def gf_transform_pack(ctx, dev_canonical, canonical_is_f64, precision, check=True):
    return _rc(ctx, lib.gf_transform_pack(ctx, dev_canonical, int(canonical_is_f64), precision), check)


def gf_transform_unpack(ctx, dev_canonical, canonical_is_f64, precision, check=True):
    return _rc(ctx, lib.gf_transform_unpack(ctx, dev_canonical, int(canonical_is_f64), precision), check)


def gf_transform_cast(ctx, from_precision, to_precision, check=True):
    return _rc(ctx, lib.gf_transform_cast(ctx, from_precision, to_precision), check)


def gf_apply_transform(ctx, g_precision, src_precision, dst_precision, check=True):
    return _rc(ctx, lib.gf_apply_transform(ctx, g_precision, src_precision, dst_precision), check)


def gf_set_coulomb_mode(ctx, defer_temporal, freeze_slices, check=True):
    return _rc(ctx, lib.gf_set_coulomb_mode(ctx, int(defer_temporal), int(freeze_slices)), check)


def gf_coulomb_finish(ctx, precision, check=True):
    return _rc(ctx, lib.gf_coulomb_finish(ctx, precision), check)


def gf_set_slice_mask(ctx, active, check=True):
    """active: sequence of Nt truth values, or None for all slices."""
    buf = None if active is None else bytes(1 if a else 0 for a in active)
    return _rc(ctx, lib.gf_set_slice_mask(ctx, buf), check)


def gf_set_slab(ctx, rank, nranks, prev_f64, prev_f32, next_f64, next_f32, flag_own, flag_prev, flag_next, check=True):
    return _rc(ctx, lib.gf_set_slab(ctx, int(rank), int(nranks), prev_f64 or None, prev_f32 or None, next_f64 or None,
                                    next_f32 or None, flag_own or None, flag_prev or None, flag_next or None), check)


def gf_enable_peer(ctx, peer_device, check=True):
    return _rc(ctx, lib.gf_enable_peer(ctx, int(peer_device)), check)


def gf_get_device(ctx):
    d = C.c_int(-1)
    _rc(ctx, lib.gf_get_device(ctx, C.byref(d)))
    return d.value


def gf_plaquette(ctx, precision, check=True):
    out = C.c_double(0.0)
    _rc(ctx, lib.gf_plaquette(ctx, precision, C.byref(out)), check)
    return out.value


def gf_unitarity(ctx, precision, check=True):
    out = (C.c_double * 2)()
    _rc(ctx, lib.gf_unitarity(ctx, precision, out), check)
    return out[0], out[1]


def gf_set_tuning(ctx, precision, lanes_per_site, block_threads, check=True):
    return _rc(ctx, lib.gf_set_tuning(ctx, precision, lanes_per_site, block_threads), check)


def gf_set_solver_precision(ctx, solver_precision, check=True):
    return _rc(ctx, lib.gf_set_solver_precision(ctx, solver_precision), check)


def gf_set_traversal(ctx, zigzag, check=True):
    return _rc(ctx, lib.gf_set_traversal(ctx, int(zigzag)), check)


def gf_set_reunitarize_every(ctx, iterations, check=True):
    return _rc(ctx, lib.gf_set_reunitarize_every(ctx, int(iterations)), check)


def gf_set_mixed_stall(ctx, ratio, check=True):
    return _rc(ctx, lib.gf_set_mixed_stall(ctx, float(ratio)), check)


def gf_set_fix_runahead(ctx, blocks, check=True):
    return _rc(ctx, lib.gf_set_fix_runahead(ctx, int(blocks)), check)


def gf_set_mixed_handoff(ctx, theta_handoff, check=True):
    return _rc(ctx, lib.gf_set_mixed_handoff(ctx, float(theta_handoff)), check)


def gf_debug_philox(ctx, n, dev_counters, dev_keys, dev_out, check=True):
    return _rc(ctx, lib.gf_debug_philox(ctx, n, dev_counters, dev_keys, dev_out), check)


def gf_launch_count(ctx):
    c = C.c_uint64(0)
    _rc(ctx, lib.gf_launch_count(ctx, C.byref(c)))
    return c.value
