"""paper_1305_3440_b200 -- B200-native SU(3) lattice gauge fixing (arXiv:1305.3440).

Thin Python binding of ``libgf_b200.so`` (C ABI: ``include/gf.h``).  The functions below have the
same names as the C entry points and only marshal arguments; every step of the method runs in
the library's CUDA kernels.  PyTorch is used for device memory and streams only.  There is no CPU
fallback: importing the binding without the built library raises.
"""
from .binding import (  # noqa: F401
    GF_OK, GF_NOT_CONVERGED, GF_EINVAL, GF_ENOMEM, GF_ECUDA, GF_ESTATE,
    GF_LANDAU, GF_COULOMB, GF_F32, GF_F64, GF_MIXED, GF_MIXED_EXACT,
    GF_RELAX, GF_OVERRELAX, GF_STOCHASTIC, GF_RECON18, GF_RECON12, GF_SOLVER_AUTO,
    GFError, lib, lib_path,
    gf_storage_bytes, gf_workspace_bytes, gf_init_lattice, gf_destroy, gf_last_error,
    gf_pack, gf_unpack, gf_load_host, gf_store_host, gf_sweep, gf_iterate, gf_functional, gf_theta,
    gf_measure, gf_measure_async, gf_measure_collect, gf_measure_static, GF_STATIC_MAX_BLOCKS, gf_fix_until, gf_set_rng, gf_get_counter, gf_reunitarize, gf_cast,
    gf_transform_bytes, gf_set_transform, gf_transform_identity, gf_transform_pack, gf_transform_unpack,
    gf_transform_cast, gf_apply_transform, gf_set_coulomb_mode, gf_coulomb_finish, gf_set_slice_mask, gf_set_slab, gf_enable_peer, gf_get_device,
    gf_plaquette, gf_unitarity, gf_set_tuning, gf_set_solver_precision, gf_set_traversal, gf_set_fix_runahead, gf_set_mixed_stall, gf_set_reunitarize_every, gf_set_mixed_handoff, gf_debug_philox, gf_launch_count,
)
from .field import GaugeField  # noqa: F401
