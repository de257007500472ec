"""State rules of the C ABI that involve the device (include/gf.h): the transformation buffer while a deferred
temporal update is outstanding, the theta a mixed-precision run returns, the device a context belongs to."""
import numpy as np
import pytest
import torch

import gf_inputs as gi
import oracle
import paper_1305_3440_b200 as gf
from paper_1305_3440_b200 import binding as B

pytestmark = pytest.mark.gpu


def test_transformation_buffer_is_protected_while_a_deferred_update_is_pending(cuda_device):
    dims = (4, 6, 4, 6)
    U = gi.smooth_random_gauge(dims, 0.5, 3)
    Ud = torch.from_numpy(U).to(cuda_device)
    fld = gf.GaugeField(dims, gauge=gf.GF_COULOMB, precisions=("f64", "f32"), seed=5, device=cuda_device)
    fld.attach_transform(("f64", "f32"))
    fld.pack(Ud, gf.GF_F64)
    fld.set_coulomb_mode(defer_temporal=True)
    fld.sweep(0, gf.GF_OVERRELAX, 1.6, 0.0, gf.GF_F64)                 # the fp64 G now holds the only copy of the update of U_0
    assert B.lib.gf_transform_identity(fld.ctx, gf.GF_F64) == gf.GF_ESTATE
    assert "deferred" in gf.gf_last_error(fld.ctx)
    canon = torch.zeros(fld.shape[:4] + (3, 3), dtype=torch.complex128, device=cuda_device)
    assert B.lib.gf_transform_pack(fld.ctx, canon.data_ptr(), 1, gf.GF_F64) == gf.GF_ESTATE
    assert B.lib.gf_transform_cast(fld.ctx, gf.GF_F32, gf.GF_F64) == gf.GF_ESTATE
    assert B.lib.gf_set_transform(fld.ctx, None, fld._gbufs[gf.GF_F32].data_ptr()) == gf.GF_ESTATE
    assert B.lib.gf_transform_identity(fld.ctx, gf.GF_F32) == gf.GF_OK     # the other precision has nothing pending
    assert B.lib.gf_pack(fld.ctx, None, 1, gf.GF_F64) == gf.GF_EINVAL      # a failed pack does not drop the update
    fld.sweep(1, gf.GF_OVERRELAX, 1.6, 0.0, gf.GF_F64)
    got = fld.unpack(gf.GF_F64).cpu().numpy()                              # finishes the temporal links
    Uo = U.copy()
    for parity in (0, 1):
        oracle.sweep(Uo, dims, parity, oracle.COULOMB, oracle.OVERRELAX, 1.6)
    assert np.abs(got - Uo).max() < 1e-12
    assert B.lib.gf_transform_identity(fld.ctx, gf.GF_F64) == gf.GF_OK     # nothing pending any more
    # an fp64 field with a pending update that is overwritten by a cast loses the update, not the new field
    fld.pack(Ud, gf.GF_F64)
    fld.pack(Ud.to(torch.complex64), gf.GF_F32)
    fld.sweep(0, gf.GF_OVERRELAX, 1.6, 0.0, gf.GF_F64)                     # pending on fp64
    fld.set_coulomb_mode(defer_temporal=False)                             # finishes it
    fld.set_coulomb_mode(defer_temporal=True)
    fld.sweep(1, gf.GF_OVERRELAX, 1.6, 0.0, gf.GF_F64)                     # pending again
    fld.cast(gf.GF_F32, gf.GF_F64)                                         # fp64 field replaced by the (re-projected) fp32 input
    back = fld.unpack(gf.GF_F64).cpu().numpy()
    assert np.abs(back - U).max() < 1e-6                                   # no stale G applied to it
    fld.close()


def test_mixed_precision_returns_the_theta_of_the_f64_field(cuda_device):
    dims = (8, 8, 8, 8)
    U = gi.smooth_random_gauge(dims, 0.5, 1234)
    for mode in (gf.GF_MIXED, gf.GF_MIXED_EXACT):
        # (a) the fp32 phase uses up max_iter; (b) the fp32 phase already meets a loose target
        for target, max_iter in ((1e-12, 20), (1e-5, 20000)):
            fld = gf.GaugeField(dims, precisions=("f32", "f64"), device=cuda_device)
            fld.pack(torch.from_numpy(U).to(cuda_device), gf.GF_F64)
            fld.pack(torch.from_numpy(U).to(cuda_device).to(torch.complex64), gf.GF_F32)
            if mode == gf.GF_MIXED_EXACT:
                fld.attach_transform(("f64", "f32"))
            rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, mode, target, max_iter, 10)
            th64 = fld.theta(gf.GF_F64)[0]
            assert th == th64, (mode, target, th, th64)                    # bit for bit: measured on the fp64 result
            tho = oracle.theta(np.ascontiguousarray(fld.unpack(gf.GF_F64).cpu().numpy()), dims)
            assert abs(th / tho - 1) < 1e-9
            if max_iter == 20:
                assert rc == gf.GF_NOT_CONVERGED and it == 20
            else:
                assert rc == gf.GF_OK and th < target
            fld.close()


def test_a_context_belongs_to_its_device(cuda_device):
    fld = gf.GaugeField((4, 4, 4, 4), device=cuda_device)
    assert gf.gf_get_device(fld.ctx) == (cuda_device.index or 0)
    assert B.lib.gf_enable_peer(fld.ctx, cuda_device.index or 0) == gf.GF_OK       # same device: nothing to do
    assert B.lib.gf_enable_peer(fld.ctx, 4096) == gf.GF_EINVAL
    assert B.lib.gf_enable_peer(fld.ctx, -1) == gf.GF_EINVAL
    fld.close()


def test_misaligned_canonical_buffers_are_refused_before_any_launch(cuda_device):
    """pack / unpack move the canonical side as 16-byte vectors: a canonical or staging pointer at an odd offset (a tensor
    view, say) is answered with GF_EINVAL on the host instead of a misaligned-address fault that would poison the CUDA
    context; the field is untouched and the context keeps working."""
    dims = (4, 4, 4, 4)
    U = torch.from_numpy(gi.smooth_random_gauge(dims, 0.4, 9)).to(cuda_device)
    fld = gf.GaugeField(dims, precisions=("f64",), device=cuda_device, staging=True)
    fld.attach_transform(("f64",))
    fld.pack(U, gf.GF_F64)
    n = U.numel() * 16
    raw = torch.zeros(n + 64, dtype=torch.uint8, device=cuda_device)
    odd = raw.data_ptr() + 8                                               # 8-byte aligned only
    host = torch.zeros(U.shape, dtype=torch.complex128).pin_memory()
    for rc in (B.lib.gf_pack(fld.ctx, odd, 1, gf.GF_F64), B.lib.gf_unpack(fld.ctx, odd, 1, gf.GF_F64),
               B.lib.gf_load_host(fld.ctx, host.data_ptr(), 1, gf.GF_F64, odd),
               B.lib.gf_store_host(fld.ctx, host.data_ptr(), 1, gf.GF_F64, odd),
               B.lib.gf_transform_pack(fld.ctx, odd, 1, gf.GF_F64), B.lib.gf_transform_unpack(fld.ctx, odd, 1, gf.GF_F64)):
        assert rc == gf.GF_EINVAL
        assert "16-byte aligned" in gf.gf_last_error(fld.ctx)
    torch.cuda.synchronize(cuda_device)                                    # nothing faulted
    assert torch.equal(fld.unpack(gf.GF_F64), U)                           # and nothing was written
    assert float(host.abs().max()) == 0.0
    fld.close()
