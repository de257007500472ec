"""gf_measure_static: F and theta for callers that cannot allocate (include/gf.h).

Some users of the library want theta at a point where they may not allocate anything: a monitor inside another
program's update loop after that program's pool allocator has taken all of the GPU's memory, a job with a memory
budget fixed at start-up, a latency-bound loop that cannot take the device-wide synchronisation of cudaMalloc /
cudaMallocHost.  They cannot create a gf_ctx (gf_init_lattice allocates pinned host memory and wants a workspace
buffer), so gf_measure_static takes only the link field and an output pointer and keeps its partial sums in an array
that is part of the library's device image.  These tests hold it to the existing path, gf_measure: same numbers, on
calls in a row that share that array, with no change in the device's free memory, and a clear refusal for lattices
whose reduction does not fit the array.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here should not hide the
parity tests.  Nothing here depends on what ran before it in the process (the first call on a device does the
entry point's one-time set-up whenever that is), so it passes alone and at the end of the whole run.
"""
import numpy as np
import pytest
import torch

import gf_inputs as gi
import oracle
import paper_1305_3440_b200 as gf
from paper_1305_3440_b200 import binding

PREC = {"f64": gf.GF_F64, "f32": gf.GF_F32}
CDTYPE = {"f64": torch.complex128, "f32": torch.complex64}
REL = 1e-12          # the tolerance of the F / theta parity tests (tests/test_gpu_parity.py); both paths accumulate in fp64


def _static(fld, prec, out):
    binding.gf_measure_static(fld.dims, fld.gauge, prec, fld.recon, fld.storage(prec).data_ptr(), out.data_ptr(),
                              fld.stream.cuda_stream)


def _close(a, b):
    return abs(a - b) <= REL * max(abs(a), abs(b))


@pytest.mark.gpu
@pytest.mark.parametrize("prec,recon", [("f64", 18), ("f32", 12)])
def test_two_calls_in_a_row_match_gf_measure(cuda_device, prec, recon):
    """Landau gauge.  Call 1 on a lattice with many blocks per slice and a ragged last block, call 2 straight after it
    on a smaller lattice (fewer partial sums than call 1 left in the shared scratch), call 3 on the first field again
    after a sweep has changed it: each must give what gf_measure gives for that field."""
    P = PREC[prec]
    big, small = (6, 10, 12, 14), (4, 4, 6, 4)        # 840 and 48 sites per (slice, parity): 7 blocks (ragged) and 1
    fa = gf.GaugeField(big, recon=recon, precisions=(prec,), device=cuda_device)
    fb = gf.GaugeField(small, recon=recon, precisions=(prec,), device=cuda_device)
    Ua = gi.smooth_random_gauge(big, 0.4, 11)
    fa.pack(torch.from_numpy(Ua).to(cuda_device).to(CDTYPE[prec]), P)
    fb.pack(torch.from_numpy(gi.hot_links(small, 12)).to(cuda_device).to(CDTYPE[prec]), P)
    out = torch.full((3, 2), float("nan"), dtype=torch.float64, device=cuda_device)

    _static(fa, P, out[0])
    _static(fb, P, out[1])                             # back to back on the same stream: ordered, sharing the scratch
    fa.iterate(1, gf.GF_OVERRELAX, 1.7, 0.0, P)
    _static(fa, P, out[2])
    got = out.cpu().numpy()

    fb_ref = fb.measure(P)
    fa_ref_after = fa.measure(P)
    fa.pack(torch.from_numpy(Ua).to(cuda_device).to(CDTYPE[prec]), P)
    fa_ref_before = fa.measure(P)
    for row, (F, th) in zip(got, (fa_ref_before, fb_ref, fa_ref_after)):
        assert _close(row[0], F[0]) and _close(row[1], th[0]), (row, F, th)
        assert row[0] == F[0] and row[1] == th[0]      # same kernels, same order: the header promises the same bits
    assert got[2][0] > got[0][0]                       # the sweep raised F: call 3 really saw the changed field
    if prec == "f64":                                  # and the numbers are the paper's F and theta, not just consistent
        assert _close(got[0][0], oracle.functional(Ua, big)) and abs(got[0][1] / oracle.theta(Ua, big) - 1) < 1e-10
    fa.close()
    fb.close()


@pytest.mark.gpu
def test_coulomb_per_slice_and_no_change_in_free_memory(cuda_device):
    """Coulomb gauge: 2 N_t outputs, (F_t, theta_t) interleaved.  After one call (whose first use on a device looks up
    the scratch address and loads the kernels) further calls leave the device's free memory where it was."""
    dims = (8, 6, 6, 8)
    fld = gf.GaugeField(dims, gauge=gf.GF_COULOMB, precisions=("f64",), device=cuda_device)
    fld.pack(torch.from_numpy(gi.smooth_random_gauge(dims, 0.5, 21)).to(cuda_device), gf.GF_F64)
    out = torch.full((2, dims[0], 2), float("nan"), dtype=torch.float64, device=cuda_device)
    _static(fld, gf.GF_F64, out[0])
    torch.cuda.synchronize(cuda_device)
    free_before = torch.cuda.mem_get_info(cuda_device)[0]
    _static(fld, gf.GF_F64, out[0])
    _static(fld, gf.GF_F64, out[1])
    torch.cuda.synchronize(cuda_device)
    assert torch.cuda.mem_get_info(cuda_device)[0] == free_before
    F, th = fld.measure(gf.GF_F64)
    got = out.cpu().numpy()
    for call in got:
        for t in range(dims[0]):
            assert _close(call[t, 0], F[t]) and _close(call[t, 1], th[t]), (t, call[t], F[t], th[t])
    assert len(set(np.round(got[0][:, 1], 15))) == dims[0]     # the slices differ: an index slip would show
    fld.close()


def test_sizes_beyond_the_static_scratch_are_refused_with_a_reason():
    """The limit is checked on the host before anything touches the GPU, so this runs anywhere: 64^4 needs 131072
    partial sums, the array holds GF_STATIC_MAX_BLOCKS = 65536; the paper's per-GPU lattices (48^4, 64^3 x 32) fit."""
    with pytest.raises(gf.GFError) as e:
        binding.gf_measure_static((64, 64, 64, 64), gf.GF_LANDAU, gf.GF_F64, 18, 256, 256, 0)
    assert e.value.code == gf.GF_EINVAL
    assert "131072" in str(e.value) and "GF_STATIC_MAX_BLOCKS = 65536" in str(e.value) and "gf_measure" in str(e.value)
    assert gf.GF_STATIC_MAX_BLOCKS == 65536
    # argument errors carry their own text too (there is no context to ask)
    for args, word in ((((4, 4, 4, 5), 0, gf.GF_F64, 18, 256, 256, 0), "even"),
                       (((4, 4, 4, 4), 0, gf.GF_MIXED, 18, 256, 256, 0), "precision"),
                       (((4, 4, 4, 4), 0, gf.GF_F64, 18, 0, 256, 0), "NULL"),
                       (((4, 4, 4, 4), 0, gf.GF_F64, 18, 264, 256, 0), "16-byte"),
                       (((4, 4, 4, 4), 0, gf.GF_F64, 18, 256, 260, 0), "8-byte")):
        with pytest.raises(gf.GFError) as e:
            binding.gf_measure_static(*args)
        assert e.value.code == gf.GF_EINVAL and word in str(e.value), str(e.value)


@pytest.mark.gpu
def test_largest_lattices_that_fit(cuda_device):
    """64^3 x 32 (the paper's per-GPU lattice of Fig. 3) uses every one of the 65536 partial sums: fp32 / 12-real
    storage (1.6 GB), static path against gf_measure."""
    dims = (32, 64, 64, 64)
    fld = gf.GaugeField(dims, recon=12, precisions=("f32",), device=cuda_device)
    U = gi.torch_hot_links(dims, 5, device=cuda_device).to(torch.complex64)
    fld.pack(U, gf.GF_F32)
    del U
    out = torch.full((2,), float("nan"), dtype=torch.float64, device=cuda_device)
    _static(fld, gf.GF_F32, out)
    F, th = fld.measure(gf.GF_F32)
    got = out.cpu().numpy()
    assert got[0] == F[0] and got[1] == th[0], (got, F, th)
    assert abs(got[0]) < 1e-2 and 1.0 < got[1] < 20.0          # a hot field: F ~ 0, theta of order N_d
    fld.close()
