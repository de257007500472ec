"""The fix loop without a host round trip per evaluation (gf_set_fix_runahead, include/gf.h): evaluation blocks
are enqueued ahead, the reduction kernel takes the stopping decision on the device and the half-sweeps enqueued
behind it leave the field alone.  Required: links, iteration count, theta and the Philox stream bitwise those of
the loop that waits for every theta (run-ahead 0) -- which the other test files compare with the oracle -- and,
directly, the oracle's iteration count and field."""
import numpy as np
import pytest
import torch

import gf_inputs as gi
import oracle
import paper_1305_3440_b200 as gf

pytestmark = pytest.mark.gpu


def run_fix(cuda_device, U, dims, runahead, *, gauge=gf.GF_LANDAU, algo=gf.GF_OVERRELAX, omega=1.7, p=0.0, mode=gf.GF_F64,
            recon=18, target=1e-12, max_iter=3000, check_every=5, seed=7, defer=False, after=0):
    """Returns (rc, iterations, theta, Philox counter after the call, launches, fixed fp field, [G])."""
    mixed = mode in (gf.GF_MIXED, gf.GF_MIXED_EXACT)
    precs = ("f64", "f32") if mixed else (("f64",) if mode == gf.GF_F64 else ("f32",))
    fld = gf.GaugeField(dims, gauge=gauge, recon=recon, precisions=precs, seed=seed, device=cuda_device)
    Ud = torch.from_numpy(U).to(cuda_device)
    if mode in (gf.GF_F64, gf.GF_MIXED_EXACT):
        fld.pack(Ud, gf.GF_F64)
    if mode in (gf.GF_F32, gf.GF_MIXED):
        fld.pack(Ud.to(torch.complex64), gf.GF_F32)
    if mode == gf.GF_MIXED_EXACT:
        fld.attach_transform(("f64", "f32"))
    if defer:
        fld.attach_transform(("f64",))
        fld.set_coulomb_mode(True, False)
    fld.set_fix_runahead(runahead)
    n0 = gf.gf_launch_count(fld.ctx)
    rc, it, th = fld.fix_until(algo, omega, p, mode, target, max_iter, check_every)
    launches = gf.gf_launch_count(fld.ctx) - n0
    counter = gf.gf_get_counter(fld.ctx)
    out_prec = gf.GF_F32 if mode == gf.GF_F32 else gf.GF_F64
    if after:            # the stop word is clear again: sweeps that follow the loop act on the field
        fld.iterate(after, algo, omega, p, out_prec)
    res = fld.unpack(out_prec, torch.complex128).cpu().numpy()
    F, ths = fld.measure(out_prec)
    fld.close()
    return rc, it, th, counter, launches, res, ths


@pytest.mark.parametrize("depth", [1, 4, 8])
@pytest.mark.parametrize("mode,recon", [(gf.GF_F64, 18), (gf.GF_F64, 12), (gf.GF_F32, 18), (gf.GF_MIXED, 18), (gf.GF_MIXED_EXACT, 12)])
def test_runahead_equals_the_waiting_loop_landau(cuda_device, depth, mode, recon):
    dims = (6, 4, 8, 6)
    U = gi.smooth_random_gauge(dims, 0.4, 314)
    target = 1e-6 if mode == gf.GF_F32 else 1e-12
    a = run_fix(cuda_device, U, dims, 0, mode=mode, recon=recon, target=target)
    b = run_fix(cuda_device, U, dims, depth, mode=mode, recon=recon, target=target)
    assert a[0] == b[0] == gf.GF_OK
    assert a[1] == b[1] and a[2] == b[2] and a[3] == b[3]          # iterations, theta, Philox counter
    assert np.array_equal(a[5], b[5])                                # the fixed field, bitwise
    assert b[4] >= a[4]                                              # the blocks enqueued ahead were launched (and did nothing)


@pytest.mark.parametrize("check_every,max_iter", [(1, 3000), (7, 3000), (10, 23), (4, 8), (5, 0)])
def test_runahead_iteration_accounting(cuda_device, check_every, max_iter):
    """Evaluation points (multiples of check_every and the last iteration), max_iter reached without convergence,
    max_iter that is not a multiple of check_every, and sweeps after the loop (the stop word is clear again)."""
    dims = (4, 6, 4, 4)
    U = gi.smooth_random_gauge(dims, 0.4, 2718)
    a = run_fix(cuda_device, U, dims, 0, check_every=check_every, max_iter=max_iter, after=2)
    b = run_fix(cuda_device, U, dims, 4, check_every=check_every, max_iter=max_iter, after=2)
    assert a[:4] == b[:4]
    assert a[0] == (gf.GF_OK if max_iter == 3000 else gf.GF_NOT_CONVERGED)
    assert np.array_equal(a[5], b[5]) and np.array_equal(a[6], b[6])
    if max_iter == 3000:                                             # and the oracle agrees on where the loop stops
        Uo = U.copy()
        it, th, conv = oracle.fix_until(Uo, dims, algo=oracle.OVERRELAX, omega=1.7, theta_target=1e-12, max_iter=3000, check_every=check_every)
        assert conv and abs(it - b[1]) <= check_every
        if it == b[1]:
            for _ in range(2):
                for parity in (0, 1):
                    oracle.sweep(Uo, dims, parity, algo=oracle.OVERRELAX, omega=1.7)
            assert np.abs(b[5] - Uo).max() < 1e-9


@pytest.mark.parametrize("defer", [False, True])
@pytest.mark.parametrize("recon", [18, 12])
def test_runahead_coulomb_stochastic(cuda_device, defer, recon):
    """Coulomb gauge: the device decides on max_t theta_t; the Philox stream (seed, half-sweep counter) must be where the
    waiting loop leaves it, also with deferred temporal links.  The oracle's fix loop gives the iteration count."""
    dims = (6, 6, 6, 6)
    U = gi.smooth_random_gauge(dims, 0.4, 1618)
    kw = dict(gauge=gf.GF_COULOMB, algo=gf.GF_STOCHASTIC, omega=1.0, p=0.8, recon=recon, seed=2013, check_every=4, defer=defer, after=1)
    a = run_fix(cuda_device, U, dims, 0, **kw)
    b = run_fix(cuda_device, U, dims, 3, **kw)
    assert a[0] == b[0] == gf.GF_OK and a[:4] == b[:4]
    assert np.array_equal(a[5], b[5]) and np.array_equal(a[6], b[6])
    if recon == 18 and not defer:
        Uo = U.copy()
        it, th, conv = oracle.fix_until(Uo, dims, gauge=oracle.COULOMB, algo=oracle.STOCHASTIC, p=0.8, seed=2013,
                                        theta_target=1e-12, max_iter=3000, check_every=4)
        assert conv and abs(it - b[1]) <= 4


def test_runahead_target_met_at_the_first_evaluation(cuda_device):
    """theta below the target at the first evaluation: every block enqueued behind it must be a no-op."""
    dims = (4, 4, 4, 6)
    U = gi.smooth_random_gauge(dims, 0.3, 99)
    a = run_fix(cuda_device, U, dims, 0, target=10.0, check_every=3)
    b = run_fix(cuda_device, U, dims, 8, target=10.0, check_every=3)
    assert a[1] == b[1] == 3 and a[:4] == b[:4] and np.array_equal(a[5], b[5])
    Uo = U.copy()
    for _ in range(3):
        for parity in (0, 1):
            oracle.sweep(Uo, dims, parity, algo=oracle.OVERRELAX, omega=1.7)
    assert np.abs(b[5] - Uo).max() < 1e-12                           # exactly three iterations were applied
    assert b[4] == a[4] + 7 * (2 * 3 + 2)                            # seven more blocks of 6 half-sweeps + 2 reduction kernels


def test_runahead_argument_errors(cuda_device):
    fld = gf.GaugeField((4, 4, 4, 4), precisions=("f64",), device=cuda_device)
    for bad in (-1, 9):
        with pytest.raises(gf.GFError):
            fld.set_fix_runahead(bad)
    fld.close()


def test_runahead_hides_the_round_trip(cuda_device):
    """On a lattice whose block of iterations is shorter than a host round trip the run-ahead loop is faster
    (8^4, theta every iteration: 5.3 against 7.5 ms)."""
    dims = (8, 8, 8, 8)
    U = torch.from_numpy(gi.smooth_random_gauge(dims, 0.5, 5)).to(cuda_device)
    times = {}
    for depth in (0, 4):
        fld = gf.GaugeField(dims, precisions=("f64",), device=cuda_device)
        fld.set_fix_runahead(depth)
        best = 1e9
        for _ in range(3):
            fld.pack(U, gf.GF_F64)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64, 1e-12, 5000, 1)
            b.record()
            torch.cuda.synchronize()
            best = min(best, a.elapsed_time(b))
        times[depth] = (best, it)
        fld.close()
    assert times[0][1] == times[4][1]
    assert times[4][0] < 0.95 * times[0][0], times           # measured 0.71


# ------------------------------------------------------------------------------ re-projection inside the fix loop

def _long_run(cuda_device, U, dims, prec_name, reunit, runahead=4, iters=1500, check=50):
    prec = gf.GF_F32 if prec_name == "f32" else gf.GF_F64
    cd = torch.complex64 if prec_name == "f32" else torch.complex128
    fld = gf.GaugeField(dims, precisions=(prec_name,), device=cuda_device)
    fld.pack(torch.from_numpy(U).to(cuda_device).to(cd), prec)
    fld.set_reunitarize_every(reunit)
    fld.set_fix_runahead(runahead)
    rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, prec, 0.0, iters, check)       # target 0: runs all iterations
    out = fld.unpack(prec, torch.complex128).cpu().numpy()
    F, _ = fld.measure(prec)
    fld.close()
    return rc, it, th, out, F[0]


def test_reprojection_keeps_a_long_fp32_run_in_SU3(cuda_device):
    """fp32 links lose unitarity linearly with the number of site updates; with gf_set_reunitarize_every the defect stays
    at the fp32 rounding level (both judged by the ORACLE's checker), the plaquette stays that of the input to fp32
    accuracy, and the run-ahead loop takes bitwise the same path as the loop that waits."""
    dims = (8, 8, 8, 8)
    U = gi.hot_links(dims, 4)
    P0 = oracle.plaquette(U, dims)
    plain = _long_run(cuda_device, U, dims, "f32", 0)
    kept = _long_run(cuda_device, U, dims, "f32", 100)
    waits = _long_run(cuda_device, U, dims, "f32", 100, runahead=0)
    assert plain[1] == kept[1] == 1500 and plain[0] == kept[0] == gf.GF_NOT_CONVERGED
    d_plain = oracle.unitarity_defect(np.ascontiguousarray(plain[3]), dims)
    d_kept = oracle.unitarity_defect(np.ascontiguousarray(kept[3]), dims)
    # measured with the default solver (K and the SU(2) solves in fp64 registers, products g U in fp32): 7.9e-5 without
    # re-projection, 9e-8 with it (the all-fp32 solver of round 2 lost unitarity faster: 1e-4 .. 8e-4)
    assert d_plain[0] > 3e-5 and d_kept[0] < 2e-6 and d_kept[1] < 2e-6, (d_plain, d_kept)
    assert abs(oracle.plaquette(np.ascontiguousarray(kept[3]), dims) - P0) < 2e-5
    assert kept[4] >= plain[4] - 1e-6                          # the functional is not worse for it
    assert np.array_equal(kept[3], waits[3]) and kept[2] == waits[2]


def test_reprojection_in_fp64_is_invisible(cuda_device):
    """In fp64 the re-projection moves the links by rounding errors only: same iteration count, links within 1e-12 of the
    run without it, result fixed as judged by the oracle."""
    dims = (4, 6, 6, 4)
    U = gi.smooth_random_gauge(dims, 0.4, 8)
    res = {}
    for reunit in (0, 10):
        fld = gf.GaugeField(dims, precisions=("f64",), device=cuda_device)
        fld.pack(torch.from_numpy(U).to(cuda_device), gf.GF_F64)
        fld.set_reunitarize_every(reunit)
        n0 = gf.gf_launch_count(fld.ctx)
        rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64, 1e-12, 3000, 5)
        res[reunit] = (rc, it, fld.unpack(gf.GF_F64).cpu().numpy(), gf.gf_launch_count(fld.ctx) - n0)
        fld.close()
    assert res[0][0] == res[10][0] == gf.GF_OK and res[0][1] == res[10][1]
    assert np.abs(res[0][2] - res[10][2]).max() < 1e-12
    assert res[10][3] > res[0][3]                              # the re-projection kernels were launched
    assert oracle.theta(np.ascontiguousarray(res[10][2]), dims) < 1e-12
    with pytest.raises(gf.GFError):
        f = gf.GaugeField(dims, precisions=("f64",), device=cuda_device)
        try:
            f.set_reunitarize_every(-1)
        finally:
            f.close()


@pytest.mark.parametrize("runahead", [0, 4])
def test_reprojection_with_the_recorded_transformation(cuda_device, runahead):
    """GF_MIXED_EXACT with gf_set_reunitarize_every: the fp32 links AND the recorded fp32 G(x) are re-projected during the
    fp32 phase; the result is still G U G^dagger of the untouched fp64 input -- plaquette kept to 1e-12, fixed to
    theta < 1e-12 and in SU(3) as judged by the oracle -- and the returned G reproduces it through eq. 3."""
    dims = (6, 4, 4, 6)
    U = gi.smooth_random_gauge(dims, 0.5, 21)
    fld = gf.GaugeField(dims, recon=12, precisions=("f64", "f32"), device=cuda_device)
    fld.pack(torch.from_numpy(U).to(cuda_device), gf.GF_F64)
    fld.attach_transform(("f64", "f32"))
    fld.set_mixed_handoff(1e-9)
    fld.set_reunitarize_every(10)
    fld.set_fix_runahead(runahead)
    rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_MIXED_EXACT, 1e-12, 5000, 5)
    assert rc == gf.GF_OK and th < 1e-12
    W = np.ascontiguousarray(fld.unpack(gf.GF_F64).cpu().numpy())
    G = np.ascontiguousarray(fld.transform(gf.GF_F64).cpu().numpy())
    fld.close()
    assert oracle.theta(W, dims) < 1e-12
    assert abs(oracle.plaquette(W, dims) - oracle.plaquette(U, dims)) < 1e-12
    du, dd = oracle.unitarity_defect(W, dims)
    assert du < 1e-12 and dd < 1e-12
    assert np.abs(oracle.apply_transform(U, G, dims) - W).max() < 1e-11


# ------------------------------------------------------------------------------ hand-off when fp32 stalls

@pytest.mark.parametrize("mode,recon", [(gf.GF_MIXED_EXACT, 18), (gf.GF_MIXED_EXACT, 12), (gf.GF_MIXED, 18)])
def test_mixed_precision_hands_over_when_fp32_stops_lowering_theta(cuda_device, mode, recon):
    """gf_set_mixed_stall: with a target (1e-20) and a hand-off theta (1e-15) that fp32 can never reach the fp32 phase ends at the first
    evaluation at which theta has not fallen; the fp64 phase finishes.  The run-ahead loop (decision on the device) and
    the loop that waits take bitwise the same path; the result is fixed, in SU(3) and -- for GF_MIXED_EXACT -- has the
    input's plaquette to 1e-12, all as judged by the oracle."""
    dims = (6, 6, 4, 6)
    U = gi.smooth_random_gauge(dims, 0.5, 33)
    out = {}
    for runahead in (0, 4):
        fld = gf.GaugeField(dims, recon=recon, precisions=("f64", "f32"), device=cuda_device)
        Ud = torch.from_numpy(U).to(cuda_device)
        if mode == gf.GF_MIXED_EXACT:
            fld.pack(Ud, gf.GF_F64)
            fld.attach_transform(("f64", "f32"))
        else:
            fld.pack(Ud.to(torch.complex64), gf.GF_F32)
        fld.set_mixed_handoff(1e-15)
        fld.set_mixed_stall(1.0)
        fld.set_fix_runahead(runahead)
        rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, mode, 1e-20, 3000, 5)
        out[runahead] = (rc, it, th, gf.gf_get_counter(fld.ctx), fld.unpack(gf.GF_F64).cpu().numpy())
        fld.close()
    a, b = out[0], out[4]
    assert a[0] == b[0] == gf.GF_OK and a[1:4] == b[1:4] and np.array_equal(a[4], b[4])
    # theta < 1e-20 is far below what fp32 reaches: the run can only have converged through the stall hand-off
    assert b[1] < 3000 and b[2] < 1e-20
    W = np.ascontiguousarray(b[4])
    assert oracle.theta(W, dims) < 2e-20
    du, dd = oracle.unitarity_defect(W, dims)
    assert du < 1e-12 and dd < 1e-12
    assert abs(oracle.plaquette(W, dims) - oracle.plaquette(U, dims)) < (1e-12 if mode == gf.GF_MIXED_EXACT else 1e-6)
    with pytest.raises(gf.GFError):
        f = gf.GaugeField(dims, precisions=("f64",), device=cuda_device)
        try:
            f.set_mixed_stall(1.5)
        finally:
            f.close()
