"""Full-field parity at the sizes and in the launch configuration bench.py times (BASELINE.json configs[2] and
configs[4]): every link of the 32^4 lattice after each half-sweep, and F / theta after 10 iterations, for all four
storage variants (fp64 / fp32 x 18- / 12-real, default tuning -- this covers the register-capped fp32/18 entry
point and the one-lane-per-site, lazy-third-row fp64/12 path at full size); one full stochastic Coulomb iteration of 32^3 x 64;
the mixed-precision runs at 32^4 judged by the oracle; the Coulomb fix loop's iteration count on a 16 x 16^3 replica.
The oracle is fed the field the device holds (unpacked after gf_pack: the fp32-rounded input, row 2 rebuilt for
12-real storage) only after that field has been compared with the independently generated input
(assert_pack_round_trip), and runs on all host cores.  Tolerances are north_star's."""
import numpy as np
import pytest
import torch

import gf_inputs as gi
import oracle
import paper_1305_3440_b200 as gf
from gpu_helpers import assert_pack_round_trip

pytestmark = pytest.mark.gpu

PREC = {"f64": gf.GF_F64, "f32": gf.GF_F32}
CDTYPE = {"f64": torch.complex128, "f32": torch.complex64}
LINK_TOL = {"f64": 1e-12, "f32": 1e-5}
REL_TOL = {"f64": 1e-10, "f32": 1e-5}


@pytest.fixture(autouse=True)
def all_host_cores():
    oracle.set_threads(0)
    yield
    oracle.set_threads(1)


def held_by_device(fld, prec):
    return np.ascontiguousarray(fld.unpack(PREC[prec], torch.complex128).cpu().numpy())


@pytest.mark.parametrize("prec,recon", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
def test_32_4_full_field_against_oracle(cuda_device, prec, recon):
    """configs[2]: 32^4, eps 0.6 smooth field + Haar gauge transform, overrelaxation omega = 1.7, the library's defaults
    (what bench.py times).

    Every link within north_star's tolerance -- 1e-12 (fp64), 1e-5 (fp32) -- of ONE oracle that runs on freely from the
    input, after each of the two half-sweeps; then F and theta after 10 iterations against the same oracle.  With fp32
    storage the default solver accumulates K(x) and runs the SU(2) solves in fp64 registers: what is left is the fp32
    rounding of the products g U (measured 2.2e-6 after the iteration, 1.2e-7 in the median).  The all-fp32 solver
    (gf_set_solver_precision(GF_F32), faster, opt-in) is checked at the end: its error per site update is
    eps32 |K| / |v| ("Tolerances"), and among the 524 288 sites of a half-sweep of this field there is one
    whose SU(2) projection |v| is 45 times smaller than its block of K: 8.8e-6 after its own half-sweep, 1.08e-5 after
    the second -- above 1e-5, which is why it is not the default."""
    dims = (32, 32, 32, 32)
    U = gi.torch_smooth_random_gauge(dims, 0.6, 1, device=cuda_device).to(CDTYPE[prec])
    fld = gf.GaugeField(dims, recon=recon, precisions=(prec,), device=cuda_device)     # default tuning = what bench.py times
    fld.pack(U, PREC[prec])
    assert_pack_round_trip(fld, PREC[prec], U)
    Uo = held_by_device(fld, prec)                # the one oracle: never re-synchronised with the device
    for parity in (0, 1):
        fld.sweep(parity, gf.GF_OVERRELAX, 1.7, 0.0, PREC[prec])
        oracle.sweep(Uo, dims, parity, oracle.LANDAU, oracle.OVERRELAX, 1.7)
        got = held_by_device(fld, prec)
        err = float(np.abs(got - Uo).max())                                    # all 4 194 304 links
        assert err < LINK_TOL[prec], (prec, recon, parity, err)
        if prec == "f32":
            assert float(np.median(np.abs(got - Uo))) < 2e-7
    del got
    fld.iterate(9, gf.GF_OVERRELAX, 1.7, 0.0, PREC[prec])                       # the call bench.py's step uses
    for it in range(9):
        for parity in (0, 1):
            oracle.sweep(Uo, dims, parity, oracle.LANDAU, oracle.OVERRELAX, 1.7)
    F, th = fld.measure(PREC[prec])
    Fo, tho = oracle.functional(Uo, dims), oracle.theta(Uo, dims)
    assert abs(F[0] / Fo - 1) < REL_TOL[prec], (F[0], Fo)
    assert abs(th[0] / tho - 1) < REL_TOL[prec], (th[0], tho)
    du, dd = oracle.unitarity_defect(held_by_device(fld, prec), dims)           # SU(3) as judged by the oracle
    # fp32: 20 site updates per link, each a product with fp32 rounding; the largest defect among 4.2 million links
    assert du < (1e-12 if prec == "f64" else 5e-5) and dd < (1e-12 if prec == "f64" else 5e-5)
    gdu, gdd = fld.unitarity(PREC[prec])
    assert abs(gdu - du) < (1e-13 if prec == "f64" else 1e-6) and abs(gdd - dd) < (1e-13 if prec == "f64" else 1e-6)
    if prec == "f32":
        # the opt-in all-fp32 solver: within 1e-5 after EACH half-sweep judged from the field the device held before it;
        # carried through both half-sweeps the worst site ends an fp32-sized error away, but above 1e-5
        fld.set_solver_precision(gf.GF_F32)
        fld.pack(U, PREC[prec])
        Uo = held_by_device(fld, prec)            # runs on freely
        Us = Uo.copy()                            # re-synchronised before every half-sweep
        for parity in (0, 1):
            fld.sweep(parity, gf.GF_OVERRELAX, 1.7, 0.0, PREC[prec])
            oracle.sweep(Uo, dims, parity, oracle.LANDAU, oracle.OVERRELAX, 1.7)
            oracle.sweep(Us, dims, parity, oracle.LANDAU, oracle.OVERRELAX, 1.7)
            got = held_by_device(fld, prec)
            assert float(np.abs(got - Us).max()) < 1e-5
            assert float(np.median(np.abs(got - Us))) < 2e-7
            Us = got
        err32 = float(np.abs(got - Uo).max())
        print("all-fp32 solver, %d-real: max |dU| after one free-running iteration %.3e" % (recon, err32))
        assert err32 < 3e-5
    fld.close()


@pytest.mark.parametrize("recon", [18, 12])
def test_config5_full_field_stochastic_coulomb_iteration(cuda_device, recon):
    """configs[4]: 32^3 x 64 Coulomb gauge, fp64, stochastic relaxation p = 0.8, Philox seed 2013: one whole
    iteration (2 097 152 site updates, the same Philox stream on both sides), every link compared; then the
    per-slice F_t and theta_t."""
    dims = (64, 32, 32, 32)
    U = gi.torch_smooth_random_gauge(dims, 0.6, 1, device=cuda_device)
    fld = gf.GaugeField(dims, gauge=gf.GF_COULOMB, recon=recon, precisions=("f64",), seed=2013, device=cuda_device)
    fld.pack(U, gf.GF_F64)
    assert_pack_round_trip(fld, gf.GF_F64, U)
    del U
    Uo = held_by_device(fld, "f64")
    for parity in (0, 1):
        fld.sweep(parity, gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64)
        oracle.sweep(Uo, dims, parity, oracle.COULOMB, oracle.STOCHASTIC, 1.0, 0.8, seed=2013, half_sweep_counter=parity)
        err = float(np.abs(held_by_device(fld, "f64") - Uo).max())
        assert err < 1e-12, (parity, err)
    F, th = fld.measure(gf.GF_F64)
    assert np.allclose(F, oracle.functional(Uo, dims, oracle.COULOMB), rtol=1e-10, atol=0)
    assert np.allclose(th, oracle.theta(Uo, dims, oracle.COULOMB), rtol=1e-10, atol=0)
    fld.close()


def test_coulomb_16x16_3_fix_loop_iteration_count(cuda_device):
    """A 16 x 16^3 replica of configs[4] (same recipe, Philox seed 2013, p = 0.8, theta_t every 20 iterations):
    gf_fix_until stops within one evaluation interval of the oracle's fix loop."""
    dims = (16, 16, 16, 16)
    U = gi.smooth_random_gauge(dims, 0.6, 1)
    Uo = U.copy()
    it_o, th_o, conv = oracle.fix_until(Uo, dims, oracle.COULOMB, oracle.STOCHASTIC, 1.0, 0.8, seed=2013,
                                        theta_target=1e-12, max_iter=50000, check_every=20)
    assert conv
    fld = gf.GaugeField(dims, gauge=gf.GF_COULOMB, precisions=("f64",), seed=2013, device=cuda_device)
    fld.pack(torch.from_numpy(U).to(cuda_device), gf.GF_F64)
    rc, it, th = fld.fix_until(gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64, 1e-12, 50000, 20)
    assert rc == gf.GF_OK and th < 1e-12
    print("coulomb 16x16^3: gpu %d iterations, oracle %d" % (it, it_o))
    assert abs(it - it_o) <= 20, (it, it_o)
    got = held_by_device(fld, "f64")
    assert oracle.theta(got, dims, oracle.COULOMB).max() < 1.01e-12            # the oracle agrees every slice is fixed
    assert abs(oracle.plaquette(got, dims) - oracle.plaquette(U, dims)) < 1e-12
    fld.close()


@pytest.mark.parametrize("mode", ["mixed", "mixed_exact"])
def test_32_4_mixed_precision_judged_by_the_oracle(cuda_device, mode):
    """configs[2], "mixed (fp32 sweeps to theta < 1e-6, then fp64 to 1e-12)": the result is fixed, in SU(3) and on
    the gauge orbit of the input AS JUDGED BY THE ORACLE.  GF_MIXED keeps the orbit to fp32 accuracy (reading A15),
    GF_MIXED_EXACT to fp64 accuracy, and returns the transformation that does it."""
    dims = (32, 32, 32, 32)
    U = gi.torch_smooth_random_gauge(dims, 0.6, 1, device=cuda_device)
    fld = gf.GaugeField(dims, precisions=("f64", "f32"), device=cuda_device)
    fld.pack(U, gf.GF_F64)
    assert_pack_round_trip(fld, gf.GF_F64, U)
    U0 = held_by_device(fld, "f64")
    P0 = oracle.plaquette(U0, dims)
    if mode == "mixed":
        fld.pack(U.to(torch.complex64), gf.GF_F32)
        rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_MIXED, 1e-12, 50000, 10)
    else:
        fld.attach_transform(("f64", "f32"))
        rc, it, th = fld.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_MIXED_EXACT, 1e-12, 50000, 10)
    assert rc == gf.GF_OK and th < 1e-12 and it % 10 == 0
    got = held_by_device(fld, "f64")
    tho = oracle.theta(got, dims)
    assert tho < 1e-12 and abs(tho / th - 1) < 1e-6, (tho, th)                  # theta returned is the fp64 field's
    du, dd = oracle.unitarity_defect(got, dims)
    assert du < 1e-12 and dd < 1e-12
    drift = abs(oracle.plaquette(got, dims) - P0)
    print("%s: %d iterations, theta %.3e, plaquette drift %.3e" % (mode, it, tho, drift))
    if mode == "mixed":
        assert drift < 1e-5
    else:
        assert drift < 1e-12
        G = np.ascontiguousarray(fld.transform(gf.GF_F64).cpu().numpy())
        assert np.abs(oracle.apply_transform(U0, G, dims) - got).max() < 1e-11  # eq. 3 by the oracle: G U0 G^dagger
    assert oracle.functional(got, dims) > oracle.functional(U0, dims) + 0.3
    fld.close()


@pytest.mark.parametrize("prec,recon", [("f64", 18), ("f32", 12)])
def test_32_4_accumulated_transformation_full_field(cuda_device, prec, recon):
    """NEXT-1 at configs[2] size in the default launch configuration with accumulation: G(x) after one iteration
    against the oracle's sweep_accumulate over the whole lattice, and the links with it."""
    dims = (32, 32, 32, 32)
    U = gi.torch_smooth_random_gauge(dims, 0.6, 1, device=cuda_device).to(CDTYPE[prec])
    fld = gf.GaugeField(dims, recon=recon, precisions=(prec,), device=cuda_device)
    fld.pack(U, PREC[prec])
    assert_pack_round_trip(fld, PREC[prec], U)
    del U
    fld.attach_transform((prec,))
    Uo = held_by_device(fld, prec)
    Go = oracle.identity_transform(dims)
    for parity in (0, 1):
        fld.sweep(parity, gf.GF_OVERRELAX, 1.7, 0.0, PREC[prec])
        oracle.sweep_accumulate(Uo, Go, dims, parity, oracle.LANDAU, oracle.OVERRELAX, 1.7)
    G = fld.transform(PREC[prec], torch.complex128).cpu().numpy()
    assert np.abs(G - Go).max() < LINK_TOL[prec]                     # every G(x) is the product of ONE site update so far
    # the links have been through both half-sweeps (fp32 storage: default solver in fp64 registers)
    assert np.abs(held_by_device(fld, prec) - Uo).max() < LINK_TOL[prec]
    fld.close()


def _max_abs_diff_by_slices(a, b):
    """max |a - b| over two large host arrays without a full-size temporary (one time slice at a time)."""
    return max(float(np.abs(a[t] - b[t]).max()) for t in range(a.shape[0]))


@pytest.mark.parametrize("prec,recon", [("f64", 18), ("f64", 12)])
def test_64_4_full_field_one_iteration_against_oracle(cuda_device, prec, recon):
    """configs[3] at full size: 64^4 = 16.8 M sites (9.66 GB of fp64 links, byte offsets beyond 2^32 in every link block),
    omega = 1.8, default launch configuration: all 67 million links after parity 0 and after parity 1 within 1e-12 of the
    oracle (running on from its own field, all host cores), then F and theta of the swept field to 1e-10.  Host memory:
    two canonical copies of the field (19 GB); the comparison goes slice by slice."""
    dims = (64, 64, 64, 64)
    U = gi.torch_smooth_random_gauge(dims, 0.6, 4, device=cuda_device)
    fld = gf.GaugeField(dims, recon=recon, precisions=(prec,), device=cuda_device)
    fld.pack(U, PREC[prec])
    assert_pack_round_trip(fld, PREC[prec], U)                            # all 67 M links, byte offsets beyond 2^32 included
    del U
    torch.cuda.empty_cache()
    Uo = fld.unpack(PREC[prec], torch.complex128).cpu().numpy()           # what the device holds (row 2 rebuilt for 12-real)
    torch.cuda.empty_cache()
    for parity in (0, 1):
        fld.sweep(parity, gf.GF_OVERRELAX, 1.8, 0.0, PREC[prec])
        oracle.sweep(Uo, dims, parity, oracle.LANDAU, oracle.OVERRELAX, 1.8)
        got = fld.unpack(PREC[prec], torch.complex128).cpu().numpy()
        torch.cuda.empty_cache()
        err = _max_abs_diff_by_slices(got, Uo)
        assert err < LINK_TOL[prec], (prec, recon, parity, err)
        del got
    F, th = fld.measure(PREC[prec])
    Fo, tho = oracle.functional(Uo, dims), oracle.theta(Uo, dims)
    assert abs(F[0] / Fo - 1) < REL_TOL[prec] and abs(th[0] / tho - 1) < REL_TOL[prec], (F[0], Fo, th[0], tho)
    assert abs(fld.plaquette(PREC[prec]) - oracle.plaquette(Uo, dims)) < 1e-12
    fld.close()
