"""The host-buffer entry points bench.py's end-to-end measurement uses (gf_load_host / gf_store_host):
canonical field in pinned HOST memory -> device -> sweeps -> back to the host, against the oracle; and
the pipelined form (several lattices in flight, one context / stream / host thread each)."""
import threading

import numpy as np
import pytest
import torch

import gf_inputs as gi
import oracle
import paper_1305_3440_b200 as gf

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("prec,cdtype,recon,tol", [("f64", torch.complex128, 18, 1e-12), ("f64", torch.complex128, 12, 1e-12),
                                                   ("f32", torch.complex64, 18, 1e-5)])
def test_load_sweep_store_through_host_buffers(cuda_device, prec, cdtype, recon, tol):
    dims = (6, 4, 8, 4)
    P = gf.GF_F64 if prec == "f64" else gf.GF_F32
    U = gi.smooth_random_gauge(dims, 0.5, 61)
    host = torch.from_numpy(U).to(cdtype).pin_memory()
    fld = gf.GaugeField(dims, recon=recon, precisions=(prec,), device=cuda_device, staging=True)
    fld.load_host(host, P)
    fld.iterate(2, gf.GF_OVERRELAX, 1.6, 0.0, P)
    out = torch.empty_like(host).pin_memory()
    fld.store_host(out, P)                           # synchronises: `out` is complete
    Uo = np.ascontiguousarray(host.numpy().astype(np.complex128))
    for _ in range(2):
        for parity in (0, 1):
            oracle.sweep(Uo, dims, parity, algo=oracle.OVERRELAX, omega=1.6)
    assert np.abs(out.numpy().astype(np.complex128) - Uo).max() < 2 * tol
    assert torch.equal(host, torch.from_numpy(U).to(cdtype))           # the input buffer is not written
    fld.close()


def test_pipelined_lattices_do_not_disturb_each_other(cuda_device):
    """Four lattices in flight as in bench.py's e2e leg (own context, stream, pinned buffer and host
    thread): every one ends bitwise where a lone run of the same input ends."""
    dims = (8, 8, 8, 8)
    inputs = [torch.from_numpy(gi.smooth_random_gauge(dims, 0.5, 70 + i)).pin_memory() for i in range(4)]
    want = []
    for h in inputs:
        f = gf.GaugeField(dims, precisions=("f64",), device=cuda_device, staging=True)
        f.load_host(h, gf.GF_F64)
        f.iterate(6, gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64)
        o = torch.empty_like(h).pin_memory()
        f.store_host(o, gf.GF_F64)
        want.append(o.clone())
        f.close()
    fields, outs = [], [torch.empty_like(h).pin_memory() for h in inputs]
    for _ in inputs:
        with torch.cuda.stream(torch.cuda.Stream(device=cuda_device)):
            fields.append(gf.GaugeField(dims, precisions=("f64",), device=cuda_device, staging=True))
    errors = []

    def worker(f, h, o):
        try:
            torch.cuda.set_device(cuda_device)
            for _ in range(3):                       # the same step three times over: last result must match
                f.load_host(h, gf.GF_F64)
                for _ in range(3):
                    f.iterate(2, gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64)
                    f.measure(gf.GF_F64)
                f.store_host(o, gf.GF_F64)
        except Exception as e:                       # surfaced below
            errors.append(e)

    threads = [threading.Thread(target=worker, args=a) for a in zip(fields, inputs, outs)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    torch.cuda.synchronize()
    assert not errors, errors
    for o, w in zip(outs, want):
        assert torch.equal(o, w)
    for f in fields:
        f.close()


@pytest.mark.parametrize("gate", [True, False, None])
def test_host_pipeline_ensemble_matches_lone_runs_and_the_oracle(cuda_device, gate):
    """HostPipeline (the form bench.py's e2e leg uses): seven configurations in host memory through three lanes;
    every fixed field is bitwise the one a lone GaugeField produces, the iteration counts are the same, and one
    of them is followed by the oracle (same count within one check interval, F and theta to 1e-10)."""
    from paper_1305_3440_b200.pipeline import HostPipeline
    dims = (4, 6, 4, 8)
    inputs = [torch.from_numpy(gi.smooth_random_gauge(dims, 0.4, 900 + i)) for i in range(7)]

    def work(f):
        return f.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64, 1e-12, 4000, 5)

    want, want_res = [], []
    lone = gf.GaugeField(dims, precisions=("f64",), device=cuda_device, staging=True)
    for h in inputs:
        b = h.clone().pin_memory()
        lone.load_host(b, gf.GF_F64)
        want_res.append(work(lone))
        lone.store_host(b, gf.GF_F64)
        want.append(b.clone())
    lone.close()

    pipe = HostPipeline(dims, precisions=("f64",), lanes=3, device=cuda_device, gate=gate)
    bufs = [h.clone().pin_memory() for h in inputs]
    res = pipe.process(bufs, work, gf.GF_F64)
    assert len(pipe.done_at) == 7 and pipe.steady_seconds_per_item() > 0
    for b, w, r, wr in zip(bufs, want, res, want_res):
        assert torch.equal(b, w)
        assert r[0] == gf.GF_OK and r[1] == wr[1] and r[2] == wr[2]
    # a second batch through the same lanes (fewer items than lanes)
    bufs2 = [h.clone().pin_memory() for h in inputs[:2]]
    pipe.process(bufs2, work, gf.GF_F64)
    assert torch.equal(bufs2[0], want[0]) and torch.equal(bufs2[1], want[1])
    pipe.close()

    Uo = np.ascontiguousarray(inputs[3].numpy())
    it, th, conv = oracle.fix_until(Uo, dims, algo=oracle.OVERRELAX, omega=1.7, theta_target=1e-12, max_iter=4000, check_every=5)
    assert conv
    assert abs(it - res[3][1]) <= 5
    got = np.ascontiguousarray(bufs[3].numpy())
    assert oracle.theta(got, dims) < 1e-12                       # fixed, as judged by the oracle
    assert abs(oracle.plaquette(got, dims) - oracle.plaquette(np.ascontiguousarray(inputs[3].numpy()), dims)) < 1e-12
    if it == res[3][1]:
        assert abs(oracle.functional(got, dims) / oracle.functional(Uo, dims) - 1) < 1e-10
        assert np.abs(got - Uo).max() < 1e-9


def test_host_pipeline_surfaces_errors(cuda_device):
    from paper_1305_3440_b200.pipeline import HostPipeline
    dims = (4, 4, 4, 4)
    pipe = HostPipeline(dims, precisions=("f64",), lanes=2, device=cuda_device)
    bufs = [torch.from_numpy(gi.smooth_random_gauge(dims, 0.4, 5)).pin_memory() for _ in range(3)]
    with pytest.raises(gf.GFError):
        pipe.process(bufs, lambda f: f.iterate(1, gf.GF_OVERRELAX, 2.5, 0.0, gf.GF_F64), gf.GF_F64)   # omega out of range
    pipe.close()


def test_errors_raised_in_a_lane_thread_reach_the_caller(cuda_device, tmp_path):
    """A callback that fails inside a lane's thread -- with an ordinary exception or with SystemExit, which threading
    would swallow -- is re-raised by the pipeline; the command line turns a file of the wrong shape into an exit message
    naming the file instead of tripping over the missing result."""
    from paper_1305_3440_b200 import fix
    from paper_1305_3440_b200.pipeline import HostPipeline
    dims = (4, 4, 4, 4)
    pipe = HostPipeline(dims, precisions=("f64",), lanes=2, device=cuda_device)

    def fill(i, buf):
        if i == 1:
            raise SystemExit("item 1 cannot be read")
        buf.copy_(torch.from_numpy(gi.smooth_random_gauge(dims, 0.4, 5)))

    with pytest.raises(SystemExit, match="item 1"):
        pipe.process_stream(3, fill, lambda f: f.iterate(1, gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64), lambda i, buf, r: i)
    pipe.close()
    paths = []
    for i, d in enumerate(((4, 4, 4, 4), (4, 4, 4, 6))):
        p = tmp_path / ("cfg%d.npy" % i)
        np.save(p, gi.smooth_random_gauge(d, 0.4, 50 + i))
        paths.append(str(p))
    with pytest.raises(SystemExit, match="cfg1.npy.*differs"):
        fix.main(paths + ["--out-dir", str(tmp_path / "fixed"), "--target", "1e-10", "--lanes", "2", "--device", str(cuda_device)])


@pytest.mark.parametrize("gauge,algo,precision,recon", [("landau", "overrelax", "f64", 18), ("landau", "overrelax", "mixed-exact", 12),
                                                        ("coulomb", "stochastic", "f64", 18), ("landau", "overrelax", "mixed", 18)])
def test_command_line_fixes_an_ensemble_of_files(cuda_device, tmp_path, gauge, algo, precision, recon):
    """python -m paper_1305_3440_b200.fix: three configurations from .npy files through the pipeline; every result is
    gauge fixed as judged by the ORACLE (theta, Coulomb: every theta_t), has the input's plaquette and lies in SU(3)."""
    from paper_1305_3440_b200 import fix
    dims = (6, 4, 4, 6)
    paths = []
    for i in range(3):
        U = gi.smooth_random_gauge(dims, 0.4, 40 + i)
        p = tmp_path / ("cfg%d.npy" % i)
        np.save(p, U)
        paths.append(str(p))
    out_dir = tmp_path / "fixed"
    rc = fix.main(paths + ["--out-dir", str(out_dir), "--gauge", gauge, "--algo", algo, "--precision", precision, "--recon", str(recon),
                           "--target", "1e-12", "--check-every", "5", "--seed", "7", "--lanes", "2", "--device", str(cuda_device)])
    assert rc == 0
    og = oracle.COULOMB if gauge == "coulomb" else oracle.LANDAU
    for p in paths:
        U = np.load(p)
        W = np.ascontiguousarray(np.load(out_dir / p.split("/")[-1]))
        assert W.shape == U.shape and W.dtype == np.complex128
        assert np.max(oracle.theta(W, dims, og)) < 1e-12
        assert abs(oracle.plaquette(W, dims) - oracle.plaquette(U, dims)) < (1e-6 if precision == "mixed" else 1e-12)
        du, dd = oracle.unitarity_defect(W, dims)
        assert du < 1e-12 and dd < 1e-12
        assert np.min(oracle.functional(W, dims, og)) > np.min(oracle.functional(np.ascontiguousarray(U), dims, og))


def test_host_pipeline_streams_an_ensemble_through_one_buffer_per_lane(cuda_device):
    """process_stream: nine items through two lanes with one pinned buffer each; fill / drain run per item in order on
    their lane; results bitwise those of process() on the same inputs."""
    from paper_1305_3440_b200.pipeline import HostPipeline
    dims = (4, 4, 6, 4)
    inputs = [torch.from_numpy(gi.smooth_random_gauge(dims, 0.4, 300 + i)) for i in range(9)]

    def work(f):
        f.iterate(7, gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64)
        return f.measure(gf.GF_F64)

    pipe = HostPipeline(dims, precisions=("f64",), lanes=2, device=cuda_device)
    want_bufs = [h.clone().pin_memory() for h in inputs]
    want = pipe.process(want_bufs, work, gf.GF_F64)
    seen = []
    got = pipe.process_stream(9, lambda i, buf: buf.copy_(inputs[i]), work,
                              lambda i, buf, r: (seen.append(i), buf.clone(), r)[1:], gf.GF_F64)
    pipe.close()
    assert sorted(seen) == list(range(9))
    for i in range(9):
        assert torch.equal(got[i][0], want_bufs[i]) and got[i][1] == want[i]
    Uo = np.ascontiguousarray(inputs[4].numpy())
    for _ in range(7):
        for parity in (0, 1):
            oracle.sweep(Uo, dims, parity, algo=oracle.OVERRELAX, omega=1.7)
    assert np.abs(got[4][0].numpy() - Uo).max() < 1e-12
