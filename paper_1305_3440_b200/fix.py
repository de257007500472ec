"""Command line: fix one configuration (or every file of an ensemble) to Landau or Coulomb gauge on the visible B200.

    python -m paper_1305_3440_b200.fix IN.npy [IN2.npy ...] --out-dir DIR [--gauge landau|coulomb]
           [--algo overrelax|relax|stochastic] [--omega 1.7] [--p 0.8] [--precision f64|f32|mixed|mixed-exact]
           [--recon 18|12] [--target 1e-12] [--max-iter 100000] [--check-every 10] [--seed 0] [--lanes 3]
           [--reunitarize-every 0] [--handoff THETA]

IN.npy holds the links in the canonical layout of include/gf.h: a complex128 array of shape (Nt, Nz, Ny, Nx, 4, 3, 3).
The fixed configuration is written to DIR/<name>.npy and one line per file reports iterations, theta, F and the drift of
the (gauge-invariant) plaquette.  Several files go through HostPipeline, one pinned buffer per lane: reading, copying and
writing one configuration overlap the sweeps of another, whatever the size of the ensemble.  Argument marshalling and file I/O only; every step of the method runs in libgf_b200.so (the
sweeps are iterated until the requested gauge precision theta has been reached).
"""
import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main(argv=None):
    import numpy as np
    import torch

    import paper_1305_3440_b200 as gf
    from paper_1305_3440_b200.pipeline import HostPipeline

    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("inputs", nargs="+")
    ap.add_argument("--out-dir", required=True)
    ap.add_argument("--gauge", default="landau", choices=["landau", "coulomb"])
    ap.add_argument("--algo", default="overrelax", choices=["overrelax", "relax", "stochastic"])
    ap.add_argument("--omega", type=float, default=1.7)
    ap.add_argument("--p", type=float, default=0.8)
    ap.add_argument("--precision", default="f64", choices=["f64", "f32", "mixed", "mixed-exact"])
    ap.add_argument("--recon", type=int, default=18, choices=[18, 12])
    ap.add_argument("--target", type=float, default=1e-12)
    ap.add_argument("--max-iter", type=int, default=100000)
    ap.add_argument("--check-every", type=int, default=10)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--handoff", type=float, default=None,
                    help="theta at which the fp32 phase of the mixed modes hands over (default: 1e-6 for mixed; for mixed-exact "
                         "out of reach, the fp32 phase then ends when it stops lowering theta)")
    ap.add_argument("--reunitarize-every", type=int, default=0,
                    help="re-project the swept field onto SU(3) every so many iterations (fp32 runs of thousands of iterations)")
    ap.add_argument("--lanes", type=int, default=3)
    ap.add_argument("--device", default="cuda:0")
    args = ap.parse_args(argv)

    gauge = gf.GF_COULOMB if args.gauge == "coulomb" else gf.GF_LANDAU
    algo = {"overrelax": gf.GF_OVERRELAX, "relax": gf.GF_RELAX, "stochastic": gf.GF_STOCHASTIC}[args.algo]
    mode = {"f64": gf.GF_F64, "f32": gf.GF_F32, "mixed": gf.GF_MIXED, "mixed-exact": gf.GF_MIXED_EXACT}[args.precision]
    omega = args.omega if algo == gf.GF_OVERRELAX else 1.0
    p = args.p if algo == gf.GF_STOCHASTIC else 0.0
    precisions = ("f64",) if mode == gf.GF_F64 else (("f32",) if mode == gf.GF_F32 else ("f64", "f32"))
    io_prec = gf.GF_F32 if mode == gf.GF_F32 else gf.GF_F64          # the field that holds the input and the result
    cdtype = torch.complex64 if mode == gf.GF_F32 else torch.complex128

    first = np.load(args.inputs[0], mmap_mode="r")
    if first.ndim != 7 or first.shape[4:] != (4, 3, 3):
        raise SystemExit("%s: expected shape (Nt, Nz, Ny, Nx, 4, 3, 3), got %r" % (args.inputs[0], first.shape))
    dims = (first.shape[0], first.shape[3], first.shape[2], first.shape[1])
    os.makedirs(args.out_dir, exist_ok=True)

    pipe = HostPipeline(dims, gauge=gauge, recon=args.recon, precisions=precisions, lanes=min(args.lanes, len(args.inputs)),
                        device=args.device, seed=args.seed)
    for f in pipe.fields:
        if mode == gf.GF_MIXED_EXACT:
            f.attach_transform(("f64", "f32"))
        f.set_reunitarize_every(args.reunitarize_every)
        if args.handoff is not None:
            f.set_mixed_handoff(args.handoff)
        elif mode == gf.GF_MIXED_EXACT:             # the result does not inherit fp32 rounding: stay in fp32 as long as it pays
            f.set_mixed_handoff(1e-15)
            f.set_mixed_stall(1.0)

    def work(f):
        P0 = f.plaquette(io_prec)
        if mode == gf.GF_MIXED:                     # gf_fix_until(GF_MIXED) starts from the fp32 field
            f.cast(gf.GF_F64, gf.GF_F32)
        gf.gf_set_rng(f.ctx, args.seed, 0)
        rc, it, th = f.fix_until(algo, omega, p, mode, args.target, args.max_iter, args.check_every)
        F, _ = f.measure(io_prec)
        return rc, it, th, float(np.mean(F)), f.plaquette(io_prec) - P0

    def fill(i, buf):                               # runs in the lane's thread: file I/O overlaps the other lanes' sweeps
        a = np.load(args.inputs[i])
        if tuple(a.shape) != tuple(first.shape):         # an ordinary exception: the pipeline hands it to the caller's thread
            raise ValueError("%s: shape %r differs from %r" % (args.inputs[i], a.shape, first.shape))
        buf.copy_(torch.from_numpy(np.ascontiguousarray(a)).to(cdtype))

    def drain(i, buf, result):
        out = os.path.join(args.out_dir, os.path.basename(args.inputs[i]))
        np.save(out, buf.numpy().astype(np.complex128))
        return out, result

    status = 0
    try:
        done = pipe.process_stream(len(args.inputs), fill, work, drain, io_prec, cdtype)
    except ValueError as e:                         # a bad input file: stop with its message (results already drained stay on disk)
        pipe.close()
        raise SystemExit(str(e))
    for path, (out, (rc, it, th, F, dP)) in zip(args.inputs, done):
        print("%s -> %s: %s after %d iterations, theta = %.3e, F = %.9f, plaquette drift %.1e" % (
            path, out, "converged" if rc == gf.GF_OK else "NOT converged", it, th, F, dP), flush=True)
        status |= 0 if rc == gf.GF_OK else 1
    pipe.close()
    return status


if __name__ == "__main__":
    sys.exit(main())
