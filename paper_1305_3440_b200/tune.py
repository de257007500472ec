"""Launch-configuration sweep for the half-sweep kernel on the visible GPU.

    python -m paper_1305_3440_b200.tune [--dims 32 32 32 32] [--variants f64-18 f64-12 f32-18 f32-12]
                                        [--algo overrelax|relax|stochastic] [--iters 50]

For every storage variant times `iters` overrelaxation iterations (CUDA events, after a warm-up) with
the library default and with every (lanes per site, block size) the C ABI accepts (gf_set_tuning),
and prints site-updates/s and the algorithmic bandwidth 16 * recon * sizeof(real) bytes per
site-update.  Inputs are the seeded synthetic field of the benchmarks (eps = 0.6 smooth field + Haar
gauge transform, generated on the device).  Marshalling only: all work is done by libgf_b200.so.
"""
import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

ALGOS = {"relax": 0, "overrelax": 1, "stochastic": 2}


def measured_hbm_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"])
    except Exception:
        return 6650.0                      # B200_PROFILING.md fallback


def main():
    import torch

    import gf_inputs as gi
    import paper_1305_3440_b200 as gf

    ap = argparse.ArgumentParser()
    ap.add_argument("--dims", type=int, nargs=4, default=[32, 32, 32, 32], metavar=("NT", "NX", "NY", "NZ"))
    ap.add_argument("--variants", nargs="+", default=["f64-18", "f64-12", "f32-18", "f32-12"])
    ap.add_argument("--algo", default="overrelax", choices=sorted(ALGOS))
    ap.add_argument("--iters", type=int, default=50)
    ap.add_argument("--solver", default="auto", choices=["auto", "f32", "f64"],
                    help="arithmetic of K(x) and the SU(2) solves with fp32 storage (gf_set_solver_precision)")
    ap.add_argument("--configs", nargs="*", default=None, metavar="L:B",
                    help="only these lanes:block pairs (default: the library default and all nine)")
    args = ap.parse_args()
    dev = torch.device("cuda:0")
    dims = tuple(args.dims)
    V = dims[0] * dims[1] * dims[2] * dims[3]
    peak = measured_hbm_gbs()
    print("# %s, %s, solver %s, %d iterations per row, percentages of %.1f GB/s; L0 b0 = library default" % (
        "x".join(map(str, dims)), args.algo, args.solver, args.iters, peak))
    U = gi.torch_smooth_random_gauge(dims, 0.6, 1, device=dev)
    for name in args.variants:
        pkey, recon = name.split("-")
        recon = int(recon)
        prec = gf.GF_F64 if pkey == "f64" else gf.GF_F32
        cdtype = torch.complex128 if pkey == "f64" else torch.complex64
        nbytes = 16 * recon * (8 if pkey == "f64" else 4)
        fld = gf.GaugeField(dims, recon=recon, precisions=(pkey,), device=dev)
        fld.pack(U.to(cdtype).contiguous(), prec)
        fld.set_solver_precision({"auto": gf.GF_SOLVER_AUTO, "f32": gf.GF_F32, "f64": gf.GF_F64}[args.solver])
        pairs = [(0, 0)] + [(l, b) for l in (1, 2, 4) for b in (64, 128, 256)]
        if args.configs:
            pairs = [tuple(int(x) for x in c.split(":")) for c in args.configs]
        for lanes, block in pairs:
            if True:
                fld.set_tuning(prec, lanes, block)
                fld.iterate(10, ALGOS[args.algo], 1.7, 0.8, prec)
                torch.cuda.synchronize()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                fld.iterate(args.iters, ALGOS[args.algo], 1.7, 0.8, prec)
                b.record()
                torch.cuda.synchronize()
                ms = a.elapsed_time(b) / args.iters
                su = V / (ms * 1e-3)
                print("%s L%d b%3d  %.4f ms/iter  %.3e su/s  alg %.0f GB/s  %.1f%%" % (
                    name, lanes, block, ms, su, su * nbytes / 1e9, 100 * su * nbytes / 1e9 / peak), flush=True)
        F, th = fld.measure(prec)
        print("   F=%.6f theta=%.3e" % (F[0], th[0]))
        fld.close()
        del fld
        torch.cuda.empty_cache()


if __name__ == "__main__":
    main()
