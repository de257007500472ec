#!/usr/bin/env python
"""bench.py -- overrelaxation site-updates/s at 32^4 on B200 (BASELINE.json metric, configs[2]).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--variant f64-18]

One STEP = the whole hot path over one 32^4 lattice: ITERS overrelaxation iterations (omega = 1.7;
each = half-sweep of parity 0 then parity 1) with an F/theta reduction every
CHECK iterations (rows a7-a9), driven through the C ABI (gf_sweep / gf_measure).  ``value`` is
site-updates/s with the field resident in HBM; ``e2e`` adds, every step, the host->device copy of
the canonical field from pinned memory (gf_load_host) and the device->host copy of the fixed field
(gf_store_host).  The field (604 MB in fp64) is larger than the 126 MB L2, so no flush is needed.
N > 1: one independent lattice per GPU (replicas only, no data-path collective), weak scaling.

--impl reference times the CPU oracle (oracle/, fp64, OpenMP over all host cores) on the same
workload, one iteration per step; rank 0 only.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

DIMS = (32, 32, 32, 32)
V = DIMS[0] * DIMS[1] * DIMS[2] * DIMS[3]
OMEGA = 1.7
EPS = 0.6
SEED = 1
FLOP_PER_SITE_UPDATE = 2136          # nominal count, SURVEY.md 8(d) / DESIGN.md
METRIC = "overrelaxation site-updates/s at 32^4"
VARIANTS = {            # name: (precision key, recon, bytes per real)
    "f64-18": ("f64", 18, 8), "f64-12": ("f64", 12, 8),
    "f32-18": ("f32", 18, 4), "f32-12": ("f32", 12, 4),
    # fp32 storage with the opt-in all-fp32 solver (gf_set_solver_precision(GF_F32)): faster, but one iteration at 32^4
    # ends 1.08e-5 from the oracle, above north_star's 1e-5; the plain f32-* rows are the library default (K(x) and the
    # SU(2) solves in fp64 registers), which meets it
    "f32-18/solver-f32": ("f32", 18, 4), "f32-12/solver-f32": ("f32", 12, 4),
}


def solver_of(name):
    """Arithmetic of K(x) and the SU(2) solves for a variant: the storage precision for fp64, fp64 registers for fp32
    storage by default, fp32 for the */solver-f32 rows."""
    return "f32" if name.endswith("/solver-f32") else "f64"


TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r3_traffic.json")


def ncu_traffic(variant):
    """dram__bytes_read.sum + dram__bytes_write.sum per sweep launch at 32^4 from the committed `ncu --set full`
    summary (averages of the ncu metrics over the captured sweep launches; commands in profiles/r3_sweep_variants_ncu.md).
    Valid only for the kernel sources it was captured at: returns (None, why, None) when they have changed since.
    Third value: the same sum from the single-pass capture of consecutive launches without ncu's L2 flush, if on record."""
    try:
        from paper_1305_3440_b200.build import source_hash
        doc = json.load(open(TRAFFIC_FILE))
        if doc.get("source_hash") != source_hash():
            return None, "profiles/r3_traffic.json was captured at sources %s, the library is at %s" % (doc.get("source_hash"), source_hash()), None
        v = doc["variants"][variant]
        warm = v.get("in_run", {}).get("traffic_bytes")
        return float(v["traffic_bytes"]), "profiles/r3_traffic.json (ncu --set full, sources %s)" % doc["source_hash"], warm
    except Exception as e:                                      # missing file or variant: no claim
        return None, "no ncu capture on record (%s)" % type(e).__name__, None


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.first = index, [], None, 0

    def mark(self):
        """The timed region starts here: only rows sampled from now on are reported (nvidia-smi is started
        earlier, during the warm-up, because it takes a few hundred ms to deliver its first row)."""
        self.first = len(self.rows)

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        rows = self.rows[self.first:] or self.rows[-1:]
        sm = [float(r[0]) for r in rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 6 and r[2 + i] == "Active" for r in rows)]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def run_ours(args):
    import torch

    import gf_inputs as gi
    import paper_1305_3440_b200 as gf
    from paper_1305_3440_b200.replicas import Replicas

    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    rep = Replicas(backend="nccl", device=dev)      # barrier + one scalar all-reduce; no data-path collective
    rank, world = rep.rank, rep.world
    barrier, max_over_ranks = rep.barrier, rep.max_over_ranks
    peak, peak_src = measured_peaks()

    # same recipe on every rank, rank-dependent seed: one independent configuration per GPU
    U64 = gi.torch_smooth_random_gauge(DIMS, EPS, rep.config_seed(SEED), device=dev)

    def bench_variant(name, steps, warmup, with_e2e):
        pkey, recon, B = VARIANTS[name]
        prec = gf.GF_F64 if pkey == "f64" else gf.GF_F32
        cdtype = torch.complex128 if pkey == "f64" else torch.complex64
        fld = gf.GaugeField(DIMS, recon=recon, precisions=(pkey,), device=dev, staging=with_e2e)
        if name.endswith("/solver-f32"):
            fld.set_solver_precision(gf.GF_F32)
        Uc = U64.to(cdtype).contiguous()
        fld.pack(Uc, prec)
        n_blocks = args.iters // args.check
        sweep_ms = []

        def step(record):
            # the F/theta reductions are enqueued between the sweeps (gf_measure_async: results land in pinned
            # host memory) and read on the host at the end of the step: no host round trip inside the step
            for k in range(n_blocks):
                if record:
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                fld.iterate(args.check, gf.GF_OVERRELAX, OMEGA, 0.0, prec)
                if record:
                    b.record()
                    sweep_ms.append((a, b))
                fld.measure_async(prec, k % 16)
                if k % 16 == 15 or k == n_blocks - 1:
                    history = [fld.measure_collect(j % 16) for j in range(k - k % 16, k + 1)]
            return history

        sampler = ClockSampler(local_rank)
        sampler.start()
        for _ in range(warmup):
            step(False)
        launches0 = gf.gf_launch_count(fld.ctx)
        barrier()
        sampler.mark()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            step(True)
        e1.record()
        barrier()
        clocks = sampler.stop()
        ms_total = max_over_ranks(e0.elapsed_time(e1))
        launches = gf.gf_launch_count(fld.ctx) - launches0
        F, th = fld.measure(prec)
        kern_ms = sum(a.elapsed_time(b) for a, b in sweep_ms) / (len(sweep_ms) * 2 * args.check)
        bytes_per_launch = (V // 2) * 16 * recon * B
        achieved = bytes_per_launch / (kern_ms * 1e-3) / 1e9
        traffic, traffic_src, traffic_warm = ncu_traffic(name)
        solver = solver_of(name)
        out = {
            "value": world * V * args.iters * steps / (ms_total * 1e-3),
            "ms_per_step": ms_total / steps,
            "gpu_launches": int(launches),
            "clocks": clocks,
            # achieved / frac: ALGORITHMIC bytes (16 * recon * sizeof(real) per site-update, every link read once and
            # written once) over the event-timed launch.  dram_*: the same launch time against the bytes ncu saw
            # cross the DRAM interface (stores still dirty in the L2 when the launch ends do not): the HBM-level figure.
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "traffic_source": traffic_src,
                         "dram_achieved": (traffic / (kern_ms * 1e-3) / 1e9) if traffic else None,
                         "dram_frac": (traffic / (kern_ms * 1e-3) / 1e9 / peak) if traffic else None,
                         # ncu flushes the L2 before a profiled launch; traffic_in_run is a single-pass capture of
                         # consecutive launches without the flush: what crosses the DRAM interface inside a step
                         "traffic_in_run": traffic_warm,
                         "dram_frac_in_run": (traffic_warm / (kern_ms * 1e-3) / 1e9 / peak) if traffic_warm else None,
                         # What bounds a streaming kernel on this part is the throughput of the L2 slices: every algorithmic
                         # byte crosses them once between SM and L2, every DRAM byte once more (fill or write-back).  The
                         # copy behind `peak` pushes 2 x peak through them.
                         "l2_slice_GBs": ((bytes_per_launch + traffic_warm) / (kern_ms * 1e-3) / 1e9) if traffic_warm else None,
                         "l2_slice_frac_of_copy": ((bytes_per_launch + traffic_warm) / (kern_ms * 1e-3) / 1e9 / (2 * peak)) if traffic_warm else None,
                         "kernel": "gf::sweep_kernel<storage %s, solver %s, recon%d>" % (pkey, solver, recon),
                         "bytes_per_launch": bytes_per_launch, "avg_launch_ms": kern_ms, "peak_source": peak_src,
                         "frac_of_8TBs_nominal": achieved / 8000.0},
            "final_F": F[0], "final_theta": th[0],
        }
        if with_e2e:
            # End to end through the public API with HOST buffers (paper_1305_3440_b200.pipeline.HostPipeline): a few
            # lattices are in flight, each with its own context, CUDA stream, staging buffer and host thread (the library
            # calls release the GIL): while one lattice sweeps, another's fixed field goes device->host and its next
            # input host->device, so the PCIe transfers overlap the kernels; the sweep phases take turns on the GPU.
            # Every step still copies its whole input from pinned host memory and its whole result back.
            from paper_1305_3440_b200.pipeline import HostPipeline
            pipe = HostPipeline(DIMS, recon=recon, precisions=(pkey,), lanes=args.e2e_lanes, device=dev,
                                gate=bool(args.e2e_gate), first_field=fld)
            bufs = [torch.empty(fld.shape, dtype=cdtype).pin_memory() for _ in pipe.fields]
            sys.setswitchinterval(1e-4)                 # the worker threads hand the GIL over quickly

            def enqueue(f):                             # one step's sweeps and reductions; nothing here waits for the GPU
                for k in range(n_blocks):
                    f.iterate(args.check, gf.GF_OVERRELAX, OMEGA, 0.0, prec)
                    f.measure_async(prec, k % 16)
                    if k % 16 == 15 and k != n_blocks - 1:
                        [f.measure_collect(j) for j in range(16)]

            def collect(f):
                return [f.measure_collect(j % 16) for j in range(n_blocks - 1 - (n_blocks - 1) % 16, n_blocks)]

            def run_pipeline(n_steps, lanes=None):
                for h in bufs:
                    h.copy_(Uc)
                n = len(bufs) if lanes is None else lanes
                barrier()
                t0 = time.perf_counter()
                pipe.process([bufs[i % n] for i in range(n_steps)], enqueue, prec, collect=collect, lanes=lanes)
                return max_over_ranks(time.perf_counter() - t0)

            run_pipeline(len(bufs) * max(1, warmup // 2))
            dt = run_pipeline(steps)
            steady = pipe.steady_seconds_per_item()
            steady = max_over_ranks(steady) if steady else None
            # the same step with ONE lattice in flight: nothing overlaps the copies -- the latency a single caller sees
            run_pipeline(1, 1)
            n_single = max(2, steps // 3)
            dt_single = run_pipeline(n_single, 1)
            nbytes = bufs[0].numel() * bufs[0].element_size()
            out["e2e"] = {"value": world * V * args.iters * steps / dt, "unit": "site-updates/s",
                          "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes + 16 * n_blocks,
                          "ms_per_step": 1e3 * dt / steps,
                          "steady_ms_per_step": 1e3 * steady if steady else None,
                          "single_lattice_ms_per_step": 1e3 * dt_single / n_single,
                          "single_lattice_value": world * V * args.iters * n_single / dt_single,
                          "pipeline": "%d lattices in flight (one context, stream, pinned buffer and host thread each): copies "
                                      "overlap sweeps%s; value and ms_per_step are wall clock over all K steps including the "
                                      "pipeline's fill and drain, steady_ms_per_step is the time per step between the first and "
                                      "the last completed step" % (len(bufs), ", sweep phases take turns" if args.e2e_gate else "")}
            pipe.close()
            del pipe, bufs
        fld.close()
        del fld, Uc
        torch.cuda.empty_cache()
        return out

    U64_host = U64.cpu().numpy() if (rank == 0 and world == 1 and not args.no_cpu_baseline) else None
    main = bench_variant(args.variant, args.steps, args.warmup, True)
    variants = {}
    if not args.no_variants:
        for name in VARIANTS:
            if name == args.variant:
                continue
            # the same steps, warm-up, timing and clock sampling as the headline variant (no end-to-end leg)
            r = bench_variant(name, args.steps, args.warmup, False)
            variants[name] = {"site_updates_per_s": r["value"], "gflops_nominal": r["value"] * FLOP_PER_SITE_UPDATE / 1e9,
                              "storage": name.split("/")[0], "solver": solver_of(name),
                              "meets_north_star_link_tolerance_at_32^4": not name.endswith("/solver-f32"),
                              "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["ms_per_step"],
                              "gpu_launches": r["gpu_launches"], "clocks": r["clocks"], "roofline": r["roofline"],
                              "final_F": r["final_F"], "final_theta": r["final_theta"]}

    # Time to solution (BASELINE.json configs[2]: "fp32, mixed and fp64"): gf_fix_until to theta < 1e-12 on the
    # same 32^4 input, theta every 10 iterations.  Context for the SP/MP/DP reading of the metric, not the headline.
    fixes = {}
    if not args.no_fix:
        # *_stall: hand-off when fp32 stops lowering theta (gf_set_mixed_stall(1.0), hand-off theta out of reach)
        runs = [("f64", gf.GF_F64, None, 18, 0.0), ("mixed_handoff_1e-6", gf.GF_MIXED, 1e-6, 18, 0.0),
                ("mixed_exact_handoff_1e-10", gf.GF_MIXED_EXACT, 1e-10, 18, 0.0), ("mixed_exact_stall", gf.GF_MIXED_EXACT, 1e-15, 18, 1.0),
                ("f64_recon12", gf.GF_F64, None, 12, 0.0), ("mixed_exact_handoff_1e-10_recon12", gf.GF_MIXED_EXACT, 1e-10, 12, 0.0),
                ("mixed_exact_stall_recon12", gf.GF_MIXED_EXACT, 1e-15, 12, 1.0)]
        for name, mode, handoff, recon, stall in runs:
            fld = gf.GaugeField(DIMS, recon=recon, precisions=("f64",) if mode == gf.GF_F64 else ("f64", "f32"), device=dev)
            fld.pack(U64, gf.GF_F64)
            if mode == gf.GF_MIXED:
                fld.pack(U64.to(torch.complex64), gf.GF_F32)
            if mode == gf.GF_MIXED_EXACT:
                fld.attach_transform(("f64", "f32"))
            if handoff:
                fld.set_mixed_handoff(handoff)
            fld.set_mixed_stall(stall)
            P0 = fld.plaquette(gf.GF_F64)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            rc, it, th = fld.fix_until(gf.GF_OVERRELAX, OMEGA, 0.0, mode, 1e-12, 50000, 10)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            fixes[name] = {"converged": rc == gf.GF_OK, "iterations": it, "theta": th, "seconds": ms * 1e-3,
                           "site_updates_per_s": V * it / (ms * 1e-3), "plaquette_drift": fld.plaquette(gf.GF_F64) - P0}
            if name == "mixed_handoff_1e-6":
                # MP of the metric (BASELINE.json configs[2], "fp32 sweeps to theta < 1e-6, then fp64"): how the iterations
                # split.  The fp32 phase IS gf_fix_until(GF_F32, 1e-6) on the same input (same kernels, deterministic), so
                # its length is measured by running exactly that, outside the timed run above.
                fld.pack(U64.to(torch.complex64), gf.GF_F32)
                a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a0.record()
                rc32, it32, th32 = fld.fix_until(gf.GF_OVERRELAX, OMEGA, 0.0, gf.GF_F32, 1e-6, 50000, 10)
                a1.record()
                torch.cuda.synchronize()
                ms32 = a0.elapsed_time(a1)
                fixes[name].update({"fp32_phase_iterations": it32, "fp64_phase_iterations": it - it32,
                                    "fp32_phase_seconds": ms32 * 1e-3, "fp32_phase_theta": th32,
                                    "fp32_phase_site_updates_per_s": V * it32 / (ms32 * 1e-3),
                                    "fp64_phase_site_updates_per_s": V * (it - it32) / max(1e-9, (ms - ms32) * 1e-3)})
            fld.close()
            del fld
            torch.cuda.empty_cache()

    others = None
    if args.all_configs and world == 1:
        others = other_configs(gf, gi, torch, dev)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(U64_host, budget_s=12.0)

    if rank == 0:
        pkey, recon, _ = VARIANTS[args.variant]
        line = {
            "metric": METRIC, "value": main["value"], "unit": "site-updates/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": main["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": pkey, "data": "synthetic",
            "config": workload_config(args, world),
            "gflops_nominal": main["value"] * FLOP_PER_SITE_UPDATE / 1e9,
            "gpu_launches": main["gpu_launches"], "clocks": main["clocks"], "e2e": main["e2e"],
            "roofline": main["roofline"], "cpu_baseline": cpu, "variants": variants, "fix_until_theta_1e-12": fixes,
            "other_configs": others,
            "final_F": main["final_F"], "final_theta": main["final_theta"],
        }
        print(json.dumps(line), flush=True)
    rep.close()


def other_configs(gf, gi, torch, dev):
    """BASELINE.json's other workloads at full size (context for BASELINE.md section 4; parity for them is in tests/):
    configs[1] 16^4, configs[3] 64^4 (omega 1.8, 200 iterations, F / theta every 10), configs[4] 32^3 x 64 Coulomb
    gauge with stochastic relaxation (iteration rate, and gf_fix_until to max theta_t < 1e-12 with the Coulomb
    options of DESIGN.md section 12), and the per-time-slice times Tab. 1 of the paper lists."""
    out = {}

    def timed(fn):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        r = fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b), r

    def fixed_iterations(fld, prec, n, omega, check):
        for k in range(n // check):
            fld.iterate(check, gf.GF_OVERRELAX, omega, 0.0, prec)
            fld.measure_async(prec, k % 16)
            if k % 16 == 15 or k == n // check - 1:
                last = [fld.measure_collect(j % 16) for j in range(k - k % 16, k + 1)][-1]
        return last

    for name, dims, eps, omega, n in (("configs[1] 16^4", (16, 16, 16, 16), 0.5, 1.7, 500),
                                      ("configs[3] 64^4", (64, 64, 64, 64), 0.6, 1.8, 200)):
        vol = dims[0] * dims[1] * dims[2] * dims[3]
        U = gi.torch_smooth_random_gauge(dims, eps, SEED, device=dev)
        for pkey, prec, cd in (("f32", gf.GF_F32, torch.complex64), ("f64", gf.GF_F64, torch.complex128)):
            Uc = U.to(cd).contiguous() if pkey == "f32" else U
            for recon in (18, 12):
                fld = gf.GaugeField(dims, recon=recon, precisions=(pkey,), device=dev)
                fld.pack(Uc, prec)
                fixed_iterations(fld, prec, 20, omega, 10)
                fld.pack(Uc, prec)
                ms, (F, th) = timed(lambda: fixed_iterations(fld, prec, n, omega, 10))
                B = 8 if pkey == "f64" else 4
                out["%s %s-%d" % (name, pkey, recon)] = {
                    "iterations": n, "theta_F_every": 10, "seconds": ms * 1e-3, "site_updates_per_s": vol * n / (ms * 1e-3),
                    "algorithmic_GBs": vol * n * 16 * recon * B / (ms * 1e-3) / 1e9, "final_F": F[0], "final_theta": th[0]}
                fld.close()
                del fld
            del Uc
        del U
        torch.cuda.empty_cache()

    dims = (64, 32, 32, 32)
    vol = 64 * 32 ** 3
    U = gi.torch_smooth_random_gauge(dims, EPS, SEED, device=dev)
    for recon in (18, 12):
        for defer, freeze in ((0, 0), (1, 0), (1, 1)):
            fld = gf.GaugeField(dims, gauge=gf.GF_COULOMB, recon=recon, precisions=("f64",), seed=2013, device=dev)
            fld.attach_transform(("f64",) if defer else ())
            fld.pack(U, gf.GF_F64)
            fld.set_coulomb_mode(defer, freeze)
            fld.iterate(5, gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64)
            ms_it, _ = timed(lambda: fld.iterate(50, gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64))
            fld.pack(U, gf.GF_F64)
            gf.gf_set_rng(fld.ctx, 2013, 0)
            ms, (rc, it, th) = timed(lambda: fld.fix_until(gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64, 1e-12, 100000, 20))
            out["configs[4] 32^3x64 Coulomb stochastic p=0.8 f64-%d defer_temporal=%d freeze_slices=%d" % (recon, defer, freeze)] = {
                "site_updates_per_s": vol * 50 / (ms_it * 1e-3), "ms_per_iteration": ms_it / 50,
                "fix_converged": rc == gf.GF_OK, "fix_iterations": it, "fix_max_theta_t": th, "fix_seconds": ms * 1e-3}
            fld.close()
            del fld
    del U
    torch.cuda.empty_cache()

    tab1 = {}
    for ns, nt in ((16, 64), (32, 32), (64, 8), (128, 4)):
        dims = (nt, ns, ns, ns)
        U = gi.torch_hot_links(dims, 3, device=dev)
        for pkey, prec, cd in (("f32", gf.GF_F32, torch.complex64), ("f64", gf.GF_F64, torch.complex128)):
            fld = gf.GaugeField(dims, precisions=(pkey,), device=dev)
            fld.pack(U.to(cd).contiguous(), prec)
            n = max(5, int(2e9 / (nt * ns ** 3) / 3))
            fld.iterate(3, gf.GF_OVERRELAX, OMEGA, 0.0, prec)
            ms, _ = timed(lambda: fld.iterate(n, gf.GF_OVERRELAX, OMEGA, 0.0, prec))
            tab1["Ns=%d Nt=%d %s-18" % (ns, nt, pkey)] = {"ms_per_time_slice_both_parities": ms / n / nt}
            fld.close()
            del fld
        del U
        torch.cuda.empty_cache()
    out["PAPER.md Tab. 1 'kernel' column re-measured"] = tab1

    # the per-GPU lattices of the paper's weak-scaling figure (Fig. 3): 64^3 x 32 and 48^4
    fig3 = {}
    for dims in ((32, 64, 64, 64), (48, 48, 48, 48)):
        vol = dims[0] * dims[1] * dims[2] * dims[3]
        U = gi.torch_smooth_random_gauge(dims, EPS, SEED, device=dev)
        for pkey, prec, cd, B in (("f32", gf.GF_F32, torch.complex64, 4), ("f64", gf.GF_F64, torch.complex128, 8)):
            for recon in (18, 12):
                fld = gf.GaugeField(dims, recon=recon, precisions=(pkey,), device=dev)
                fld.pack(U.to(cd).contiguous(), prec)
                n = max(20, int(4e9 / vol))
                fld.iterate(5, gf.GF_OVERRELAX, OMEGA, 0.0, prec)
                ms, _ = timed(lambda: fld.iterate(n, gf.GF_OVERRELAX, OMEGA, 0.0, prec))
                fig3["%dx%d^3 %s-%d" % (dims[0], dims[1], pkey, recon)] = {
                    "site_updates_per_s": vol * n / (ms * 1e-3), "gflops_nominal": vol * n * FLOP_PER_SITE_UPDATE / (ms * 1e-3) / 1e9,
                    "algorithmic_GBs": vol * n * 16 * recon * B / (ms * 1e-3) / 1e9}
                fld.close()
                del fld
        del U
        torch.cuda.empty_cache()
    out["PAPER.md Fig. 3 per-GPU lattices, overrelaxation sweeps only"] = fig3
    return out


def cpu_baseline(U, budget_s):
    """The oracle as it stands, all host cores, full iterations of the same 32^4 workload until
    `budget_s` seconds of wall time have passed (at least one iteration)."""
    import oracle
    cores = oracle.set_threads(0)
    n, t0 = 0, time.perf_counter()
    while True:
        oracle.sweep(U, DIMS, 0, oracle.LANDAU, oracle.OVERRELAX, OMEGA)
        oracle.sweep(U, DIMS, 1, oracle.LANDAU, oracle.OVERRELAX, OMEGA)
        n += 1
        dt = time.perf_counter() - t0
        if dt >= budget_s:
            break
    oracle.set_threads(1)
    return {"value": n * V / dt, "unit": "site-updates/s", "cores": cores, "kind": "oracle",
            "sample": "%d full overrelaxation iteration(s) of the same 32^4 field, fp64, %.1f s" % (n, dt)}


def workload_config(args, world):
    """The `config` object of the JSON line: the workload both arms (--impl ours / reference) measure."""
    pkey, recon, nbytes = VARIANTS[args.variant]
    return {"workload": "BASELINE.json configs[2]: SU(3) Landau 32^4, overrelaxation omega=1.7, %s links "
                        "stored as %d reals, eps=0.6 smooth field + Haar gauge transform" % (pkey, recon),
            "lattice": list(DIMS), "iterations_per_step": args.iters, "theta_F_every": args.check,
            "l2": "field (%d MB) larger than L2, no flush" % (V * 4 * recon * nbytes // 2**20),
            "parallelism": "replicas only (one lattice per GPU)" if world > 1 else "single GPU"}


def run_reference(args):
    """The reference arm of this tier = the CPU oracle, timed as it stands on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import gf_inputs as gi
    import oracle
    dims = DIMS
    t_gen = time.perf_counter()
    # a step is a bounded sample of the workload: ONE full iteration of the 32^4 lattice (about a
    # second on a few cores), where a step of the CUDA arm is `--iters` iterations
    U = gi.smooth_random_gauge(dims, EPS, SEED)
    t_gen = time.perf_counter() - t_gen
    cores = oracle.set_threads(0)

    def step():
        oracle.sweep(U, dims, 0, oracle.LANDAU, oracle.OVERRELAX, OMEGA)
        oracle.sweep(U, dims, 1, oracle.LANDAU, oracle.OVERRELAX, OMEGA)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    val = args.steps * V / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "site-updates/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        # the CUDA arm's config: the workload is the same, a step of this arm is a bounded sample of it (see `sample`)
        "config": workload_config(args, int(os.environ.get("WORLD_SIZE", "1"))),
        "cpu_baseline": {"value": val, "unit": "site-updates/s", "cores": cores, "kind": "oracle",
                         "sample": "each step = ONE of the %d overrelaxation iterations of a step of the workload, on the same 32^4 field, "
                                   "fp64 oracle (canonical 18-real layout), no F/theta reduction (input generated in %.0f s)" % (args.iters, t_gen)},
        "e2e": {"value": val, "unit": "site-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gflops_nominal": val * FLOP_PER_SITE_UPDATE / 1e9,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--variant", default="f64-18", choices=sorted(VARIANTS))
    ap.add_argument("--iters", type=int, default=100, help="iterations per step")
    ap.add_argument("--check", type=int, default=10, help="F/theta reduction every CHECK iterations")
    ap.add_argument("--e2e-lanes", type=int, default=4, help="lattices in flight in the end-to-end pipeline")
    ap.add_argument("--e2e-gate", type=int, default=1, help="1: the sweep phases of the lattices in flight take turns on the GPU")
    ap.add_argument("--no-variants", action="store_true")
    ap.add_argument("--no-fix", action="store_true", help="skip the time-to-solution runs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--all-configs", action="store_true",
                    help="also time BASELINE.json configs[1], [3], [4] and the Tab. 1 slice sizes (adds about two minutes)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
