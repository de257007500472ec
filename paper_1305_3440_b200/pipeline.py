"""HostPipeline: an ensemble of configurations in HOST memory through one GPU.

The usual workload is an ensemble of independent configurations.  A lone lattice that
comes from host memory pays its two PCIe copies in full (32^4 fp64: 2 x 11 ms around 37 ms of sweeps);
with a few lattices in flight -- one context, CUDA stream, staging buffer and host thread each -- the copies,
pack and unpack of one lattice overlap the sweeps of another.  The sweep phases themselves take turns on the
GPU (an event chain through the streams, in the order the host threads arrive): two half-sweeps of different
lattices running side by side would halve each other's share of the SMs and evict the links the zigzag
traversal expects to find in the L2.

Plumbing only: threads, streams, events and the gf_load_host / gf_store_host calls.  What runs between load
and store is the caller's `work(field)` -- calls into the C ABI through GaugeField.
"""
import threading
import time

import torch

from . import binding as B
from .field import GaugeField


class HostPipeline:
    """`lanes` lattices of the same shape in flight on one device.

    process(hosts, work): every tensor of `hosts` (CPU, canonical layout, ideally pinned; complex128 or complex64)
    is loaded into a lane's field, `work(field)` runs, and the field is stored back into the same tensor.
    Host tensor i goes to lane i % lanes, in order, so a tensor may appear several times as long as all
    its appearances fall on one lane.
    """

    def __init__(self, dims, gauge=B.GF_LANDAU, recon=B.GF_RECON18, precisions=("f64",), lanes=3, device="cuda:0",
                 seed=0, gate=None, first_field=None):
        self.device = torch.device(device)
        # gate = None: the sweep phases take turns when a half-sweep fills the GPU by itself.  Lattices of a few
        # thousand sites per parity (less than one wave of blocks) are bound by the latency of one site update and
        # share the GPU instead: 8^4, eight lanes: 0.74 against 2.5 ms per configuration fixed to theta < 1e-12.
        sites_per_parity = 1
        for d in dims:
            sites_per_parity *= int(d)
        sites_per_parity //= 2
        self.gate = sites_per_parity > 4096 if gate is None else bool(gate)
        self.fields = [] if first_field is None else [first_field]
        self._borrowed = first_field is not None
        for _ in range(int(lanes) - len(self.fields)):
            with torch.cuda.stream(torch.cuda.Stream(device=self.device)):
                self.fields.append(GaugeField(dims, gauge=gauge, recon=recon, precisions=precisions, seed=seed,
                                              device=self.device, staging=True))
        self._lock = threading.Lock()
        self._last = None                   # event recorded after the latest sweep phase that was enqueued
        self.done_at = []                   # perf_counter() at which each item's result was on the host

    def _run_work(self, f, work):
        if not self.gate:
            return work(f)
        # The lock is held while the phase is enqueued (or, if `work` synchronises, while it runs): the next lattice's
        # stream waits for the event recorded behind this one's kernels.
        with self._lock:
            if self._last is not None:
                f.stream.wait_event(self._last)
            try:
                return work(f)
            finally:
                ev = torch.cuda.Event()
                ev.record(f.stream)
                self._last = ev

    def process(self, hosts, work, precision=B.GF_F64, collect=None, lanes=None):
        """Returns [collect(field) or work's return value] per host tensor, in input order.  `work(field)` runs in
        its lane's turn; `collect(field)`, if given, after the turn has been handed on (the place for calls that
        wait for results, e.g. gf_measure_collect) and before the field is stored."""
        fields = self.fields[:len(self.fields) if lanes is None else int(lanes)]
        hosts = list(hosts)
        results, errors = [None] * len(hosts), []
        self.done_at = []

        def lane(k):
            try:
                torch.cuda.set_device(self.device)
                f = fields[k]
                for i in range(k, len(hosts), len(fields)):
                    f.load_host(hosts[i], precision)
                    r = self._run_work(f, work)
                    if collect is not None:
                        r = collect(f)
                    f.store_host(hosts[i], precision)       # synchronises the lane's stream
                    results[i] = r
                    self.done_at.append(time.perf_counter())
            except BaseException as e:                      # re-raised in the caller's thread (SystemExit from a callback too:
                errors.append(e)                            # threading would swallow it and the item would just be missing)

        threads = [threading.Thread(target=lane, args=(k,)) for k in range(min(len(fields), len(hosts)))]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        torch.cuda.synchronize(self.device)
        if errors:
            raise errors[0]
        return results

    def process_stream(self, n_items, fill, work, drain, precision=B.GF_F64, dtype=torch.complex128):
        """An ensemble that does not fit host memory at once.  Every lane owns ONE pinned buffer of the canonical shape;
        for item i (lane i % lanes, in order) `fill(i, buffer)` writes the configuration into it (e.g. from a file),
        the buffer is loaded, `work(field)` runs in the lane's turn, the result is stored back into the buffer and
        `drain(i, buffer, result)` consumes it (e.g. writes a file) before the lane goes on.  fill and drain run in the
        lane's host thread: file I/O of one lane overlaps the copies and sweeps of the others.  Returns the list of
        whatever drain returned."""
        fields = self.fields
        bufs = [torch.empty(f.shape, dtype=dtype).pin_memory() for f in fields]
        out, errors = [None] * int(n_items), []
        self.done_at = []

        def lane(k):
            try:
                torch.cuda.set_device(self.device)
                f, buf = fields[k], bufs[k]
                for i in range(k, int(n_items), len(fields)):
                    fill(i, buf)
                    f.load_host(buf, precision)
                    r = self._run_work(f, work)
                    f.store_host(buf, precision)
                    out[i] = drain(i, buf, r)
                    self.done_at.append(time.perf_counter())
            except BaseException as e:
                errors.append(e)

        threads = [threading.Thread(target=lane, args=(k,)) for k in range(min(len(fields), int(n_items)))]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        torch.cuda.synchronize(self.device)
        if errors:
            raise errors[0]
        return out

    def steady_seconds_per_item(self):
        """Between the first and the last completed item of the latest process() the pipeline is full: the time per
        item without the one copy before the first sweep and the one after the last that nothing overlaps."""
        d = sorted(self.done_at)
        return (d[-1] - d[0]) / (len(d) - 1) if len(d) > 1 else None

    def close(self):
        for f in self.fields[1 if self._borrowed else 0:]:
            f.close()
        self.fields = []
