"""Slab decomposition along t over peer memory (include/gf.h: gf_set_slab).

Host-side wiring only: which field is whose neighbour, in which order the slabs issue their
operations, and the one scalar sum of theta / F over the slabs.  Every sweep and reduction runs in
the library's kernels; the slabs share the boundary temporal links in place through device
pointers (no halo buffers, no collective on the data path).

* ``SlabSet``: all slabs driven by ONE process -- several slabs on one GPU (how the tests check the
  scheme on this pool's single GPU).  With several devices each context runs under its own device
  (the library switches devices per call) and peer access to the two neighbours' devices is enabled
  with ``gf_enable_peer``; that multi-device path is UNMEASURED ON HARDWARE (this pool has one GPU).
* ``SlabRank``: one slab per process under ``torch.distributed`` (one rank per GPU); the neighbours'
  fields and flags are mapped with CUDA IPC (torch's shared CUDA storages) and theta is summed
  with one scalar all-reduce.  Needs >= 2 GPUs: UNMEASURED ON HARDWARE on this pool.
"""
import torch

from . import binding as B
from .field import GaugeField


def local_dims(global_dims, nslabs):
    nt = int(global_dims[0])
    if nt % nslabs or (nt // nslabs) % 2:
        raise ValueError("N_t = %d must split into %d slabs of even length" % (nt, nslabs))
    return (nt // nslabs,) + tuple(int(d) for d in global_dims[1:])


def neighbours(rank, nslabs):
    """(rank below, rank above) on the periodic ring of slabs."""
    return (rank - 1) % nslabs, (rank + 1) % nslabs


def _ptr(field, prec):
    buf = field._bufs.get(prec)
    return buf.data_ptr() if buf is not None else 0


class SlabSet:
    """nslabs slabs of one lattice, all driven by this process (slab r on devices[r % len(devices)])."""

    def __init__(self, global_dims, nslabs, gauge=B.GF_LANDAU, recon=B.GF_RECON18, precisions=("f64",), seed=0,
                 devices=("cuda:0",)):
        self.global_dims = tuple(int(d) for d in global_dims)
        self.nslabs, self.gauge = nslabs, gauge
        self.dims = local_dims(global_dims, nslabs)
        self.fields, self.flags, self.streams = [], [], []
        for r in range(nslabs):
            dev = torch.device(devices[r % len(devices)])
            st = torch.cuda.Stream(device=dev)
            with torch.cuda.device(dev), torch.cuda.stream(st):
                self.fields.append(GaugeField(self.dims, gauge=gauge, recon=recon, precisions=precisions, seed=seed, device=dev))
            self.streams.append(st)
            self.flags.append(torch.zeros(4, dtype=torch.int32, device=dev))
        for dev in {f.device for f in self.fields}:
            torch.cuda.synchronize(dev)
        for r, f in enumerate(self.fields):
            lo, hi = neighbours(r, nslabs)
            for other in (self.fields[lo], self.fields[hi]):
                if other.device != f.device:        # this slab's kernels dereference pointers into the neighbour's field
                    B.gf_enable_peer(f.ctx, other.device.index)
            B.gf_set_slab(f.ctx, r, nslabs, _ptr(self.fields[lo], B.GF_F64), _ptr(self.fields[lo], B.GF_F32),
                          _ptr(self.fields[hi], B.GF_F64), _ptr(self.fields[hi], B.GF_F32),
                          self.flags[r].data_ptr(), self.flags[lo].data_ptr(), self.flags[hi].data_ptr())

    def close(self):
        for f in self.fields:
            f.close()

    def _sync(self):
        for dev in {f.device for f in self.fields}:
            torch.cuda.synchronize(dev)

    # every method below issues the same operation on every slab, in slab order
    def pack(self, canonical, precision):
        nt = self.dims[0]
        parts = [canonical[r * nt:(r + 1) * nt].to(f.device).contiguous() for r, f in enumerate(self.fields)]
        self._sync()                        # the slices were made on torch's stream, the slabs run on their own
        for f, part in zip(self.fields, parts):
            f.pack(part, precision)
        self._sync()

    def unpack(self, precision, dtype=torch.complex128):
        self._sync()
        parts = [f.unpack(precision, dtype) for f in self.fields]
        self._sync()
        return torch.cat([p.to(parts[0].device) for p in parts], dim=0)

    def sweep(self, parity, algo, omega, p, precision):
        for f in self.fields:
            f.sweep(parity, algo, omega, p, precision)

    def iterate(self, n, algo, omega, p, precision):
        for _ in range(n):
            self.sweep(0, algo, omega, p, precision)
            self.sweep(1, algo, omega, p, precision)

    def measure(self, precision):
        """Landau: (F, theta) of the whole lattice; Coulomb: per-slice lists over all N_t slices."""
        parts = [f.measure(precision) for f in self.fields]
        if self.gauge == B.GF_COULOMB:
            return sum((p[0] for p in parts), []), sum((p[1] for p in parts), [])
        return [sum(p[0][0] for p in parts)], [sum(p[1][0] for p in parts)]

    def plaquette(self, precision):
        return sum(f.plaquette(precision) for f in self.fields)

    def unitarity(self, precision):
        vals = [f.unitarity(precision) for f in self.fields]
        return max(v[0] for v in vals), max(v[1] for v in vals)

    def fix_until(self, algo, omega, p, precision, theta_target, max_iter, check_every=1):
        """The fix loop of gf_fix_until with theta added up over the slabs."""
        it, theta = 0, float("inf")
        while it < max_iter:
            n = min(check_every - it % check_every, max_iter - it)
            self.iterate(n, algo, omega, p, precision)
            it += n
            theta = max(self.measure(precision)[1])
            if theta < theta_target:
                return B.GF_OK, it, theta
        return B.GF_NOT_CONVERGED, it, theta


class SlabRank:
    """One slab per process (rank r of torch.distributed owns slab r, one GPU each)."""

    def __init__(self, global_dims, gauge=B.GF_LANDAU, recon=B.GF_RECON18, precisions=("f64",), seed=0, device=None,
                 group=None, _field=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.nslabs = dist.get_rank(group), dist.get_world_size(group)
        self.gauge = gauge
        self.dims = local_dims(global_dims, self.nslabs)
        if _field is not None:
            # host-logic tests (gloo, no GPU): a stand-in with iterate() / measure(); nothing is wired
            self.field, self.device = _field, torch.device("cpu")
            return
        self.device = torch.device(device if device is not None else "cuda:%d" % torch.cuda.current_device())
        self.field = GaugeField(self.dims, gauge=gauge, recon=recon, precisions=precisions, seed=seed, device=self.device)
        self.flag = torch.zeros(4, dtype=torch.int32, device=self.device)
        # CUDA IPC: publish this slab's buffers, map the two neighbours'
        mine = {"flag": _share(self.flag)}
        for prec, buf in self.field._bufs.items():
            mine[prec] = _share(buf)
        everyone = [None] * self.nslabs
        dist.all_gather_object(everyone, mine, group=group)
        lo, hi = neighbours(self.rank, self.nslabs)
        self._mapped = {}                                   # keeps the mappings alive
        def peer(r, key):
            if r == self.rank:
                return self.flag if key == "flag" else self.field._bufs.get(key)
            if key not in everyone[r]:
                return None
            return self._mapped.setdefault((r, key), _open(everyone[r][key], self.device))
        ptr = lambda t: t.data_ptr() if t is not None else 0
        B.gf_set_slab(self.field.ctx, self.rank, self.nslabs,
                      ptr(peer(lo, B.GF_F64)), ptr(peer(lo, B.GF_F32)), ptr(peer(hi, B.GF_F64)), ptr(peer(hi, B.GF_F32)),
                      self.flag.data_ptr(), ptr(peer(lo, "flag")), ptr(peer(hi, "flag")))
        dist.barrier(group=group)

    def close(self):
        self.field.close()

    def pack(self, local_canonical, precision):
        self.field.pack(local_canonical, precision)

    def unpack(self, precision, dtype=torch.complex128):
        return self.field.unpack(precision, dtype)

    def iterate(self, n, algo, omega, p, precision):
        self.field.iterate(n, algo, omega, p, precision)

    def measure(self, precision):
        F, th = self.field.measure(precision)
        if self.gauge == B.GF_COULOMB:
            return F, th                                    # this slab's time slices
        t = torch.tensor([F[0], th[0]], dtype=torch.float64, device=self.device)
        self.dist.all_reduce(t, group=self.group)           # one scalar sum: not on the data path
        return [float(t[0])], [float(t[1])]

    def fix_until(self, algo, omega, p, precision, theta_target, max_iter, check_every=1):
        it, theta = 0, float("inf")
        while it < max_iter:
            n = min(check_every - it % check_every, max_iter - it)
            self.iterate(n, algo, omega, p, precision)
            it += n
            theta = max(self.measure(precision)[1])
            if self.gauge == B.GF_COULOMB:
                t = torch.tensor([theta], dtype=torch.float64, device=self.device)
                self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX, group=self.group)
                theta = float(t[0])
            if theta < theta_target:
                return B.GF_OK, it, theta
        return B.GF_NOT_CONVERGED, it, theta


def _share(tensor):
    """CUDA IPC description of a device tensor's storage (picklable), plus its byte offset and size."""
    st = tensor.untyped_storage()
    return {"ipc": st._share_cuda_(), "offset": tensor.storage_offset() * tensor.element_size(),
            "nbytes": tensor.numel() * tensor.element_size()}


def _open(desc, device):
    with torch.cuda.device(device):
        st = torch.UntypedStorage._new_shared_cuda(*desc["ipc"])
    return torch.empty(0, dtype=torch.uint8, device=device).set_(st, desc["offset"], (desc["nbytes"],))
