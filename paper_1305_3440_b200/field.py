"""GaugeField: owns the torch buffers a gf_ctx borrows and forwards to the C ABI.

No arithmetic here: allocation, pointer hand-over and dtype checks only.
"""
import torch

from . import binding as B


class GaugeField:
    """A lattice on one GPU.

    dims = (Nt, Nx, Ny, Nz); precisions: any of ("f32", "f64") to allocate storage for
    (GF_MIXED needs both).  Canonical tensors are complex, shape (Nt, Nz, Ny, Nx, 4, 3, 3).
    """

    def __init__(self, dims, gauge=B.GF_LANDAU, recon=B.GF_RECON18, precisions=("f64",), seed=0,
                 device="cuda:0", staging=False):
        self.dims = tuple(int(d) for d in dims)
        self.gauge, self.recon = gauge, recon
        self.device = torch.device(device)
        self.n_out = self.dims[0] if gauge == B.GF_COULOMB else 1
        self.shape = (self.dims[0], self.dims[3], self.dims[2], self.dims[1], 4, 3, 3)
        self._bufs = {}
        for name, prec in (("f32", B.GF_F32), ("f64", B.GF_F64)):
            if name in precisions:
                n = B.gf_storage_bytes(self.dims, prec, recon)
                if n == 0:
                    raise ValueError("invalid dims/recon %r %r" % (dims, recon))
                self._bufs[prec] = torch.empty(n, dtype=torch.uint8, device=self.device)
        self._ws = torch.empty(B.gf_workspace_bytes(self.dims), dtype=torch.uint8, device=self.device)
        self._staging = None
        if staging:
            self._staging = torch.empty(self.shape, dtype=torch.complex128, device=self.device)
        with torch.cuda.device(self.device):
            self.stream = torch.cuda.current_stream()
            self.ctx = B.gf_init_lattice(
                self.dims, gauge, recon,
                self._bufs[B.GF_F64].data_ptr() if B.GF_F64 in self._bufs else 0,
                self._bufs[B.GF_F32].data_ptr() if B.GF_F32 in self._bufs else 0,
                self._ws.data_ptr(), self.stream.cuda_stream, seed)

    def close(self):
        if getattr(self, "ctx", None):
            torch.cuda.synchronize(self.device)
            B.gf_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def storage(self, precision):
        """The uint8 tensor holding the internal link field of `precision` (what the context borrows): for calls that
        take the field itself rather than the context, such as binding.gf_measure_static."""
        return self._bufs[precision]

    # ---- layout conversion
    def _canon(self, t):
        if t.dtype not in (torch.complex128, torch.complex64) or tuple(t.shape) != self.shape \
                or not t.is_contiguous() or t.device != self.device:
            raise ValueError("canonical tensor must be contiguous complex %r on %s" % (self.shape, self.device))
        return t.data_ptr(), t.dtype == torch.complex128

    def pack(self, canonical, precision):
        ptr, is64 = self._canon(canonical)
        B.gf_pack(self.ctx, ptr, is64, precision)

    def unpack(self, precision, dtype=torch.complex128):
        out = torch.empty(self.shape, dtype=dtype, device=self.device)
        B.gf_unpack(self.ctx, out.data_ptr(), dtype == torch.complex128, precision)
        return out

    def load_host(self, host_canonical, precision):
        """host_canonical: CPU (ideally pinned) complex tensor; needs staging=True."""
        B.gf_load_host(self.ctx, host_canonical.data_ptr(), host_canonical.dtype == torch.complex128, precision,
                       self._staging.data_ptr())

    def store_host(self, host_canonical, precision):
        B.gf_store_host(self.ctx, host_canonical.data_ptr(), host_canonical.dtype == torch.complex128, precision,
                        self._staging.data_ptr())

    # ---- the method
    def sweep(self, parity, algo, omega, p, precision):
        B.gf_sweep(self.ctx, parity, algo, omega, p, precision)

    def iterate(self, n, algo, omega, p, precision):
        B.gf_iterate(self.ctx, n, algo, omega, p, precision)

    def functional(self, precision):
        return B.gf_functional(self.ctx, precision, self.n_out)

    def theta(self, precision):
        return B.gf_theta(self.ctx, precision, self.n_out)

    def measure(self, precision):
        return B.gf_measure(self.ctx, precision, self.n_out)

    def measure_async(self, precision, slot):
        B.gf_measure_async(self.ctx, precision, slot)

    def measure_collect(self, slot):
        return B.gf_measure_collect(self.ctx, slot, self.n_out)

    def fix_until(self, algo, omega, p, precision, theta_target, max_iter, check_every=1):
        return B.gf_fix_until(self.ctx, algo, omega, p, precision, theta_target, max_iter, check_every)

    def plaquette(self, precision):
        return B.gf_plaquette(self.ctx, precision)

    def unitarity(self, precision):
        return B.gf_unitarity(self.ctx, precision)

    # ---- the accumulated transformation G(x)
    def attach_transform(self, precisions=("f64",)):
        """Allocates G(x) for the given precisions, sets it to the identity and attaches it: sweeps of
        those precisions then record G(x) <- g(x) G(x).  attach_transform(()) detaches."""
        self._gbufs = {}
        for name, prec in (("f32", B.GF_F32), ("f64", B.GF_F64)):
            if name in precisions:
                n = B.gf_transform_bytes(self.dims, prec, self.recon)
                self._gbufs[prec] = torch.empty(n, dtype=torch.uint8, device=self.device)
        B.gf_set_transform(self.ctx,
                           self._gbufs[B.GF_F64].data_ptr() if B.GF_F64 in self._gbufs else 0,
                           self._gbufs[B.GF_F32].data_ptr() if B.GF_F32 in self._gbufs else 0)
        for prec in self._gbufs:
            B.gf_transform_identity(self.ctx, prec)

    def transform(self, precision, dtype=torch.complex128):
        """G(x) as a canonical tensor (Nt, Nz, Ny, Nx, 3, 3)."""
        out = torch.empty(self.shape[:4] + (3, 3), dtype=dtype, device=self.device)
        B.gf_transform_unpack(self.ctx, out.data_ptr(), dtype == torch.complex128, precision)
        return out

    def set_transform(self, canonical, precision):
        if canonical.dtype not in (torch.complex128, torch.complex64) or tuple(canonical.shape) != self.shape[:4] + (3, 3) \
                or not canonical.is_contiguous() or canonical.device != self.device:
            raise ValueError("transformation must be contiguous complex %r on %s" % (self.shape[:4] + (3, 3), self.device))
        B.gf_transform_pack(self.ctx, canonical.data_ptr(), canonical.dtype == torch.complex128, precision)

    def transform_identity(self, precision):
        B.gf_transform_identity(self.ctx, precision)

    def transform_cast(self, from_precision, to_precision):
        B.gf_transform_cast(self.ctx, from_precision, to_precision)

    def apply_transform(self, g_precision, src_precision, dst_precision):
        B.gf_apply_transform(self.ctx, g_precision, src_precision, dst_precision)

    # ---- Coulomb specialisation
    def set_coulomb_mode(self, defer_temporal=False, freeze_slices=False):
        B.gf_set_coulomb_mode(self.ctx, defer_temporal, freeze_slices)

    def coulomb_finish(self, precision):
        B.gf_coulomb_finish(self.ctx, precision)

    def set_slice_mask(self, active):
        B.gf_set_slice_mask(self.ctx, active)

    def cast(self, from_precision, to_precision):
        B.gf_cast(self.ctx, from_precision, to_precision)

    def set_tuning(self, precision, lanes, block):
        B.gf_set_tuning(self.ctx, precision, lanes, block)

    def set_solver_precision(self, solver_precision):
        B.gf_set_solver_precision(self.ctx, solver_precision)

    def set_mixed_handoff(self, theta_handoff):
        B.gf_set_mixed_handoff(self.ctx, theta_handoff)

    def set_traversal(self, zigzag):
        B.gf_set_traversal(self.ctx, zigzag)

    def set_fix_runahead(self, blocks):
        B.gf_set_fix_runahead(self.ctx, blocks)

    def set_reunitarize_every(self, iterations):
        B.gf_set_reunitarize_every(self.ctx, iterations)

    def set_mixed_stall(self, ratio):
        B.gf_set_mixed_stall(self.ctx, ratio)
