"""`Lattice`: owns the device buffers (torch tensors) and a context of libu1u1.so; its methods are the
C-ABI calls of include/u1u1.h under the same names (init_fields, step, diagnostics, gauss_violation,
...).  Argument marshalling only -- all arithmetic happens in the CUDA kernels."""
from __future__ import annotations

import ctypes

import numpy as np

from . import binding as B


class Lattice:
    def __init__(self, N: int, device: str = "cuda:0", stream=None, aux: bool = False):
        """aux=True also allocates the second momentum buffer (u1u1_set_aux): step() then takes two steps per pass."""
        import torch
        if not torch.cuda.is_available():
            raise B.U1U1Error("CUDA device required: libu1u1 has no CPU fallback")
        self._torch = torch
        self.lib = B.load()
        self.N = int(N)
        self.device = torch.device(device)
        sb, cb = B.state_bytes(self.N), B.scratch_bytes(self.N)
        if sb == 0:
            raise B.U1U1Error(f"unsupported lattice size N={N}")
        with torch.cuda.device(self.device):
            self.state = torch.empty(sb, dtype=torch.uint8, device=self.device)
            self.scratch = torch.empty(cb, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._ctx = ctypes.c_void_p()
        rc = self.lib.u1u1_create(ctypes.byref(self._ctx), self.state.data_ptr(), sb,
                                  self.scratch.data_ptr(), cb, self.stream.cuda_stream)
        if rc:
            raise B.U1U1Error(f"u1u1_create: {self.lib.u1u1_last_error(None).decode()}")
        self.aux = None
        if aux:
            self.set_aux(True)

    def set_aux(self, on: bool):
        """Attach (allocate) or detach (free) the second momentum buffer."""
        if on and self.aux is None:
            ab = self.lib.u1u1_aux_bytes(self.N)
            with self._torch.cuda.device(self.device):
                buf = self._torch.empty(ab, dtype=self._torch.uint8, device=self.device)
            self._check(self.lib.u1u1_set_aux(self._ctx, buf.data_ptr(), ab), "set_aux")
            self.aux = buf
        elif not on and self.aux is not None:
            self._check(self.lib.u1u1_set_aux(self._ctx, None, 0), "set_aux")
            self.aux = None

    # -- helpers ---------------------------------------------------------------------------------
    def _check(self, rc, what):
        if rc:
            msg = self.lib.u1u1_last_error(self._ctx).decode()
            raise B.U1U1Error(f"{what}: {B.ERRORS.get(rc, rc)}: {msg}")

    def close(self):
        if self._ctx:
            self.lib.u1u1_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C ABI, same names ---------------------------------------------------------------------
    def set_tuning(self, flags: int):
        """Experimental switches (include/u1u1_tuning.h); 0 in production."""
        self._check(self.lib.u1u1_set_tuning(self._ctx, int(flags)), "set_tuning")

    def configure(self, dx: float, params: B.Params):
        self.set_tuning(getattr(params, "tuning", 0))
        self._check(self.lib.u1u1_configure(self._ctx, self.N, dx, ctypes.byref(params)), "configure")

    def init_fields(self, seed: int, dx: float, params: B.Params):
        self.set_tuning(getattr(params, "tuning", 0))
        self._check(self.lib.u1u1_init_fields(self._ctx, seed, self.N, dx, ctypes.byref(params)), "init_fields")

    def set_params(self, params: B.Params):
        self.set_tuning(getattr(params, "tuning", 0))
        self._check(self.lib.u1u1_set_params(self._ctx, ctypes.byref(params)), "set_params")

    def set_time(self, tau: float, era_m: float, s: float):
        self._check(self.lib.u1u1_set_time(self._ctx, tau, era_m, s), "set_time")

    def step(self, n: int, tau: float, era_m: float, s: float):
        self._check(self.lib.u1u1_step(self._ctx, n, tau, era_m, s), "step")

    def cool(self, n: int, dcool: float):
        self._check(self.lib.u1u1_cool(self._ctx, n, dcool), "cool")

    def diagnostics(self) -> dict:
        out = (ctypes.c_double * B.DIAG_LEN)()
        self._check(self.lib.u1u1_diagnostics(self._ctx, out), "diagnostics")
        return {k: out[i] for i, k in enumerate(B.DIAG_SLOTS)}

    def gauss_violation(self) -> np.ndarray:
        out = (ctypes.c_double * B.GAUSS_LEN)()
        self._check(self.lib.u1u1_gauss_violation(self._ctx, out), "gauss_violation")
        return np.array(out[:])

    def export_state(self):
        """Canonical float32 [20, N, N, N] torch tensor on the device."""
        t = self._torch.empty((20, self.N, self.N, self.N), dtype=self._torch.float32, device=self.device)
        self._check(self.lib.u1u1_export_state(self._ctx, t.data_ptr()), "export_state")
        return t

    def import_state(self, t):
        torch = self._torch
        t = t.to(device=self.device, dtype=torch.float32).contiguous()
        assert tuple(t.shape) == (20, self.N, self.N, self.N), t.shape
        self._check(self.lib.u1u1_import_state(self._ctx, t.data_ptr()), "import_state")
        self.stream.synchronize()   # `t` may be a temporary

    def import_state_tiled(self, t):
        """Periodic tiling of a smaller canonical state [20, n, n, n] (N a multiple of n)."""
        torch = self._torch
        t = t.to(device=self.device, dtype=torch.float32).contiguous()
        assert t.shape[0] == 20 and t.shape[1] == t.shape[2] == t.shape[3], t.shape
        self._check(self.lib.u1u1_import_state_tiled(self._ctx, t.data_ptr(), int(t.shape[1])), "import_state_tiled")
        self.stream.synchronize()

    def export_state_host(self, host_tensor):
        self._check(self.lib.u1u1_export_state_host(self._ctx, host_tensor.data_ptr()), "export_state_host")

    def import_state_host(self, host_tensor):
        self._check(self.lib.u1u1_import_state_host(self._ctx, host_tensor.data_ptr()), "import_state_host")

    def export_windings(self, sector: int):
        """(W int8 [3,N,N,N], near uint8 [3,N,N,N], cells uint8 [N,N,N]) after diagnostics()."""
        torch, N = self._torch, self.N
        W = torch.empty((3, N, N, N), dtype=torch.int8, device=self.device)
        near = torch.empty((3, N, N, N), dtype=torch.uint8, device=self.device)
        cells = torch.empty((N, N, N), dtype=torch.uint8, device=self.device)
        self._check(self.lib.u1u1_export_windings(self._ctx, sector, W.data_ptr(), near.data_ptr(),
                                                  cells.data_ptr()), "export_windings")
        self.stream.synchronize()
        return W, near, cells

    def pq_segments(self, min_cells: int = 1, tolerant: bool = False) -> dict:
        out = (ctypes.c_double * B.SEG_LEN)()
        self._check(self.lib.u1u1_pq_segments(self._ctx, min_cells, int(tolerant), out), "pq_segments")
        return {k: out[i] for i, k in enumerate(B.SEG_SLOTS)}

    def export_labels(self):
        t = self._torch.empty((self.N, self.N, self.N), dtype=self._torch.int32, device=self.device)
        self._check(self.lib.u1u1_export_labels(self._ctx, t.data_ptr()), "export_labels")
        self.stream.synchronize()
        return t

    def export_block(self, x0, y0, z0, bx, by, bz):
        t = self._torch.empty((20, bz, by, bx), dtype=self._torch.float32, device=self.device)
        self._check(self.lib.u1u1_export_block(self._ctx, x0, y0, z0, bx, by, bz, t.data_ptr()), "export_block")
        self.stream.synchronize()
        return t

    def launch_count(self) -> int:
        return int(self.lib.u1u1_launch_count(self._ctx))


class Slab:
    """One z slab of a lattice split over several GPUs (include/u1u1.h, "z slabs"): owns the slab's state buffer and a
    context; the methods are the slab calls of the C ABI.  Argument marshalling only."""

    def __init__(self, N: int, nz_own: int, z_first: int, device: str = "cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise B.U1U1Error("CUDA device required: libu1u1 has no CPU fallback")
        self._torch = torch
        self.lib = B.load()
        self.N, self.nz_own, self.z_first = int(N), int(nz_own), int(z_first)
        self.device = torch.device(device)
        sb = self.lib.u1u1_slab_state_bytes(self.N, self.nz_own)
        if sb == 0:
            raise B.U1U1Error(f"unsupported slab N={N}, nz_own={nz_own}")
        with torch.cuda.device(self.device):
            self.state = torch.zeros(sb, dtype=torch.uint8, device=self.device)
            self.scratch = torch.empty(self.lib.u1u1_slab_scratch_bytes(self.N, self.nz_own), dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._ctx = ctypes.c_void_p()
        rc = self.lib.u1u1_create(ctypes.byref(self._ctx), self.state.data_ptr(), sb, self.scratch.data_ptr(),
                                  self.scratch.numel(), self.stream.cuda_stream)
        if rc:
            raise B.U1U1Error(f"u1u1_create: {self.lib.u1u1_last_error(None).decode()}")

    _check = Lattice._check
    close = Lattice.close
    __del__ = Lattice.__del__
    set_params = Lattice.set_params
    step = Lattice.step
    launch_count = Lattice.launch_count

    set_tuning = Lattice.set_tuning

    def configure_slab(self, dx: float, params: B.Params):
        self.set_tuning(getattr(params, "tuning", 0))
        self._check(self.lib.u1u1_configure_slab(self._ctx, self.N, self.nz_own, self.z_first, dx, ctypes.byref(params)),
                    "configure_slab")

    def set_slab_peers(self, up_state_ptr: int, dn_state_ptr: int):
        self._check(self.lib.u1u1_set_slab_peers(self._ctx, up_state_ptr, dn_state_ptr), "set_slab_peers")

    def init_slab(self, seed: int):
        self._check(self.lib.u1u1_init_slab(self._ctx, seed), "init_slab")

    def push_halos(self):
        self._check(self.lib.u1u1_push_halos(self._ctx), "push_halos")

    def push_diag_halos(self):
        self._check(self.lib.u1u1_push_diag_halos(self._ctx), "push_diag_halos")

    def slab_diagnostics_partial(self) -> np.ndarray:
        raw = (ctypes.c_double * B.SLAB_NRAW)()
        self._check(self.lib.u1u1_slab_diagnostics_partial(self._ctx, raw), "slab_diagnostics_partial")
        return np.array(raw[:])

    def slab_diagnostics_finish(self, raw_reduced, nz_global: int) -> dict:
        raw = (ctypes.c_double * B.SLAB_NRAW)(*[float(v) for v in raw_reduced])
        out = (ctypes.c_double * B.DIAG_LEN)()
        self._check(self.lib.u1u1_slab_diagnostics_finish(self._ctx, raw, nz_global, out), "slab_diagnostics_finish")
        return {k: out[i] for i, k in enumerate(B.DIAG_SLOTS)}

    def export_slab(self):
        t = self._torch.empty((20, self.nz_own, self.N, self.N), dtype=self._torch.float32, device=self.device)
        self._check(self.lib.u1u1_export_slab(self._ctx, t.data_ptr()), "export_slab")
        return t

    def import_slab(self, t):
        torch = self._torch
        t = t.to(device=self.device, dtype=torch.float32).contiguous()
        assert tuple(t.shape) == (20, self.nz_own, self.N, self.N), t.shape
        self._check(self.lib.u1u1_import_slab(self._ctx, t.data_ptr()), "import_slab")
        self.stream.synchronize()


def gauss_violation_static(state, dx: float, e1: float, e2: float, cG: float, out=None, stream=None):
    """u1u1_gauss_violation_static: the Gauss-law norms of a canonical float32 [20, N, N, N] device tensor, for callers
    that cannot hand the library a scratch buffer (their framework's pool owns the whole GPU, or they run where a
    cudaMalloc would stall the device).  No context is involved and the library allocates nothing: the partial sums go
    through a fixed array inside libu1u1.so, shared by every call on that GPU -- so keep calls on one stream, or order
    them.  `out` (8 float64 on the same device) is filled asynchronously on `stream` and returned; pass your own to keep
    this wrapper allocation-free as well.  Raises U1U1Error with the library's message, e.g. for N > STATIC_MAX_N."""
    import torch
    lib = B.load()
    if state.dtype != torch.float32 or not state.is_cuda or not state.is_contiguous() or state.dim() != 4 \
            or state.shape[0] != 20 or not (state.shape[1] == state.shape[2] == state.shape[3]):
        raise B.U1U1Error("gauss_violation_static: need a contiguous float32 CUDA tensor [20, N, N, N]")
    with torch.cuda.device(state.device):
        if out is None:
            out = torch.empty(B.GAUSS_LEN, dtype=torch.float64, device=state.device)
        st = stream if stream is not None else torch.cuda.current_stream(state.device)
        err = ctypes.create_string_buffer(256)
        rc = lib.u1u1_gauss_violation_static(state.data_ptr(), int(state.shape[1]), dx, e1, e2, cG, out.data_ptr(),
                                             st.cuda_stream, err, len(err))
    if rc:
        raise B.U1U1Error(f"{B.ERRORS.get(rc, rc)}: {err.value.decode()}")
    return out
