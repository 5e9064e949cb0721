"""Thin ctypes binding of libfcg.so -- same names as the C calls of include/fcg.h, argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; torch is used for device memory and
streams.  There is no CPU fallback: loading fails loudly when libfcg.so is missing, and fcg_create
fails when there is no CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("FCG_LIB") or os.path.join(_HERE, "libfcg.so")      # FCG_LIB: a variant build for A/B measurements

FCG_F32, FCG_F64 = 0, 1
FCG_OK, FCG_NOT_CONVERGED = 0, 1
FCG_INVALID_ARG, FCG_UNSUPPORTED, FCG_CUDA_ERROR, FCG_BREAKDOWN, FCG_NO_SPECTRUM, FCG_NO_CANDIDATE = -1, -2, -3, -4, -5, -6
FCG_OPT_LOOP_MODE, FCG_OPT_CHUNK, FCG_OPT_ROW_VARIANT, FCG_OPT_ENGINE, FCG_OPT_UNROLL, FCG_OPT_PDL, FCG_OPT_FUSED = 0, 1, 2, 3, 4, 5, 6
FCG_OPT_L2_HINTS = 7
FCG_OPT_SPECTRAL_ALPHA = 8
FCG_OPT_COL_PERSISTENT = 9
FCG_OPT_BARRIER_START = 10
FCG_OPT_FFT_DIRECT = 11
FCG_OPT_FUSED_TWO = 12
FCG_OPT_STAGGER_P1, FCG_OPT_STAGGER_P2, FCG_OPT_STAGGER_P3 = 13, 14, 15
FCG_SLAB_IPC_BYTES = 80

EXPORTS = ["fcg_workspace_bytes", "fcg_create", "fcg_destroy", "fcg_set_option", "fcg_set_spectrum", "fcg_apply",
           "fcg_solve", "fcg_solve_host", "fcg_profile_iteration", "fcg_fft_fwd", "fcg_fft_inv", "fcg_break_step", "fcg_fracture",
           "fcg_last_launch_count", "fcg_last_error", "fcg_version",
           "fcg_set_preconditioner", "fcg_pcg_solve", "fcg_profile_pcg_iteration", "fcg_pcg_fracture",
           "fcg_fracture_begin", "fcg_fracture_end",
           "fcg_green_function", "fcg_kernel_spectrum", "fcg_force_apply", "fcg_force_solve", "fcg_force_break_step",
           "fcg_force_fracture", "fcg_inverse_spectrum", "fcg_force_rhs", "fcg_force_from_displacement",
           "fcg_force_fracture_displacement", "fcg_force_fracture_displacement_begin", "fcg_force_fracture_displacement_end",
           "fcg_set_stream", "fcg_get_option", "fcg_solve_host_submit", "fcg_solve_host_wait", "fcg_slab_shape_of", "fcg_slab_configure", "fcg_slab_buffers", "fcg_slab_set_peers", "fcg_slab_ipc_export", "fcg_slab_ipc_open", "fcg_slab_setup", "fcg_slab_rows_fwd", "fcg_slab_cols", "fcg_slab_cols_energy", "fcg_slab_kpp0", "fcg_slab_rows_inv", "fcg_slab_update_r", "fcg_slab_scalar", "fcg_slab_finish", "fcg_slab_poll",
           "fcg_break_step_static", "fcg_static_last_error"]


class SlabShape(C.Structure):
    """fcg_slab_shape of include/fcg.h."""
    _fields_ = [("nranks", C.c_int), ("rank", C.c_int), ("columns_per_line", C.c_int), ("column_blocks", C.c_int),
                ("column_blocks_local", C.c_int), ("row_pairs_local", C.c_int), ("rows_local", C.c_int), ("columns_local", C.c_int),
                ("column0", C.c_int), ("line_bytes", C.c_size_t), ("chunk_bytes", C.c_size_t), ("buffer_bytes", C.c_size_t)]

_lib = None


class FcgError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"fcg status {status}: {msg}")
        self.status = status


def lib() -> C.CDLL:
    """Load libfcg.so (built in-tree by paper_1305_3625_b200.build). Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} not found: run `python -m paper_1305_3625_b200.build` (there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i, d, ll = C.c_void_p, C.c_int, C.c_double, C.c_longlong
        L.fcg_workspace_bytes.argtypes = [i, i]; L.fcg_workspace_bytes.restype = C.c_size_t
        L.fcg_create.argtypes = [i, i, vp, vp, C.POINTER(vp)]; L.fcg_create.restype = i
        L.fcg_destroy.argtypes = [vp]; L.fcg_destroy.restype = i
        L.fcg_set_option.argtypes = [vp, i, i]; L.fcg_set_option.restype = i
        L.fcg_set_spectrum.argtypes = [vp, vp]; L.fcg_set_spectrum.restype = i
        L.fcg_apply.argtypes = [vp, vp, vp, vp]; L.fcg_apply.restype = i
        L.fcg_solve.argtypes = [vp, vp, vp, vp, d, i, C.POINTER(i), C.POINTER(d)]; L.fcg_solve.restype = i
        L.fcg_solve_host.argtypes = [vp, vp, vp, vp, d, i, C.POINTER(i), C.POINTER(d)]; L.fcg_solve_host.restype = i
        L.fcg_fft_fwd.argtypes = [vp, vp, vp]; L.fcg_fft_fwd.restype = i
        L.fcg_fft_inv.argtypes = [vp, vp, vp]; L.fcg_fft_inv.restype = i
        L.fcg_break_step.argtypes = [vp, vp, vp, vp, C.POINTER(ll), C.POINTER(d)]; L.fcg_break_step.restype = i
        L.fcg_fracture.argtypes = [vp, vp, vp, vp, vp, i, d, i, vp, vp, C.POINTER(i)]; L.fcg_fracture.restype = i
        L.fcg_pcg_fracture.argtypes = [vp, vp, vp, vp, vp, i, d, i, vp, vp, C.POINTER(i)]; L.fcg_pcg_fracture.restype = i
        L.fcg_fracture_begin.argtypes = [vp, vp, vp, vp, vp, i, d, i, i]; L.fcg_fracture_begin.restype = i
        L.fcg_fracture_end.argtypes = [vp, vp, vp, C.POINTER(i)]; L.fcg_fracture_end.restype = i
        L.fcg_profile_iteration.argtypes = [vp, vp, vp, vp, i, C.POINTER(d)]; L.fcg_profile_iteration.restype = i
        L.fcg_set_preconditioner.argtypes = [vp, vp, d]; L.fcg_set_preconditioner.restype = i
        L.fcg_pcg_solve.argtypes = [vp, vp, vp, vp, d, i, C.POINTER(i), C.POINTER(d)]; L.fcg_pcg_solve.restype = i
        L.fcg_profile_pcg_iteration.argtypes = [vp, vp, vp, vp, i, C.POINTER(d)]; L.fcg_profile_pcg_iteration.restype = i
        L.fcg_green_function.argtypes = [vp, d, d, d, vp]; L.fcg_green_function.restype = i
        L.fcg_kernel_spectrum.argtypes = [vp, vp, vp]; L.fcg_kernel_spectrum.restype = i
        L.fcg_force_apply.argtypes = [vp, vp, vp, vp]; L.fcg_force_apply.restype = i
        L.fcg_inverse_spectrum.argtypes = [vp, vp, vp]; L.fcg_inverse_spectrum.restype = i
        L.fcg_force_fracture_displacement.argtypes = [vp, vp, d, vp, vp, i, d, i, i, vp, vp, vp, C.POINTER(i)]
        L.fcg_force_fracture_displacement.restype = i
        L.fcg_force_fracture_displacement_begin.argtypes = [vp, vp, d, vp, vp, i, d, i, i]
        L.fcg_force_fracture_displacement_begin.restype = i
        L.fcg_force_fracture_displacement_end.argtypes = [vp, vp, vp, vp, C.POINTER(i)]
        L.fcg_force_fracture_displacement_end.restype = i
        L.fcg_force_rhs.argtypes = [vp, vp, d, vp]; L.fcg_force_rhs.restype = i
        L.fcg_force_from_displacement.argtypes = [vp, vp, d, vp, vp]; L.fcg_force_from_displacement.restype = i
        L.fcg_force_solve.argtypes = [vp, vp, d, vp, d, i, C.POINTER(i), C.POINTER(d)]; L.fcg_force_solve.restype = i
        L.fcg_force_break_step.argtypes = [vp, vp, vp, vp, C.POINTER(ll), C.POINTER(d)]; L.fcg_force_break_step.restype = i
        L.fcg_force_fracture.argtypes = [vp, vp, d, vp, vp, i, d, i, vp, vp, vp, C.POINTER(i)]; L.fcg_force_fracture.restype = i
        L.fcg_slab_shape_of.argtypes = [i, i, i, i, C.POINTER(SlabShape)]; L.fcg_slab_shape_of.restype = i
        L.fcg_slab_configure.argtypes = [vp, i, i]; L.fcg_slab_configure.restype = i
        L.fcg_slab_buffers.argtypes = [vp, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]; L.fcg_slab_buffers.restype = i
        L.fcg_slab_set_peers.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]; L.fcg_slab_set_peers.restype = i
        L.fcg_slab_ipc_export.argtypes = [vp, vp]; L.fcg_slab_ipc_export.restype = i
        L.fcg_slab_ipc_open.argtypes = [vp, vp]; L.fcg_slab_ipc_open.restype = i
        L.fcg_slab_setup.argtypes = [vp, d, i]; L.fcg_slab_setup.restype = i
        L.fcg_slab_rows_fwd.argtypes = [vp, i, vp]; L.fcg_slab_rows_fwd.restype = i
        L.fcg_set_stream.argtypes = [vp, vp]; L.fcg_set_stream.restype = i
        L.fcg_get_option.argtypes = [vp, i, C.POINTER(i)]; L.fcg_get_option.restype = i
        L.fcg_solve_host_submit.argtypes = [vp, vp, vp, vp, C.c_double, i]; L.fcg_solve_host_submit.restype = i
        L.fcg_solve_host_wait.argtypes = [vp, C.POINTER(i), C.POINTER(C.c_double)]; L.fcg_solve_host_wait.restype = i
        L.fcg_slab_cols.argtypes = [vp]; L.fcg_slab_cols.restype = i
        L.fcg_slab_cols_energy.argtypes = [vp, vp]; L.fcg_slab_cols_energy.restype = i
        L.fcg_slab_kpp0.argtypes = [vp, vp, vp]; L.fcg_slab_kpp0.restype = i
        L.fcg_slab_rows_inv.argtypes = [vp, i, vp, vp, vp, vp]; L.fcg_slab_rows_inv.restype = i
        L.fcg_slab_update_r.argtypes = [vp, vp]; L.fcg_slab_update_r.restype = i
        L.fcg_slab_scalar.argtypes = [vp, i, vp]; L.fcg_slab_scalar.restype = i
        L.fcg_slab_finish.argtypes = [vp, vp]; L.fcg_slab_finish.restype = i
        L.fcg_slab_poll.argtypes = [vp, C.POINTER(i), C.POINTER(i), C.POINTER(d), C.POINTER(i)]; L.fcg_slab_poll.restype = i
        L.fcg_break_step_static.argtypes = [i, ll, vp, vp, vp, vp, vp]; L.fcg_break_step_static.restype = i
        L.fcg_static_last_error.argtypes = []; L.fcg_static_last_error.restype = C.c_char_p
        L.fcg_last_launch_count.argtypes = [vp]; L.fcg_last_launch_count.restype = ll
        L.fcg_last_error.argtypes = [vp]; L.fcg_last_error.restype = C.c_char_p
        L.fcg_version.argtypes = []; L.fcg_version.restype = C.c_char_p
        _lib = L
    return _lib


def _dt(dtype) -> int:
    if dtype == torch.float64:
        return FCG_F64
    if dtype == torch.float32:
        return FCG_F32
    raise TypeError(f"fcg supports torch.float32/float64, got {dtype}")


class Fcg:
    """One handle = one lattice size and dtype on the current CUDA device and stream (fcg_create)."""

    def __init__(self, L: int, dtype=torch.float64, device="cuda", stream: torch.cuda.Stream | None = None,
                 own_workspace: bool = False):
        self.L, self.N, self.dtype = L, L * L, dtype
        self.device = torch.device(device)
        self._lib = lib()
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            self.stream = stream or torch.cuda.current_stream(self.device)
            nbytes = self._lib.fcg_workspace_bytes(L, _dt(dtype))
            if nbytes == 0:
                raise FcgError(FCG_UNSUPPORTED, f"L={L} unsupported (power of two, 16..8192)")
            self._ws = None if own_workspace else torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            ws_ptr = None if own_workspace else self._ws.data_ptr()
            st = self._lib.fcg_create(L, _dt(dtype), ws_ptr, self.stream.cuda_stream, C.byref(self._h))
        if st != FCG_OK:
            self._h = C.c_void_p()
            raise FcgError(st, "fcg_create failed (no CUDA device, or unsupported size)")

    # -- helpers -------------------------------------------------------------------------------
    def _chk(self, t: torch.Tensor, numel: int | None = None, dtype=None) -> int:
        dtype = dtype or self.dtype
        if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
            raise ValueError(f"expected contiguous CUDA tensor of {dtype}")
        if numel is not None and t.numel() != numel:
            raise ValueError(f"expected {numel} elements, got {t.numel()}")
        return t.data_ptr()

    def _raise(self, st: int):
        raise FcgError(st, self._lib.fcg_last_error(self._h).decode())

    def last_error(self) -> str:
        return self._lib.fcg_last_error(self._h).decode()

    def close(self):
        if self._h:
            self._lib.fcg_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C calls -----------------------------------------------------------------------------
    def fcg_set_option(self, option: int, value: int):
        st = self._lib.fcg_set_option(self._h, option, value)
        if st != FCG_OK:
            self._raise(st)

    def fcg_set_spectrum(self, s: torch.Tensor):
        st = self._lib.fcg_set_spectrum(self._h, self._chk(s, self.N))
        if st != FCG_OK:
            self._raise(st)

    def fcg_apply(self, k: torch.Tensor, x: torch.Tensor, y: torch.Tensor | None = None) -> torch.Tensor:
        y = torch.empty_like(x) if y is None else y
        st = self._lib.fcg_apply(self._h, self._chk(k, self.N), self._chk(x, self.N), self._chk(y, self.N))
        if st != FCG_OK:
            self._raise(st)
        return y

    def fcg_solve(self, k: torch.Tensor, f: torch.Tensor, u: torch.Tensor, tol: float, maxit: int):
        """In place on u. Returns (iters, rel_residual, status); raises on error statuses other than BREAKDOWN."""
        it = C.c_int(0); rr = C.c_double(0.0)
        st = self._lib.fcg_solve(self._h, self._chk(k, self.N), self._chk(f, self.N), self._chk(u, self.N),
                                 float(tol), int(maxit), C.byref(it), C.byref(rr))
        if st < 0 and st != FCG_BREAKDOWN:
            self._raise(st)
        return int(it.value), float(rr.value), int(st)

    def fcg_set_preconditioner(self, s: torch.Tensor, kbar: float):
        st = self._lib.fcg_set_preconditioner(self._h, self._chk(s, self.N), float(kbar))
        if st != FCG_OK:
            self._raise(st)

    def fcg_pcg_solve(self, k: torch.Tensor, f: torch.Tensor, u: torch.Tensor, tol: float, maxit: int):
        """Preconditioned CG, in place on u. Returns (iters, rel_residual, status) like fcg_solve."""
        it = C.c_int(0); rr = C.c_double(0.0)
        st = self._lib.fcg_pcg_solve(self._h, self._chk(k, self.N), self._chk(f, self.N), self._chk(u, self.N),
                                     float(tol), int(maxit), C.byref(it), C.byref(rr))
        if st < 0 and st != FCG_BREAKDOWN:
            self._raise(st)
        return int(it.value), float(rr.value), int(st)

    def fcg_solve_host(self, k: torch.Tensor, f: torch.Tensor, u: torch.Tensor, tol: float, maxit: int):
        """Same with HOST tensors (pinned for full copy speed); u updated in place."""
        for t in (k, f, u):
            if t.is_cuda or not t.is_contiguous() or t.dtype != self.dtype or t.numel() != self.N:
                raise ValueError("expected contiguous host tensors of the handle's dtype and size")
        it = C.c_int(0); rr = C.c_double(0.0)
        st = self._lib.fcg_solve_host(self._h, k.data_ptr(), f.data_ptr(), u.data_ptr(), float(tol), int(maxit),
                                      C.byref(it), C.byref(rr))
        if st < 0 and st != FCG_BREAKDOWN:
            self._raise(st)
        return int(it.value), float(rr.value), int(st)

    def fcg_solve_host_submit(self, k: torch.Tensor, f: torch.Tensor, u: torch.Tensor, tol: float, maxit: int):
        """Pipelined fcg_solve_host: returns once the copies and the solve are enqueued (up to two outstanding); keep k, f, u alive
        and untouched until the matching fcg_solve_host_wait."""
        for t in (k, f, u):
            if t.is_cuda or not t.is_contiguous() or t.dtype != self.dtype or t.numel() != self.N:
                raise ValueError("expected contiguous host tensors of the handle's dtype and size")
        self._ok(self._lib.fcg_solve_host_submit(self._h, k.data_ptr(), f.data_ptr(), u.data_ptr(), float(tol), int(maxit)))

    def fcg_solve_host_wait(self):
        """(iters, rel_residual, status) of the oldest outstanding fcg_solve_host_submit; its u tensor now holds the solution."""
        it = C.c_int(0); rr = C.c_double(0.0)
        st = self._lib.fcg_solve_host_wait(self._h, C.byref(it), C.byref(rr))
        if st < 0 and st != FCG_BREAKDOWN:
            self._raise(st)
        return int(it.value), float(rr.value), int(st)

    def fcg_fft_fwd(self, x: torch.Tensor, X: torch.Tensor | None = None) -> torch.Tensor:
        cdt = torch.complex128 if self.dtype == torch.float64 else torch.complex64
        X = torch.empty((self.L, self.L // 2 + 1), dtype=cdt, device=x.device) if X is None else X
        st = self._lib.fcg_fft_fwd(self._h, self._chk(x, self.N), self._chk(X, self.L * (self.L // 2 + 1), cdt))
        if st != FCG_OK:
            self._raise(st)
        return X

    def fcg_fft_inv(self, X: torch.Tensor, x: torch.Tensor | None = None) -> torch.Tensor:
        cdt = torch.complex128 if self.dtype == torch.float64 else torch.complex64
        x = torch.empty((self.L, self.L), dtype=self.dtype, device=X.device) if x is None else x
        st = self._lib.fcg_fft_inv(self._h, self._chk(X, self.L * (self.L // 2 + 1), cdt), self._chk(x, self.N))
        if st != FCG_OK:
            self._raise(st)
        return x

    def fcg_break_step(self, k: torch.Tensor, u: torch.Tensor, t: torch.Tensor):
        """In place on k. Returns (index, ratio, status)."""
        idx = C.c_longlong(-1); ratio = C.c_double(0.0)
        st = self._lib.fcg_break_step(self._h, self._chk(k, self.N), self._chk(u, self.N), self._chk(t, self.N),
                                      C.byref(idx), C.byref(ratio))
        if st < 0 and st != FCG_NO_CANDIDATE:
            self._raise(st)
        return int(idx.value), float(ratio.value), int(st)

    def fcg_fracture_begin(self, k, f, u, t, nsteps: int, tol: float, maxit: int, use_pcg: bool = False):
        """Enqueue a quasi-static loop (returns at once where the loop is one cooperative kernel); finish with fcg_fracture_end."""
        st = self._lib.fcg_fracture_begin(self._h, self._chk(k, self.N), self._chk(f, self.N), self._chk(u, self.N),
                                          self._chk(t, self.N), int(nsteps), float(tol), int(maxit), 1 if use_pcg else 0)
        if st < 0 and st not in (FCG_BREAKDOWN, FCG_NO_CANDIDATE):
            self._raise(st)
        self._pending = (k, f, u, t, int(nsteps))              # keep the tensors alive

    def fcg_fracture_end(self):
        """Returns (index, iters, steps_done, status) of the loop started by fcg_fracture_begin."""
        import numpy as np
        if getattr(self, "_pending", None) is None:
            raise FcgError(FCG_INVALID_ARG, "no quasi-static loop pending on this handle")
        nsteps = self._pending[4]
        index = np.full(nsteps, -1, np.int64); iters = np.zeros(nsteps, np.int32); done = C.c_int(0)
        st = self._lib.fcg_fracture_end(self._h, index.ctypes.data_as(C.c_void_p), iters.ctypes.data_as(C.c_void_p), C.byref(done))
        self._pending = None
        if st < 0 and st not in (FCG_BREAKDOWN, FCG_NO_CANDIDATE):
            self._raise(st)
        return index, iters, int(done.value), int(st)

    def fcg_pcg_fracture(self, k, f, u, t, nsteps: int, tol: float, maxit: int):
        """fcg_fracture with preconditioned-CG solves (fcg_set_preconditioner first)."""
        return self.fcg_fracture(k, f, u, t, nsteps, tol, maxit, _fn="fcg_pcg_fracture")

    def fcg_fracture(self, k: torch.Tensor, f: torch.Tensor, u: torch.Tensor, t: torch.Tensor, nsteps: int,
                     tol: float, maxit: int, _fn: str = "fcg_fracture"):
        """In place on k and u. Returns (index[int64 numpy], iters[int32 numpy], steps_done, status)."""
        import numpy as np
        index = np.full(nsteps, -1, np.int64); iters = np.zeros(nsteps, np.int32); done = C.c_int(0)
        st = getattr(self._lib, _fn)(self._h, self._chk(k, self.N), self._chk(f, self.N), self._chk(u, self.N),
                                    self._chk(t, self.N), int(nsteps), float(tol), int(maxit),
                                    index.ctypes.data_as(C.c_void_p), iters.ctypes.data_as(C.c_void_p), C.byref(done))
        if st < 0 and st not in (FCG_BREAKDOWN, FCG_NO_CANDIDATE):
            self._raise(st)
        return index, iters, int(done.value), int(st)

    def fcg_profile_iteration(self, k: torch.Tensor, f: torch.Tensor, u: torch.Tensor, iters: int):
        """Mean device milliseconds of the four loop kernels [row_fwd, col, row_inv, update_r]; overwrites u."""
        ms = (C.c_double * 4)()
        st = self._lib.fcg_profile_iteration(self._h, self._chk(k, self.N), self._chk(f, self.N), self._chk(u, self.N),
                                             int(iters), ms)
        if st != FCG_OK:
            self._raise(st)
        return [float(x) for x in ms]

    def fcg_profile_pcg_iteration(self, k: torch.Tensor, f: torch.Tensor, u: torch.Tensor, iters: int):
        """Mean device milliseconds of the six kernels of one PCG iteration; overwrites u."""
        ms = (C.c_double * 6)()
        st = self._lib.fcg_profile_pcg_iteration(self._h, self._chk(k, self.N), self._chk(f, self.N), self._chk(u, self.N),
                                                 int(iters), ms)
        if st != FCG_OK:
            self._raise(st)
        return [float(x) for x in ms]

    # -- the paper's formulation in the bond forces, (I + K G) f = K D (include/fcg.h) ---------------------
    def fcg_green_function(self, nu: float, E: float, a: float, G: torch.Tensor | None = None) -> torch.Tensor:
        G = torch.empty((self.L, self.L), dtype=self.dtype, device=self.device) if G is None else G
        st = self._lib.fcg_green_function(self._h, float(nu), float(E), float(a), self._chk(G, self.N))
        if st != FCG_OK:
            self._raise(st)
        return G

    def fcg_kernel_spectrum(self, G: torch.Tensor, s: torch.Tensor | None = None) -> torch.Tensor:
        s = torch.empty((self.L, self.L), dtype=self.dtype, device=G.device) if s is None else s
        st = self._lib.fcg_kernel_spectrum(self._h, self._chk(G, self.N), self._chk(s, self.N))
        if st != FCG_OK:
            self._raise(st)
        return s

    def fcg_inverse_spectrum(self, g: torch.Tensor, s: torch.Tensor | None = None) -> torch.Tensor:
        s = torch.empty_like(g) if s is None else s
        st = self._lib.fcg_inverse_spectrum(self._h, self._chk(g, self.N), self._chk(s, self.N))
        if st != FCG_OK:
            self._raise(st)
        return s

    def fcg_force_rhs(self, k: torch.Tensor, D: float, b: torch.Tensor | None = None) -> torch.Tensor:
        b = torch.empty_like(k) if b is None else b
        st = self._lib.fcg_force_rhs(self._h, self._chk(k, self.N), float(D), self._chk(b, self.N))
        if st != FCG_OK:
            self._raise(st)
        return b

    def fcg_force_from_displacement(self, k: torch.Tensor, D: float, u: torch.Tensor, f: torch.Tensor | None = None) -> torch.Tensor:
        f = torch.empty_like(u) if f is None else f
        st = self._lib.fcg_force_from_displacement(self._h, self._chk(k, self.N), float(D), self._chk(u, self.N), self._chk(f, self.N))
        if st != FCG_OK:
            self._raise(st)
        return f

    def fcg_force_apply(self, k: torch.Tensor, x: torch.Tensor, y: torch.Tensor | None = None) -> torch.Tensor:
        y = torch.empty_like(x) if y is None else y
        st = self._lib.fcg_force_apply(self._h, self._chk(k, self.N), self._chk(x, self.N), self._chk(y, self.N))
        if st != FCG_OK:
            self._raise(st)
        return y

    def fcg_force_solve(self, k: torch.Tensor, D: float, f: torch.Tensor, tol: float, maxit: int):
        """In place on f. Returns (iters, rel_residual, status) like fcg_solve."""
        it = C.c_int(0); rr = C.c_double(0.0)
        st = self._lib.fcg_force_solve(self._h, self._chk(k, self.N), float(D), self._chk(f, self.N), float(tol), int(maxit),
                                       C.byref(it), C.byref(rr))
        if st < 0 and st != FCG_BREAKDOWN:
            self._raise(st)
        return int(it.value), float(rr.value), int(st)

    def fcg_force_break_step(self, k: torch.Tensor, f: torch.Tensor, t: torch.Tensor):
        """In place on k and f. Returns (index, ratio, status)."""
        idx = C.c_longlong(-1); ratio = C.c_double(0.0)
        st = self._lib.fcg_force_break_step(self._h, self._chk(k, self.N), self._chk(f, self.N), self._chk(t, self.N),
                                            C.byref(idx), C.byref(ratio))
        if st < 0 and st != FCG_NO_CANDIDATE:
            self._raise(st)
        return int(idx.value), float(ratio.value), int(st)

    def fcg_force_fracture(self, k: torch.Tensor, D: float, f: torch.Tensor, t: torch.Tensor, nsteps: int, tol: float, maxit: int):
        """In place on k and f. Returns (index[int64], iters[int32], ratio[float64], steps_done, status)."""
        import numpy as np
        index = np.full(nsteps, -1, np.int64); iters = np.zeros(nsteps, np.int32); ratio = np.full(nsteps, np.nan, np.float64)
        done = C.c_int(0)
        st = self._lib.fcg_force_fracture(self._h, self._chk(k, self.N), float(D), self._chk(f, self.N), self._chk(t, self.N),
                                          int(nsteps), float(tol), int(maxit), index.ctypes.data_as(C.c_void_p),
                                          iters.ctypes.data_as(C.c_void_p), ratio.ctypes.data_as(C.c_void_p), C.byref(done))
        if st < 0 and st not in (FCG_BREAKDOWN, FCG_NO_CANDIDATE):
            self._raise(st)
        return index, iters, ratio, int(done.value), int(st)

    def fcg_force_fracture_displacement(self, k: torch.Tensor, D: float, u: torch.Tensor, t: torch.Tensor, nsteps: int, tol: float,
                                        maxit: int, use_pcg: bool = False):
        """In place on k and u. Returns (index[int64], iters[int32], ratio[float64], steps_done, status)."""
        import numpy as np
        index = np.full(nsteps, -1, np.int64); iters = np.zeros(nsteps, np.int32); ratio = np.full(nsteps, np.nan, np.float64)
        done = C.c_int(0)
        st = self._lib.fcg_force_fracture_displacement(self._h, self._chk(k, self.N), float(D), self._chk(u, self.N), self._chk(t, self.N),
                                                       int(nsteps), float(tol), int(maxit), 1 if use_pcg else 0,
                                                       index.ctypes.data_as(C.c_void_p), iters.ctypes.data_as(C.c_void_p),
                                                       ratio.ctypes.data_as(C.c_void_p), C.byref(done))
        if st < 0 and st not in (FCG_BREAKDOWN, FCG_NO_CANDIDATE):
            self._raise(st)
        return index, iters, ratio, int(done.value), int(st)

    def fcg_force_fracture_displacement_begin(self, k: torch.Tensor, D: float, u: torch.Tensor, t: torch.Tensor, nsteps: int, tol: float,
                                              maxit: int, use_pcg: bool = False) -> None:
        """Enqueue half; keep k, u, t alive and untouched until fcg_force_fracture_displacement_end()."""
        st = self._lib.fcg_force_fracture_displacement_begin(self._h, self._chk(k, self.N), float(D), self._chk(u, self.N),
                                                             self._chk(t, self.N), int(nsteps), float(tol), int(maxit), 1 if use_pcg else 0)
        if st < 0 and st not in (FCG_BREAKDOWN, FCG_NO_CANDIDATE):
            self._raise(st)
        self._pend = (k, u, t, int(nsteps))

    def fcg_force_fracture_displacement_end(self):
        """Collect half. Returns (index[int64], iters[int32], ratio[float64], steps_done, status)."""
        import numpy as np
        if getattr(self, "_pend", None) is None:
            raise FcgError(FCG_INVALID_ARG, "no quasi-static loop pending on this handle")
        nsteps = self._pend[3]
        index = np.full(nsteps, -1, np.int64); iters = np.zeros(nsteps, np.int32); ratio = np.full(nsteps, np.nan, np.float64)
        done = C.c_int(0)
        st = self._lib.fcg_force_fracture_displacement_end(self._h, index.ctypes.data_as(C.c_void_p), iters.ctypes.data_as(C.c_void_p),
                                                           ratio.ctypes.data_as(C.c_void_p), C.byref(done))
        self._pend = None
        if st < 0 and st not in (FCG_BREAKDOWN, FCG_NO_CANDIDATE):
            self._raise(st)
        return index, iters, ratio, int(done.value), int(st)

    # -- slab-decomposed CG over several ranks (include/fcg.h): the local passes of one rank -------------------
    def _ok(self, st: int):
        if st != FCG_OK:
            self._raise(st)

    def fcg_slab_configure(self, nranks: int, rank: int):
        self._ok(self._lib.fcg_slab_configure(self._h, int(nranks), int(rank)))

    def fcg_slab_buffers(self):
        """(send, recv): uint8 views of the handle's workspace -- the two exchange buffers of this rank."""
        if self._ws is None:
            raise ValueError("slab buffers are views of the caller-owned workspace (own_workspace=False)")
        so, ro, nb = C.c_size_t(0), C.c_size_t(0), C.c_size_t(0)
        self._ok(self._lib.fcg_slab_buffers(self._h, C.byref(so), C.byref(ro), C.byref(nb)))
        return self._ws[so.value: so.value + nb.value], self._ws[ro.value: ro.value + nb.value]

    def fcg_slab_set_peers(self, peer_send, peer_recv):
        """peer_send / peer_recv: device addresses (ints) of every rank's S and R buffer, valid on this device; None, None: off."""
        if peer_send is None:
            self._ok(self._lib.fcg_slab_set_peers(self._h, None, None))
            return
        n = len(peer_send)
        a = (C.c_void_p * n)(*[int(x) for x in peer_send]); b = (C.c_void_p * n)(*[int(x) for x in peer_recv])
        self._ok(self._lib.fcg_slab_set_peers(self._h, a, b))

    def fcg_slab_ipc_export(self) -> bytes:
        buf = C.create_string_buffer(FCG_SLAB_IPC_BYTES)
        self._ok(self._lib.fcg_slab_ipc_export(self._h, buf))
        return buf.raw

    def fcg_slab_ipc_open(self, blobs: bytes):
        buf = C.create_string_buffer(bytes(blobs), len(blobs))
        self._ok(self._lib.fcg_slab_ipc_open(self._h, buf))

    def fcg_get_option(self, option: int) -> int:
        """The effective value of an option (automatic choices resolved for this size and dtype)."""
        v = C.c_int(0)
        self._ok(self._lib.fcg_get_option(self._h, int(option), C.byref(v)))
        return int(v.value)

    def fcg_set_stream(self, stream: torch.cuda.Stream):
        self._ok(self._lib.fcg_set_stream(self._h, stream.cuda_stream))
        self.stream = stream

    def fcg_slab_setup(self, tol: float, maxit: int):
        self._ok(self._lib.fcg_slab_setup(self._h, float(tol), int(maxit)))

    def fcg_slab_rows_fwd(self, cg: bool, xu: torch.Tensor):
        self._ok(self._lib.fcg_slab_rows_fwd(self._h, 1 if cg else 0, self._chk(xu)))

    def fcg_slab_cols(self):
        self._ok(self._lib.fcg_slab_cols(self._h))

    def fcg_slab_cols_energy(self, xch: torch.Tensor):
        self._ok(self._lib.fcg_slab_cols_energy(self._h, self._chk(xch, 4, torch.float64)))

    def fcg_slab_kpp0(self, k: torch.Tensor, xch: torch.Tensor):
        self._ok(self._lib.fcg_slab_kpp0(self._h, self._chk(k), self._chk(xch, 4, torch.float64)))

    def fcg_slab_rows_inv(self, residual, k: torch.Tensor, u, f, xch: torch.Tensor):
        """residual: 0 / False (q = A p), 1 / True (r = f - A u), 2 (fused: r -= alpha A p)."""
        self._ok(self._lib.fcg_slab_rows_inv(self._h, int(residual), self._chk(k), self._chk(u) if u is not None else None,
                                             self._chk(f) if f is not None else None, self._chk(xch, 4, torch.float64)))

    def fcg_slab_update_r(self, xch: torch.Tensor):
        self._ok(self._lib.fcg_slab_update_r(self._h, self._chk(xch, 4, torch.float64)))

    def fcg_slab_scalar(self, what: int, xch: torch.Tensor):
        self._ok(self._lib.fcg_slab_scalar(self._h, int(what), self._chk(xch, 4, torch.float64)))

    def fcg_slab_finish(self, u: torch.Tensor):
        self._ok(self._lib.fcg_slab_finish(self._h, self._chk(u)))

    def fcg_slab_poll(self):
        """(done, iters, rel_residual, status) of the scalar block; blocks."""
        dn, it, st = C.c_int(0), C.c_int(0), C.c_int(0); rr = C.c_double(0.0)
        self._ok(self._lib.fcg_slab_poll(self._h, C.byref(dn), C.byref(it), C.byref(rr), C.byref(st)))
        return bool(dn.value), int(it.value), float(rr.value), int(st.value)

    def fcg_last_launch_count(self) -> int:
        return int(self._lib.fcg_last_launch_count(self._h))


def fcg_slab_shape_of(L: int, dtype, nranks: int, rank: int) -> dict:
    """Pure host arithmetic in libfcg (no device needed): how an L x L lattice of this dtype splits over nranks."""
    sh = SlabShape()
    st = lib().fcg_slab_shape_of(int(L), _dt(dtype), int(nranks), int(rank), C.byref(sh))
    if st != FCG_OK:
        raise FcgError(st, f"slab decomposition of L={L} over {nranks} ranks is not supported")
    return {name: getattr(sh, name) for name, _ in SlabShape._fields_}


FCG_BREAK_STATIC_MAX_N = 8192 * 8192


def fcg_break_step_static(k: torch.Tensor, u: torch.Tensor, t: torch.Tensor, result: torch.Tensor, stream: torch.cuda.Stream | None = None):
    """The allocation-free break step (include/fcg.h): enqueues on `stream` (default: the current one) and returns at once.
    k (in/out), u, t: contiguous CUDA tensors of one dtype and size; result: caller-owned CUDA tensor of 3 int64 that receives
    the fcg_break_result block (read it with break_result())."""
    if not (k.is_cuda and u.is_cuda and t.is_cuda and result.is_cuda and k.is_contiguous() and u.is_contiguous() and t.is_contiguous()):
        raise ValueError("expected contiguous CUDA tensors")
    if not (k.dtype == u.dtype == t.dtype and k.numel() == u.numel() == t.numel()):
        raise ValueError("k, u, t must agree in dtype and size")
    if result.dtype != torch.int64 or result.numel() < 3 or not result.is_contiguous():
        raise ValueError("result must be a contiguous int64 tensor of >= 3 elements")
    st = stream or torch.cuda.current_stream(k.device)
    rc = lib().fcg_break_step_static(_dt(k.dtype), k.numel(), k.data_ptr(), u.data_ptr(), t.data_ptr(), result.data_ptr(), st.cuda_stream)
    if rc != FCG_OK:
        raise FcgError(rc, lib().fcg_static_last_error().decode())


def break_result(result: torch.Tensor):
    """(index, ratio, status) from the block fcg_break_step_static filled; synchronises (a device-to-host read)."""
    r = result[:3].cpu()
    return int(r[0]), float(r[1:2].view(torch.float64)[0]), int(r[2:3].view(torch.int32)[0])


def fcg_version() -> str:
    return lib().fcg_version().decode()
