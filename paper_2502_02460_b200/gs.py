"""Thin ctypes binding of the C ABI in include/gs.h (same names, argument marshalling only).

PyTorch is used for device memory and streams; every step of the path runs in the CUDA kernels of
libgs.so.  Loading fails loudly if the library has not been built -- there is no fallback.

    plan = gs.Plan(N, nev=nev)                 # gs_plan_create + workspace from torch
    plan.cholesky(S)                           # in place, S column-major torch tensor on the GPU
    plan.invert_triangular(U, Uinv)
    plan.to_standard(H, Uinv, Htilde)
    plan.backtransform(Uinv, Ctilde, C)
    plan.last_info()                           # synchronises; raises GsError on numerical failure
"""
from __future__ import annotations

import ctypes
import os

import torch

from .workloads import is_colmajor

GS_REAL64, GS_COMPLEX128 = 0, 1
GS_PUSH_UINV, GS_PUSH_G, GS_PUSH_HTILDE, GS_PUSH_C = 0, 1, 2, 3
GS_OK = 0
STATUS_NAMES = {
    0: "GS_OK", 1: "GS_ERR_INVALID_ARG", 2: "GS_ERR_NOT_POSDEF", 3: "GS_ERR_SINGULAR",
    4: "GS_ERR_CUDA", 5: "GS_ERR_WORKSPACE", 6: "GS_ERR_UNSUPPORTED_DEVICE", 7: "GS_ERR_NO_CONVERGENCE",
}
EXPORTS = (
    "gs_plan_create", "gs_plan_destroy", "gs_plan_workspace_bytes", "gs_plan_set_workspace",
    "gs_cholesky", "gs_cholesky_leading", "gs_cholesky_sharded", "gs_cholesky_sharded_epochs", "gs_invert_triangular", "gs_to_standard", "gs_backtransform", "gs_density_matrix", "gs_density_matrix_static", "gs_last_info", "gs_plan_clear_info",
    "gs_invert_triangular_cols", "gs_to_standard_g_cols", "gs_to_standard_cols", "gs_backtransform_cols",
    "gs_plan_set_push_targets", "gs_ipc_export", "gs_ipc_open", "gs_ipc_close", "gs_exchange_signal", "gs_exchange_wait",
    "gs_reduce_host_scratch_bytes", "gs_reduce_host_h2d_bytes", "gs_reduce_host_d2h_bytes", "gs_reduce_host", "gs_backtransform_host",
    "gs_plan_launch_count", "gs_status_string", "gs_plan_last_cuda_error",
    "gs_plan_set_timing", "gs_plan_launch_times", "gs_plan_launch_trace",
    "gs_evp_workspace_bytes", "gs_evp_set_workspace", "gs_evp_tridiagonalize", "gs_evp_tridiag_solve", "gs_evp_backtransform",
    "gs_standard_eigh", "gs_generalized_eigh", "gs_evp_tridiag_eigenvalues", "gs_standard_eigenvalues", "gs_truncated_workspace_bytes", "gs_truncated_to_standard", "gs_truncated_rank", "gs_backtransform_dense",
)


class LaunchTime(ctypes.Structure):
    _fields_ = [("label", ctypes.c_char * 32), ("launches", ctypes.c_int64), ("ms", ctypes.c_double)]

class LaunchTrace(ctypes.Structure):
    _fields_ = [("label", ctypes.c_char * 32), ("side_stream", ctypes.c_int32),
                ("t0_ms", ctypes.c_double), ("t1_ms", ctypes.c_double)]


_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgs.so")
PEAK_LIB_PATH = os.path.join(_HERE, "libgs_peak.so")
_lib = None
_peak = None


class GsError(RuntimeError):
    def __init__(self, status: int, info: int = 0, detail: str = ""):
        self.status = status
        self.info = info
        name = STATUS_NAMES.get(status, f"status {status}")
        super().__init__(f"{name}" + (f" (info={info})" if info else "") + (f": {detail}" if detail else ""))


def lib() -> ctypes.CDLL:
    """Load libgs.so.  Raises (never falls back) if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} not found: build it with `python -m paper_2502_02460_b200.build` "
                "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_size_t
        L.gs_plan_create.argtypes = [ctypes.POINTER(vp), i64, ctypes.c_int, i64]
        L.gs_plan_destroy.argtypes = [vp]
        L.gs_plan_workspace_bytes.argtypes = [vp, ctypes.POINTER(sz)]
        L.gs_plan_set_workspace.argtypes = [vp, vp, sz]
        L.gs_cholesky.argtypes = [vp, vp, vp]
        L.gs_cholesky_leading.argtypes = [vp, vp, i64, vp]
        L.gs_invert_triangular.argtypes = [vp, vp, vp, vp]
        L.gs_cholesky_sharded.argtypes = [vp, vp, ctypes.c_int, ctypes.c_int, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.c_uint32, vp]
        L.gs_cholesky_sharded_epochs.argtypes = [vp, ctypes.POINTER(ctypes.c_uint32)]
        L.gs_to_standard.argtypes = [vp, vp, vp, vp, vp]
        L.gs_backtransform.argtypes = [vp, vp, vp, vp, vp]
        L.gs_density_matrix.argtypes = [vp, vp, vp, vp, vp]
        L.gs_density_matrix_static.argtypes = [vp, vp, vp, vp, vp]
        L.gs_invert_triangular_cols.argtypes = [vp, vp, vp, i64, i64, vp]
        L.gs_to_standard_g_cols.argtypes = [vp, vp, vp, vp, i64, i64, vp]
        L.gs_to_standard_cols.argtypes = [vp, vp, vp, vp, i64, i64, vp]
        L.gs_backtransform_cols.argtypes = [vp, vp, vp, vp, i64, i64, vp]
        L.gs_last_info.argtypes = [vp, vp, ctypes.POINTER(i64)]
        L.gs_plan_clear_info.argtypes = [vp, vp]
        L.gs_plan_set_push_targets.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.POINTER(vp)]
        L.gs_exchange_signal.argtypes = [vp, ctypes.c_int, ctypes.POINTER(vp), ctypes.c_uint32, vp]
        L.gs_exchange_wait.argtypes = [vp, ctypes.c_int, ctypes.POINTER(vp), ctypes.c_uint32, vp]
        L.gs_ipc_export.argtypes = [vp, ctypes.c_char_p, ctypes.POINTER(ctypes.c_uint64)]
        L.gs_ipc_open.argtypes = [ctypes.c_char_p, ctypes.c_uint64, ctypes.POINTER(vp)]
        L.gs_ipc_close.argtypes = [vp, ctypes.c_uint64]
        L.gs_reduce_host_scratch_bytes.argtypes = [vp, ctypes.POINTER(sz)]
        L.gs_reduce_host_h2d_bytes.argtypes = [vp, ctypes.POINTER(sz)]
        L.gs_reduce_host_d2h_bytes.argtypes = [vp, ctypes.POINTER(sz)]
        L.gs_reduce_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, sz, vp]
        L.gs_backtransform_host.argtypes = [vp, vp, vp, vp, sz, vp]
        L.gs_plan_set_timing.argtypes = [vp, ctypes.c_int]
        L.gs_plan_launch_times.argtypes = [vp, ctypes.POINTER(LaunchTime), ctypes.c_int, ctypes.POINTER(ctypes.c_int)]
        L.gs_plan_launch_trace.argtypes = [vp, ctypes.POINTER(LaunchTrace), ctypes.c_int, ctypes.POINTER(ctypes.c_int)]
        L.gs_plan_launch_count.argtypes = [vp, ctypes.POINTER(i64)]
        L.gs_evp_workspace_bytes.argtypes = [vp, ctypes.POINTER(sz)]
        L.gs_evp_set_workspace.argtypes = [vp, vp, sz]
        L.gs_evp_tridiagonalize.argtypes = [vp, vp, vp, vp, vp, vp]
        L.gs_evp_tridiag_solve.argtypes = [vp, vp, vp, vp, vp, vp]
        L.gs_evp_backtransform.argtypes = [vp, vp, vp, vp, vp]
        L.gs_standard_eigh.argtypes = [vp, vp, vp, vp, vp]
        L.gs_generalized_eigh.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.gs_evp_tridiag_eigenvalues.argtypes = [vp, vp, vp, i64, vp, vp]
        L.gs_standard_eigenvalues.argtypes = [vp, vp, i64, vp, vp]
        L.gs_truncated_workspace_bytes.argtypes = [vp, ctypes.POINTER(sz)]
        L.gs_truncated_to_standard.argtypes = [vp, vp, vp, ctypes.c_double, vp, vp, vp, vp]
        L.gs_truncated_rank.argtypes = [vp, vp, ctypes.POINTER(i64)]
        L.gs_backtransform_dense.argtypes = [vp, vp, vp, vp, vp]
        L.gs_status_string.argtypes = [ctypes.c_int]
        L.gs_status_string.restype = ctypes.c_char_p
        L.gs_plan_last_cuda_error.argtypes = [vp]
        L.gs_plan_last_cuda_error.restype = ctypes.c_char_p
        for name in EXPORTS:
            if name not in ("gs_status_string", "gs_plan_last_cuda_error"):
                getattr(L, name).restype = ctypes.c_int
        _lib = L
    return _lib


def peak_lib() -> ctypes.CDLL:
    global _peak
    if _peak is None:
        if not os.path.exists(PEAK_LIB_PATH):
            raise FileNotFoundError(f"{PEAK_LIB_PATH} not found: run `python -m paper_2502_02460_b200.build`")
        L = ctypes.CDLL(PEAK_LIB_PATH)
        L.gs_peak_fp64.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.POINTER(ctypes.c_double)]
        L.gs_peak_fp64.restype = ctypes.c_double
        _peak = L
    return _peak


def measure_fp64_peak(kind: int = 0, seconds: float = 1.0):
    """(sustained TFLOP/s, burst TFLOP/s) of the FP64 tensor pipe (kind 0, DMMA) or DFMA (kind 1)."""
    burst = ctypes.c_double(0.0)
    sus = peak_lib().gs_peak_fp64(kind, seconds, ctypes.byref(burst))
    if sus < 0:
        raise RuntimeError("FP64 peak microbenchmark failed (CUDA error)")
    return float(sus), float(burst.value)


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _dev_ptr(t: torch.Tensor, rows: int, cols: int, dtype) -> int:
    if not t.is_cuda:
        raise ValueError("expected a CUDA tensor")
    if t.dtype != dtype or tuple(t.shape) != (rows, cols) or not is_colmajor(t):
        raise ValueError(f"expected column-major {dtype} tensor of shape ({rows}, {cols}), got "
                         f"{t.dtype} {tuple(t.shape)} strides {t.stride()}")
    return t.data_ptr()


class Plan:
    """gs_plan_t plus its torch-owned workspace."""

    def __init__(self, N: int, nev: int | None = None, dtype: int = GS_REAL64, device=None):
        self.N = int(N)
        self.nev = self.N if nev is None else int(nev)
        self.dtype = dtype
        self.tdtype = torch.float64 if dtype == GS_REAL64 else torch.complex128
        self._h = ctypes.c_void_p()
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        L = lib()
        with torch.cuda.device(self.device):
            self._check(L.gs_plan_create(ctypes.byref(self._h), self.N, dtype, self.nev))
            n = ctypes.c_size_t(0)
            self._check(L.gs_plan_workspace_bytes(self._h, ctypes.byref(n)))
            self.workspace = torch.empty(n.value, dtype=torch.uint8, device=self.device)
            self._check(L.gs_plan_set_workspace(self._h, self.workspace.data_ptr(), n.value))

    def _check(self, status: int, info: int = 0):
        if status != GS_OK:
            detail = ""
            if self._h:
                detail = lib().gs_plan_last_cuda_error(self._h).decode()
            raise GsError(status, info, detail)

    def close(self):
        if self._h:
            lib().gs_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the four steps of PAPER.md:61-67 ----
    def cholesky(self, S: torch.Tensor, stream=None):
        self._check(lib().gs_cholesky(self._h, _dev_ptr(S, self.N, self.N, self.tdtype), _stream_ptr(stream)))

    def cholesky_leading(self, S: torch.Tensor, ncols: int, stream=None):
        """Step 1 on the leading ncols x ncols block only (sharded path)."""
        self._check(lib().gs_cholesky_leading(self._h, _dev_ptr(S, self.N, self.N, self.tdtype), ncols, _stream_ptr(stream)))

    def cholesky_sharded_epochs(self) -> int:
        n = ctypes.c_uint32(0)
        self._check(lib().gs_cholesky_sharded_epochs(self._h, ctypes.byref(n)))
        return int(n.value)

    def cholesky_sharded(self, S: torch.Tensor, rank: int, nranks: int, peer_S=None, peer_workspace=None, flags=None, epoch0: int = 0, stream=None):
        """Step 1 over `nranks` GPUs (gs_cholesky_sharded): peer_S / peer_workspace / flags are lists of nranks device
        addresses (ints) as mapped in this process; entry `rank` = S.data_ptr() / self.workspace.data_ptr() / the local flags."""
        def arr(v):
            return None if v is None else (ctypes.c_void_p * nranks)(*[int(x) for x in v])
        self._check(lib().gs_cholesky_sharded(self._h, _dev_ptr(S, self.N, self.N, self.tdtype), rank, nranks, arr(peer_S), arr(peer_workspace),
                                              arr(flags), epoch0 & 0xFFFFFFFF, _stream_ptr(stream)))

    def invert_triangular(self, U: torch.Tensor, Uinv: torch.Tensor, stream=None):
        self._check(lib().gs_invert_triangular(self._h, _dev_ptr(U, self.N, self.N, self.tdtype),
                                               _dev_ptr(Uinv, self.N, self.N, self.tdtype), _stream_ptr(stream)))

    def to_standard(self, H: torch.Tensor, Uinv: torch.Tensor, Htilde: torch.Tensor, stream=None):
        self._check(lib().gs_to_standard(self._h, _dev_ptr(H, self.N, self.N, self.tdtype),
                                         _dev_ptr(Uinv, self.N, self.N, self.tdtype),
                                         _dev_ptr(Htilde, self.N, self.N, self.tdtype), _stream_ptr(stream)))

    def backtransform(self, Uinv: torch.Tensor, Ctilde: torch.Tensor, C: torch.Tensor, stream=None):
        if self.nev == 0:
            self._check(lib().gs_backtransform(self._h, None, None, None, _stream_ptr(stream)))
            return
        self._check(lib().gs_backtransform(self._h, _dev_ptr(Uinv, self.N, self.N, self.tdtype),
                                           _dev_ptr(Ctilde, self.N, self.nev, self.tdtype),
                                           _dev_ptr(C, self.N, self.nev, self.tdtype), _stream_ptr(stream)))

    # ---- column-range forms (sharded path, sharded.py) ----
    @property
    def block(self) -> int:
        """Block order the column ranges are aligned to: 128 (real) or 64 (complex)."""
        return 128 if self.dtype == GS_REAL64 else 64

    def invert_triangular_cols(self, U: torch.Tensor, Uinv: torch.Tensor, col0: int, ncols: int, stream=None):
        self._check(lib().gs_invert_triangular_cols(self._h, _dev_ptr(U, self.N, self.N, self.tdtype),
                                                    _dev_ptr(Uinv, self.N, self.N, self.tdtype), col0, ncols,
                                                    _stream_ptr(stream)))

    def to_standard_g_cols(self, H: torch.Tensor, Uinv: torch.Tensor, G: torch.Tensor, col0: int, ncols: int, stream=None):
        self._check(lib().gs_to_standard_g_cols(self._h, _dev_ptr(H, self.N, self.N, self.tdtype),
                                                _dev_ptr(Uinv, self.N, self.N, self.tdtype),
                                                _dev_ptr(G, self.N, self.N, self.tdtype), col0, ncols, _stream_ptr(stream)))

    def to_standard_cols(self, Uinv: torch.Tensor, G: torch.Tensor, Htilde: torch.Tensor, col0: int, ncols: int, stream=None):
        self._check(lib().gs_to_standard_cols(self._h, _dev_ptr(Uinv, self.N, self.N, self.tdtype),
                                              _dev_ptr(G, self.N, self.N, self.tdtype),
                                              _dev_ptr(Htilde, self.N, self.N, self.tdtype), col0, ncols, _stream_ptr(stream)))

    def backtransform_cols(self, Uinv: torch.Tensor, Ctilde: torch.Tensor, C: torch.Tensor, col0: int, ncols: int, stream=None):
        self._check(lib().gs_backtransform_cols(self._h, _dev_ptr(Uinv, self.N, self.N, self.tdtype),
                                                _dev_ptr(Ctilde, self.N, self.nev, self.tdtype),
                                                _dev_ptr(C, self.N, self.nev, self.tdtype), col0, ncols, _stream_ptr(stream)))

    def set_push_targets(self, kind: int, ptrs):
        """Fused exchange: device pointers (ints) the column-range call of `kind` also stores into."""
        arr = (ctypes.c_void_p * max(1, len(ptrs)))(*ptrs)
        self._check(lib().gs_plan_set_push_targets(self._h, kind, len(ptrs), arr))

    def exchange_signal(self, flag_ptrs, value: int, stream=None):
        """Behind everything enqueued on the stream: write `value` to every flag address (device-side ordering)."""
        arr = (ctypes.c_void_p * max(1, len(flag_ptrs)))(*flag_ptrs)
        self._check(lib().gs_exchange_signal(self._h, len(flag_ptrs), arr, value & 0xFFFFFFFF, _stream_ptr(stream)))

    def exchange_wait(self, flag_ptrs, value: int, stream=None):
        """The stream continues only when every (local) flag is >= value."""
        arr = (ctypes.c_void_p * max(1, len(flag_ptrs)))(*flag_ptrs)
        self._check(lib().gs_exchange_wait(self._h, len(flag_ptrs), arr, value & 0xFFFFFFFF, _stream_ptr(stream)))

    def density_matrix(self, C: torch.Tensor, f: torch.Tensor, P: torch.Tensor, stream=None):
        """P(i,j) = sum_l f[l] conj(C(i,l)) C(j,l); upper triangle of P is written."""
        if self.nev == 0:
            self._check(lib().gs_density_matrix(self._h, None, None, _dev_ptr(P, self.N, self.N, self.tdtype), _stream_ptr(stream)))
            return
        if not (f.is_cuda and f.dtype == torch.float64 and f.dim() == 1 and f.numel() == self.nev and f.is_contiguous()):
            raise ValueError("f: expected a contiguous CUDA float64 vector of length nev")
        self._check(lib().gs_density_matrix(self._h, _dev_ptr(C, self.N, self.nev, self.tdtype), f.data_ptr(),
                                            _dev_ptr(P, self.N, self.N, self.tdtype), _stream_ptr(stream)))

    def density_matrix_static(self, C: torch.Tensor, f: torch.Tensor, P: torch.Tensor, stream=None):
        """gs_density_matrix_static: the same result with the scratch in libgs's static device array -- no allocation,
        no plan workspace; N * nev is limited (GS_STATIC_SCRATCH_BYTES) and overlapping calls race (include/gs.h)."""
        if self.nev == 0:
            self._check(lib().gs_density_matrix_static(self._h, None, None, _dev_ptr(P, self.N, self.N, self.tdtype), _stream_ptr(stream)))
            return
        if not (f.is_cuda and f.dtype == torch.float64 and f.dim() == 1 and f.numel() == self.nev and f.is_contiguous()):
            raise ValueError("f: expected a contiguous CUDA float64 vector of length nev")
        self._check(lib().gs_density_matrix_static(self._h, _dev_ptr(C, self.N, self.nev, self.tdtype), f.data_ptr(),
                                                   _dev_ptr(P, self.N, self.N, self.tdtype), _stream_ptr(stream)))

    # ---- NEXT-4: the standard eigenproblem H~ C~ = C~ eps between step 3 and the back-transformation ----
    def evp_workspace_bytes(self) -> int:
        n = ctypes.c_size_t(0)
        self._check(lib().gs_evp_workspace_bytes(self._h, ctypes.byref(n)))
        return int(n.value)

    def ensure_evp_workspace(self, alloc=None, truncated: bool = False):
        """Allocates (once) and registers the eigensolver's scratch; `alloc(nbytes)` may supply the uint8 buffer.
        truncated=True sizes it for the truncated-basis route (all N eigenvectors of S)."""
        n = self.evp_workspace_bytes()
        if truncated:
            nt = ctypes.c_size_t(0)
            self._check(lib().gs_truncated_workspace_bytes(self._h, ctypes.byref(nt)))
            n = max(n, int(nt.value))
        if getattr(self, "evp_workspace", None) is None or self.evp_workspace.numel() < n:
            self.evp_workspace = alloc(n) if alloc is not None else torch.empty(n, dtype=torch.uint8, device=self.device)
            self._check(lib().gs_evp_set_workspace(self._h, self.evp_workspace.data_ptr(), n))

    def _vec(self, n: int, dtype=torch.float64) -> torch.Tensor:
        return torch.empty(n, dtype=dtype, device=self.device)

    def evp_tridiagonalize(self, A: torch.Tensor, stream=None):
        """"Tridiag.": A (upper triangle = H~) -> Householder vectors in A, returns (d, e, tau)."""
        self.ensure_evp_workspace()
        d, e, tau = self._vec(self.N), self._vec(self.N), self._vec(self.N, self.tdtype)
        self._check(lib().gs_evp_tridiagonalize(self._h, _dev_ptr(A, self.N, self.N, self.tdtype), d.data_ptr(), e.data_ptr(),
                                                tau.data_ptr(), _stream_ptr(stream)))
        return d, e[:max(self.N - 1, 0)], tau

    def evp_tridiag_solve(self, d: torch.Tensor, e: torch.Tensor, stream=None):
        """"Solve": lowest nev eigenvalues of tridiag(e, d, e) and their eigenvectors Z (N x nev, real)."""
        from .workloads import colmajor_empty
        self.ensure_evp_workspace()
        ebuf = self._vec(self.N)
        ebuf[:e.numel()].copy_(e)
        eps = self._vec(max(self.nev, 1))[:self.nev]
        Z = colmajor_empty(self.N, max(self.nev, 1), device=self.device)[:, :self.nev]
        self._check(lib().gs_evp_tridiag_solve(self._h, d.contiguous().data_ptr(), ebuf.data_ptr(), eps.data_ptr(), Z.data_ptr(),
                                               _stream_ptr(stream)))
        return eps, Z

    def evp_backtransform(self, A: torch.Tensor, Z: torch.Tensor, out: torch.Tensor | None = None, stream=None) -> torch.Tensor:
        """"Back": C~ = Q Z with the reflectors evp_tridiagonalize left in A."""
        from .workloads import colmajor_empty
        self.ensure_evp_workspace()
        Ct = colmajor_empty(self.N, max(self.nev, 1), dtype=self.tdtype, device=self.device)[:, :self.nev] if out is None else out
        if self.nev > 0:
            self._check(lib().gs_evp_backtransform(self._h, _dev_ptr(A, self.N, self.N, self.tdtype),
                                                   _dev_ptr(Z, self.N, self.nev, torch.float64),
                                                   _dev_ptr(Ct, self.N, self.nev, self.tdtype), _stream_ptr(stream)))
        return Ct

    def standard_eigh(self, Htilde: torch.Tensor, eps: torch.Tensor | None = None, out: torch.Tensor | None = None,
                      workspace_alloc=None, stream=None):
        """The three stages in a row on the upper triangle of Htilde (DESTROYED): returns (eps, C~), lowest nev pairs."""
        from .workloads import colmajor_empty
        self.ensure_evp_workspace(workspace_alloc)
        if eps is None:
            eps = self._vec(max(self.nev, 1))[:self.nev]
        Ct = colmajor_empty(self.N, max(self.nev, 1), dtype=self.tdtype, device=self.device)[:, :self.nev] if out is None else out
        self._check(lib().gs_standard_eigh(self._h, _dev_ptr(Htilde, self.N, self.N, self.tdtype), eps.data_ptr(),
                                           _dev_ptr(Ct, self.N, self.nev, self.tdtype) if self.nev > 0 else None,
                                           _stream_ptr(stream)))
        return eps, Ct

    def evp_tridiag_eigenvalues(self, d: torch.Tensor, e: torch.Tensor, count: int | None = None, stream=None) -> torch.Tensor:
        """The `count` (default N) smallest eigenvalues of tridiag(e, d, e) by bisection (gs_evp_tridiag_eigenvalues)."""
        count = self.N if count is None else int(count)
        ebuf = self._vec(max(self.N, 1))
        ebuf[:e.numel()].copy_(e)
        eps = self._vec(max(count, 1))[:count]
        self._check(lib().gs_evp_tridiag_eigenvalues(self._h, d.data_ptr(), ebuf.data_ptr(), count, eps.data_ptr() if count > 0 else None,
                                                     _stream_ptr(stream)))
        return eps

    def standard_eigenvalues(self, Htilde: torch.Tensor, count: int | None = None, stream=None) -> torch.Tensor:
        """The `count` (default N) smallest eigenvalues of the Hermitian matrix in the upper triangle of Htilde (DESTROYED)."""
        self.ensure_evp_workspace()
        count = self.N if count is None else int(count)
        eps = self._vec(max(count, 1))[:count]
        self._check(lib().gs_standard_eigenvalues(self._h, _dev_ptr(Htilde, self.N, self.N, self.tdtype), count,
                                                  eps.data_ptr() if count > 0 else None, _stream_ptr(stream)))
        return eps

    def generalized_eigh(self, H: torch.Tensor, S: torch.Tensor, stream=None):
        """gs_generalized_eigh: the whole solve H C = eps S C in one call.  S is not modified (a copy is
        factored).  Returns (eps, C, U, Uinv): the lowest nev eigenvalues, their eigenvectors, the factor and its inverse."""
        from .workloads import colmajor_empty, colmajor_zeros
        self.ensure_evp_workspace()
        N, nev, dt = self.N, self.nev, self.tdtype
        U = colmajor_empty(N, N, dtype=dt, device=self.device)
        U.copy_(S)
        Uinv = colmajor_empty(N, N, dtype=dt, device=self.device)
        Ht = colmajor_zeros(N, N, dtype=dt, device=self.device)
        Ct = colmajor_empty(N, max(nev, 1), dtype=dt, device=self.device)[:, :nev]
        C = colmajor_empty(N, max(nev, 1), dtype=dt, device=self.device)[:, :nev]
        eps = self._vec(max(nev, 1))[:nev]
        self._check(lib().gs_generalized_eigh(self._h, _dev_ptr(H, N, N, dt), _dev_ptr(U, N, N, dt), _dev_ptr(Uinv, N, N, dt), _dev_ptr(Ht, N, N, dt),
                                              Ct.data_ptr() if nev > 0 else None, eps.data_ptr() if nev > 0 else None,
                                              C.data_ptr() if nev > 0 else None, _stream_ptr(stream)))
        return eps, C, U, Uinv

    # ---- (5) ill-conditioned S: the truncated-basis route of PAPER.md:73 ----
    def truncated_to_standard(self, H: torch.Tensor, S: torch.Tensor, delta: float, stream=None):
        """S (upper triangle) is DESTROYED.  Returns (X, Hr, sigma): then standard_eigh(Hr) and backtransform_dense(X, C~)."""
        from .workloads import colmajor_empty, colmajor_zeros
        self.ensure_evp_workspace(truncated=True)
        X = colmajor_empty(self.N, self.N, dtype=self.tdtype, device=self.device)
        Hr = colmajor_zeros(self.N, self.N, dtype=self.tdtype, device=self.device)
        sigma = self._vec(self.N)
        self._check(lib().gs_truncated_to_standard(self._h, _dev_ptr(H, self.N, self.N, self.tdtype), _dev_ptr(S, self.N, self.N, self.tdtype),
                                                   float(delta), X.data_ptr(), Hr.data_ptr(), sigma.data_ptr(), _stream_ptr(stream)))
        return X, Hr, sigma

    def truncated_rank(self, stream=None) -> int:
        n = ctypes.c_int64(0)
        self._check(lib().gs_truncated_rank(self._h, _stream_ptr(stream), ctypes.byref(n)))
        return int(n.value)

    def backtransform_dense(self, X: torch.Tensor, Ctilde: torch.Tensor, C: torch.Tensor, stream=None):
        if self.nev == 0:
            return
        self._check(lib().gs_backtransform_dense(self._h, _dev_ptr(X, self.N, self.N, self.tdtype),
                                                 _dev_ptr(Ctilde, self.N, self.nev, self.tdtype),
                                                 _dev_ptr(C, self.N, self.nev, self.tdtype), _stream_ptr(stream)))

    def last_info(self, stream=None, raise_on_failure: bool = True) -> int:
        info = ctypes.c_int64(0)
        status = lib().gs_last_info(self._h, _stream_ptr(stream), ctypes.byref(info))
        self.last_status = int(status)     # which failure `info` belongs to (NOT_POSDEF / SINGULAR)
        if status != GS_OK and raise_on_failure:
            self._check(status, int(info.value))
        return int(info.value)

    def clear_info(self, stream=None):
        """Clears the numerical-failure flag (gs_cholesky does so itself when it starts)."""
        self._check(lib().gs_plan_clear_info(self._h, _stream_ptr(stream)))

    def launch_count(self) -> int:
        n = ctypes.c_int64(0)
        self._check(lib().gs_plan_launch_count(self._h, ctypes.byref(n)))
        return int(n.value)

    # ---- host-buffer entry points (end-to-end measurement) ----
    def host_scratch_bytes(self) -> int:
        n = ctypes.c_size_t(0)
        self._check(lib().gs_reduce_host_scratch_bytes(self._h, ctypes.byref(n)))
        return int(n.value)

    def reduce_host_h2d_bytes(self) -> int:
        n = ctypes.c_size_t(0)
        self._check(lib().gs_reduce_host_h2d_bytes(self._h, ctypes.byref(n)))
        return int(n.value)

    def reduce_host_d2h_bytes(self) -> int:
        n = ctypes.c_size_t(0)
        self._check(lib().gs_reduce_host_d2h_bytes(self._h, ctypes.byref(n)))
        return int(n.value)

    def reduce_host(self, H: torch.Tensor, S: torch.Tensor, U, Uinv, Htilde, scratch: torch.Tensor, stream=None):
        """H, S (and the optional outputs) are pinned HOST tensors, column-major."""
        def hp(t):
            return None if t is None else t.data_ptr()
        self._check(lib().gs_reduce_host(self._h, hp(H), hp(S), hp(U), hp(Uinv), hp(Htilde), scratch.data_ptr(),
                                         scratch.numel() * scratch.element_size(), _stream_ptr(stream)))

    def backtransform_host(self, Ctilde, C, scratch: torch.Tensor, stream=None):
        """Uses the U^-1 that reduce_host left in `scratch`."""
        self._check(lib().gs_backtransform_host(self._h, Ctilde.data_ptr(), C.data_ptr(),
                                                scratch.data_ptr(), scratch.numel() * scratch.element_size(),
                                                _stream_ptr(stream)))

    # ---- optional per-launch timing (roofline reports) ----
    def set_timing(self, mode: int):
        self._check(lib().gs_plan_set_timing(self._h, mode))

    def launch_trace(self, cap: int = 8192) -> list:
        """[(label, side_stream, t0_ms, t1_ms)] per launch since set_timing(1); call before launch_times()."""
        buf = (LaunchTrace * cap)()
        n = ctypes.c_int(0)
        self._check(lib().gs_plan_launch_trace(self._h, buf, cap, ctypes.byref(n)))
        return [(buf[i].label.decode(), int(buf[i].side_stream), float(buf[i].t0_ms), float(buf[i].t1_ms))
                for i in range(min(n.value, cap))]

    def launch_times(self) -> dict:
        """{label: (launches, total_ms)} since the last set_timing; call after a stream synchronise."""
        buf = (LaunchTime * 32)()
        n = ctypes.c_int(0)
        self._check(lib().gs_plan_launch_times(self._h, buf, 32, ctypes.byref(n)))
        return {buf[i].label.decode(): (int(buf[i].launches), float(buf[i].ms)) for i in range(min(n.value, 32))}


def ipc_export(t: torch.Tensor):
    """(64-byte handle, byte offset) of the device allocation behind a CUDA tensor, for another process."""
    buf = ctypes.create_string_buffer(64)
    off = ctypes.c_uint64(0)
    st = lib().gs_ipc_export(t.data_ptr(), buf, ctypes.byref(off))
    if st != GS_OK:
        raise GsError(st, 0, "gs_ipc_export")
    return bytes(buf.raw), int(off.value)


def ipc_open(handle: bytes, offset: int) -> int:
    """Maps a peer's allocation into this process; returns the device pointer of the peer's tensor."""
    ptr = ctypes.c_void_p()
    st = lib().gs_ipc_open(handle, offset, ctypes.byref(ptr))
    if st != GS_OK:
        raise GsError(st, 0, "gs_ipc_open")
    return int(ptr.value)


def ipc_close(ptr: int, offset: int) -> None:
    lib().gs_ipc_close(ptr, offset)


def generalized_to_standard(H: torch.Tensor, S: torch.Tensor, nev: int | None = None):
    """Convenience: run steps 1-3 on fresh buffers.  Returns (plan, U, Uinv, Htilde); S is not modified."""
    from .workloads import colmajor_empty, colmajor_zeros
    N = H.shape[0]
    cplx = H.dtype == torch.complex128
    plan = Plan(N, nev, dtype=GS_COMPLEX128 if cplx else GS_REAL64)
    U = colmajor_empty(N, N, dtype=H.dtype, device=H.device)
    U.copy_(S)
    Uinv = colmajor_empty(N, N, dtype=H.dtype, device=H.device)
    Ht = colmajor_zeros(N, N, dtype=H.dtype, device=H.device)
    plan.cholesky(U)
    plan.invert_triangular(U, Uinv)
    plan.to_standard(H, Uinv, Ht)
    plan.last_info()
    return plan, U, Uinv, Ht
