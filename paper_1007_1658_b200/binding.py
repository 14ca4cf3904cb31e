"""Thin ctypes binding over the C ABI of include/lsp.h -- argument marshalling only.

Every step of the hot path runs in the CUDA library (csrc/); PyTorch is used here only for
device memory and streams.  There is NO CPU fallback: if the shared library is missing and
cannot be built, or no sm_100 device is present, the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

from . import build as _build

LSP_OK, LSP_EINVAL, LSP_ECUDA, LSP_ENOMEM, LSP_ELIMIT = 0, -1, -2, -3, -4
STATIC_SCRATCH_BYTES, STATIC_MAX_NT, STATIC_MAX_NF = 8 << 20, 16384, 262144
PARAM_K, PARAM_THREADS, PARAM_NSPLIT, PARAM_PIPE, PARAM_FLUSH, PARAM_TIMING, PARAM_TABLE_MB, PARAM_COARSE, PARAM_TRUNC, PARAM_SHARED, PARAM_PDL, PARAM_CORR, PARAM_REFINE, PARAM_ORDER = 1, 2, 3, 4, 5, 6, 7, 8, 9, 11, 13, 15, 16, 17
PIPE_AUTO, PIPE_FP32, PIPE_TENSOR = 0, 1, 2

# every symbol include/lsp.h declares (checked by tests/test_abi.py against the header text)
SYMBOLS = (
    "lsp_create", "lsp_destroy", "lsp_set_param", "lsp_get_param",
    "lsp_periodogram", "lsp_periodogram_batched",
    "lsp_periodogram_host", "lsp_periodogram_batched_host",
    "lsp_false_alarm", "lsp_periodogram_gls", "lsp_periodogram_gls_batched",
    "lsp_periodogram_gls_weighted", "lsp_periodogram_gls_weighted_batched", "lsp_reserve",
    "lsp_last_plan", "lsp_last_timing", "lsp_call_timing", "lsp_plan_query", "lsp_plan_query_form", "lsp_last_kernel_name", "lsp_last_host_chunks", "lsp_probe_mma_accumulate", "lsp_last_cuda_error",
    "lsp_status_string", "lsp_version", "lsp_periodogram_static",
)

_lib = None


class LspError(RuntimeError):
    def __init__(self, status: int, where: str, cuda_error: int = 0):
        self.status = status
        self.cuda_error = cuda_error
        msg = "%s failed: %s (status %d" % (where, status_string(status), status)
        if cuda_error:
            msg += ", cudaError %d" % cuda_error
        super().__init__(msg + ")")


def load(rebuild: bool = False):
    """dlopen paper_1007_1658_b200/liblsp_b200.so, building it with nvcc first if it is absent or older than a source
    (build() is a no-op when the library is fresh, so a stale binary is never loaded silently)."""
    global _lib
    if _lib is not None and not rebuild:
        return _lib
    path = _build.build(force=rebuild)
    lib = ctypes.CDLL(path)
    vp, i64, dbl, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int
    lib.lsp_create.argtypes = [ctypes.POINTER(vp), ci]
    lib.lsp_destroy.argtypes = [vp]
    lib.lsp_set_param.argtypes = [vp, ci, i64]
    lib.lsp_get_param.argtypes = [vp, ci, ctypes.POINTER(i64)]
    lib.lsp_periodogram.argtypes = [vp, vp, vp, i64, dbl, dbl, i64, vp, vp]
    lib.lsp_periodogram_batched.argtypes = [vp, vp, i64, vp, i64, i64, i64, dbl, dbl, i64,
                                            vp, i64, vp, vp, vp]
    lib.lsp_periodogram_host.argtypes = [vp, vp, vp, i64, dbl, dbl, i64, vp, vp]
    lib.lsp_periodogram_batched_host.argtypes = [vp, vp, ci, vp, i64, i64, dbl, dbl, i64,
                                                 vp, vp, vp, vp]
    lib.lsp_periodogram_gls.argtypes = lib.lsp_periodogram.argtypes
    lib.lsp_periodogram_gls_batched.argtypes = lib.lsp_periodogram_batched.argtypes
    lib.lsp_periodogram_gls_weighted.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, i64, vp, vp]
    lib.lsp_periodogram_gls_weighted_batched.argtypes = [vp, vp, i64, vp, i64, vp, i64, i64, i64, dbl, dbl, i64,
                                                         vp, i64, vp, vp, vp]
    lib.lsp_false_alarm.argtypes = [vp, vp, i64, i64, dbl, vp, vp]
    lib.lsp_periodogram_static.argtypes = [vp, vp, i64, dbl, dbl, i64, vp, vp, vp, vp]
    lib.lsp_reserve.argtypes = [vp, i64, ci, i64, i64, ci]
    lib.lsp_last_plan.argtypes = [vp, ctypes.POINTER(i64)]
    lib.lsp_last_timing.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    lib.lsp_call_timing.argtypes = [vp, ci, ctypes.POINTER(ctypes.c_float)]
    lib.lsp_plan_query.argtypes = [ci, i64, i64, i64, ctypes.POINTER(i64)]
    lib.lsp_plan_query_form.argtypes = [ci, i64, i64, i64, ci, ctypes.POINTER(i64)]
    lib.lsp_last_kernel_name.argtypes = [vp]
    lib.lsp_last_kernel_name.restype = ctypes.c_char_p
    lib.lsp_last_host_chunks.argtypes = [vp]
    lib.lsp_probe_mma_accumulate.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    lib.lsp_last_cuda_error.argtypes = [vp]
    lib.lsp_status_string.argtypes = [ci]
    lib.lsp_status_string.restype = ctypes.c_char_p
    lib.lsp_version.argtypes = []
    lib.lsp_version.restype = ctypes.c_char_p
    for name in SYMBOLS:
        fn = getattr(lib, name)
        if fn.restype is ctypes.c_int or fn.restype is None:
            fn.restype = ci
    _lib = lib
    return lib


def status_string(status: int) -> str:
    return load().lsp_status_string(int(status)).decode()


def version() -> str:
    return load().lsp_version().decode()


def _stream_ptr(stream) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def periodogram_static(t, x, f_min: float, df: float, Nf: int, out=None, peak_idx=None, peak_val=None, stream=None):
    """lsp_periodogram_static: one series on the current device with no allocation inside the library (its workspace is a fixed
    8 MiB device array; Nt <= 16,384, Nf <= 262,144, else LspError with status LSP_ELIMIT).  t float64[Nt], x float32[Nt] CUDA
    tensors; `out` float32[Nf] and the optional int32[1] / float32[1] peak tensors are the caller's (pass them to keep this
    call allocation-free on the Python side too).  Returns `out`."""
    import torch
    _want(t, torch.float64, 1, "t"); _want(x, torch.float32, 1, "x")
    if t.shape != x.shape:
        raise ValueError("t and x must have the same length")
    P = out if out is not None else torch.empty(int(Nf), dtype=torch.float32, device=t.device)
    _want(P, torch.float32, 1, "P")
    if P.numel() < Nf:
        raise ValueError("P too small")
    if (peak_idx is None) != (peak_val is None):
        raise ValueError("peak_idx and peak_val go together")
    if peak_idx is not None:
        _want(peak_idx, torch.int32, 1, "peak_idx"); _want(peak_val, torch.float32, 1, "peak_val")
    with torch.cuda.device(t.device):
        st = load().lsp_periodogram_static(t.data_ptr(), x.data_ptr(), t.numel(), float(f_min), float(df), int(Nf), P.data_ptr(),
                                           peak_idx.data_ptr() if peak_idx is not None else None,
                                           peak_val.data_ptr() if peak_val is not None else None, _stream_ptr(stream))
    if st != LSP_OK:
        raise LspError(st, "lsp_periodogram_static")
    return P


def plan_query(sm_count: int, B: int, Nt: int, Nf: int) -> dict:
    """lsp_plan_query: the automatic launch plan for a problem size (host-only, no GPU needed)."""
    out = (ctypes.c_int64 * 8)()
    st = load().lsp_plan_query(int(sm_count), int(B), int(Nt), int(Nf), out)
    if st != LSP_OK:
        raise LspError(st, "lsp_plan_query")
    keys = ("K", "threads", "nsplit", "pipe", "n_freq_blocks", "split_len", "ctas_per_sm", "score_e6")
    return dict(zip(keys, [int(v) for v in out]))


def plan_query_form(sm_count: int, B: int, Nt: int, Nf: int, pipe: int = 0) -> dict:
    """lsp_plan_query_form: the launch plan of one form of steps 3-5 (PIPE_AUTO / PIPE_FP32 / PIPE_TENSOR) and its estimated cycles."""
    out = (ctypes.c_int64 * 8)()
    st = load().lsp_plan_query_form(int(sm_count), int(B), int(Nt), int(Nf), int(pipe), out)
    if st != LSP_OK:
        raise LspError(st, "lsp_plan_query_form")
    keys = ("K", "threads", "nsplit", "pipe", "n_freq_blocks", "split_len", "chunks_or_ctas_per_sm", "est_cycles")
    return dict(zip(keys, [int(v) for v in out]))


class Handle:
    """lsp_handle: owns the device workspace.  One handle serves one stream at a time."""

    def __init__(self, device: int = -1):
        self._lib = load()
        h = ctypes.c_void_p()
        st = self._lib.lsp_create(ctypes.byref(h), int(device))
        if st != LSP_OK:
            raise LspError(st, "lsp_create")
        self._h = h

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None):
            self._lib.lsp_destroy(self._h)
            self._h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st: int, where: str):
        if st != LSP_OK:
            raise LspError(st, where, self._lib.lsp_last_cuda_error(self._h))

    # -- tunables / introspection
    def set_param(self, key: int, value: int):
        self._check(self._lib.lsp_set_param(self._h, int(key), int(value)), "lsp_set_param")

    def get_param(self, key: int) -> int:
        v = ctypes.c_int64()
        self._check(self._lib.lsp_get_param(self._h, int(key), ctypes.byref(v)), "lsp_get_param")
        return v.value

    def reserve(self, B: int, Nt: int, Nf: int, shared_t: bool = False, gls: bool = False):
        """lsp_reserve: size the workspace now, so that the call itself allocates nothing (CUDA-graph capture)."""
        self._check(self._lib.lsp_reserve(self._h, int(B), int(bool(shared_t)), int(Nt), int(Nf), int(bool(gls))), "lsp_reserve")

    def last_plan(self) -> dict:
        out = (ctypes.c_int64 * 8)()
        self._check(self._lib.lsp_last_plan(self._h, out), "lsp_last_plan")
        keys = ("K", "threads", "nsplit", "pipe", "n_freq_blocks", "split_len", "launches",
                "lane_ops_per_term")
        d = dict(zip(keys, [int(v) for v in out]))
        d["kernel"] = self._lib.lsp_last_kernel_name(self._h).decode()
        return d

    def probe_mma_accumulate(self):
        """lsp_probe_mma_accumulate: the accumulator after eight one-element tcgen05.mma sequences (hardware check of DESIGN.md section 8)."""
        out = (ctypes.c_float * 8)()
        self._check(self._lib.lsp_probe_mma_accumulate(self._h, out), "lsp_probe_mma_accumulate")
        return [float(v) for v in out]

    def last_host_chunks(self) -> int:
        """Chunks of series the last host-buffer batched call was pipelined over (1: not pipelined)."""
        return int(self._lib.lsp_last_host_chunks(self._h))

    def last_timing(self) -> dict:
        """Per-kernel milliseconds of the last call (requires set_param(PARAM_TIMING, 1))."""
        out = (ctypes.c_float * 4)()
        self._check(self._lib.lsp_last_timing(self._h, out), "lsp_last_timing")
        return dict(zip(("moments", "records", "accumulate", "finish"), [float(v) for v in out]))

    def call_timing(self, calls_back: int = 0) -> dict:
        """Per-kernel milliseconds of the call `calls_back` timed calls ago (ring of 64)."""
        out = (ctypes.c_float * 4)()
        self._check(self._lib.lsp_call_timing(self._h, int(calls_back), out), "lsp_call_timing")
        return dict(zip(("moments", "records", "accumulate", "finish"), [float(v) for v in out]))

    # -- device-pointer entry points (torch CUDA tensors in, enqueue only)
    def periodogram(self, t, x, f_min: float, df: float, Nf: int, out=None, stream=None, gls: bool = False, weights=None):
        """lsp_periodogram (gls=True: lsp_periodogram_gls; weights float32[Nt]: lsp_periodogram_gls_weighted):
        t float64[Nt], x float32[Nt] CUDA tensors -> P float32[Nf] (CUDA)."""
        import torch
        _want(t, torch.float64, 1, "t"); _want(x, torch.float32, 1, "x")
        if t.shape != x.shape:
            raise ValueError("t and x must have the same length")
        P = out if out is not None else torch.empty(int(Nf), dtype=torch.float32, device=t.device)
        _want(P, torch.float32, 1, "P")
        if P.numel() < Nf:
            raise ValueError("P too small")
        if weights is not None:
            _want(weights, torch.float32, 1, "weights")
            if weights.shape != x.shape:
                raise ValueError("weights and x must have the same length")
            st = self._lib.lsp_periodogram_gls_weighted(self._h, t.data_ptr(), x.data_ptr(), weights.data_ptr(), t.numel(),
                                                        float(f_min), float(df), int(Nf), P.data_ptr(), _stream_ptr(stream))
            self._check(st, "lsp_periodogram_gls_weighted")
            return P
        fn = self._lib.lsp_periodogram_gls if gls else self._lib.lsp_periodogram
        st = fn(self._h, t.data_ptr(), x.data_ptr(), t.numel(),
                float(f_min), float(df), int(Nf), P.data_ptr(), _stream_ptr(stream))
        self._check(st, "lsp_periodogram_gls" if gls else "lsp_periodogram")
        return P

    def periodogram_batched(self, t, x, f_min: float, df: float, Nf: int,
                            want_P: bool = True, want_peaks: bool = True, stream=None, gls: bool = False, weights=None):
        """lsp_periodogram_batched: x float32[B,Nt]; t float64[B,Nt] or float64[Nt] (shared); gls=True: the generalised
        periodogram; weights float32[B,Nt] or float32[Nt] (shared): lsp_periodogram_gls_weighted_batched.

        Returns (P float32[B,Nf] or None, peak_idx int32[B] or None, peak_val float32[B] or None)."""
        import torch
        _want(x, torch.float32, 2, "x")
        B, Nt = x.shape
        if t.dim() == 1:
            _want(t, torch.float64, 1, "t"); t_stride = 0
            if t.numel() != Nt:
                raise ValueError("shared t must have length Nt")
        else:
            _want(t, torch.float64, 2, "t"); t_stride = Nt
            if tuple(t.shape) != (B, Nt):
                raise ValueError("t must be [B, Nt]")
        P = torch.empty((B, int(Nf)), dtype=torch.float32, device=x.device) if want_P else None
        pi = torch.empty(B, dtype=torch.int32, device=x.device) if want_peaks else None
        pv = torch.empty(B, dtype=torch.float32, device=x.device) if want_peaks else None
        if weights is not None:
            _want(weights, torch.float32, weights.dim(), "weights")
            if tuple(weights.shape) not in ((B, Nt), (Nt,)):
                raise ValueError("weights must be [B, Nt] or [Nt]")
            st = self._lib.lsp_periodogram_gls_weighted_batched(
                self._h, t.data_ptr(), t_stride, x.data_ptr(), Nt, weights.data_ptr(), Nt if weights.dim() == 2 else 0,
                B, Nt, float(f_min), float(df), int(Nf),
                P.data_ptr() if want_P else None, int(Nf),
                pi.data_ptr() if want_peaks else None, pv.data_ptr() if want_peaks else None,
                _stream_ptr(stream))
            self._check(st, "lsp_periodogram_gls_weighted_batched")
            return P, pi, pv
        fn = self._lib.lsp_periodogram_gls_batched if gls else self._lib.lsp_periodogram_batched
        st = fn(
            self._h, t.data_ptr(), t_stride, x.data_ptr(), Nt, B, Nt, float(f_min), float(df), int(Nf),
            P.data_ptr() if want_P else None, int(Nf),
            pi.data_ptr() if want_peaks else None, pv.data_ptr() if want_peaks else None,
            _stream_ptr(stream))
        self._check(st, "lsp_periodogram_batched")
        return P, pi, pv

    def false_alarm(self, P, Nt: int, N_ind: float, out=None, stream=None):
        """lsp_false_alarm: eq. (3) for a CUDA float32 tensor of periodogram values (any shape, contiguous)."""
        import torch
        if P.dtype != torch.float32 or not P.is_cuda or not P.is_contiguous():
            raise ValueError("P must be a contiguous float32 CUDA tensor")
        Q = out if out is not None else torch.empty_like(P)
        st = self._lib.lsp_false_alarm(self._h, P.data_ptr(), P.numel(), int(Nt), float(N_ind), Q.data_ptr(),
                                       _stream_ptr(stream))
        self._check(st, "lsp_false_alarm")
        return Q

    # -- host-pointer entry points (CPU tensors / numpy arrays in and out; synchronous)
    def periodogram_host(self, t, x, f_min: float, df: float, Nf: int, out=None, stream=None):
        """lsp_periodogram_host: CPU (ideally pinned) torch tensors; copies + compute + sync."""
        import torch
        _want(t, torch.float64, 1, "t", cuda=False); _want(x, torch.float32, 1, "x", cuda=False)
        P = out if out is not None else torch.empty(int(Nf), dtype=torch.float32)
        st = self._lib.lsp_periodogram_host(self._h, t.data_ptr(), x.data_ptr(), t.numel(),
                                            float(f_min), float(df), int(Nf), P.data_ptr(), _stream_ptr(stream))
        self._check(st, "lsp_periodogram_host")
        return P

    def periodogram_batched_host(self, t, x, f_min: float, df: float, Nf: int,
                                 P=None, peak_idx=None, peak_val=None, stream=None):
        import torch
        _want(x, torch.float32, 2, "x", cuda=False)
        B, Nt = x.shape
        share = 1 if t.dim() == 1 else 0
        _want(t, torch.float64, t.dim(), "t", cuda=False)
        st = self._lib.lsp_periodogram_batched_host(
            self._h, t.data_ptr(), share, x.data_ptr(), B, Nt, float(f_min), float(df), int(Nf),
            P.data_ptr() if P is not None else None,
            peak_idx.data_ptr() if peak_idx is not None else None,
            peak_val.data_ptr() if peak_val is not None else None, _stream_ptr(stream))
        self._check(st, "lsp_periodogram_batched_host")
        return P, peak_idx, peak_val


def _want(tensor, dtype, ndim, name, cuda: bool = True):
    if tensor.dtype != dtype or tensor.dim() != ndim or not tensor.is_contiguous():
        raise ValueError("%s must be a contiguous %s tensor with %d dim(s)" % (name, dtype, ndim))
    if tensor.is_cuda != cuda:
        raise ValueError("%s must live on %s" % (name, "the GPU" if cuda else "the host"))
