"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain fp64 CPU implementation of the Lomb-Scargle periodogram as the paper defines
it (two-pass eqs (1)+(2)).  Two independent spellings live here:

  * `lsp_oracle.c`   -- C, OpenMP over frequencies; the oracle proper, used for parity
                        and timed by bench.py's cpu_baseline / --impl reference legs.
  * `periodogram_numpy` -- the same definition in ~20 lines of numpy, used by the unit
                        tests to check the C build on small inputs.

Nothing under paper_1007_1658_b200/ imports this package, and this package imports
nothing from it.  Only tests/, __graft_entry__.smoke() and bench.py (cpu_baseline and
--impl reference) may import it.  Every function cites the passage it follows.

Pins: tests/test_oracle_pins.py (P1..P9 of DESIGN.md; GP1..GP5 for the generalised periodogram, GW1..GW5 for its
weighted form).
No function here is "parity unpinned" (false_alarm_probability: pins F1-F3).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lsp_oracle.c")
_LIB = os.path.join(_HERE, "liblsp_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile lsp_oracle.c with gcc (-O2, OpenMP, no fast-math).  Returns the .so path."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99",
           "-fno-fast-math", "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.lsp_oracle_periodogram.restype = ctypes.c_int
        lib.lsp_oracle_periodogram.argtypes = [
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
            ctypes.c_double, ctypes.c_double, ctypes.c_void_p, ctypes.c_int64,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
        lib.lsp_oracle_gls.restype = ctypes.c_int
        lib.lsp_oracle_gls.argtypes = lib.lsp_oracle_periodogram.argtypes
        lib.lsp_oracle_gls_weighted.restype = ctypes.c_int
        lib.lsp_oracle_gls_weighted.argtypes = [
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
            ctypes.c_double, ctypes.c_double, ctypes.c_void_p, ctypes.c_int64,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
        lib.lsp_oracle_moments.restype = None
        lib.lsp_oracle_moments.argtypes = [ctypes.c_void_p, ctypes.c_int64,
                                           ctypes.c_void_p, ctypes.c_void_p]
        lib.lsp_oracle_argmax.restype = ctypes.c_int64
        lib.lsp_oracle_argmax.argtypes = [ctypes.c_void_p, ctypes.c_int64]
        _lib = lib
    return _lib


def host_threads() -> int:
    """Cores this process may use (what the timed oracle legs report as `cores`)."""
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:                                   # pragma: no cover
        return os.cpu_count() or 1


def moments(x: np.ndarray):
    """Mean and sample variance (N-1) of the fp32 series in fp64 (reading G1)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    m = ctypes.c_double()
    v = ctypes.c_double()
    _load().lsp_oracle_moments(x.ctypes.data, x.size, ctypes.byref(m), ctypes.byref(v))
    return m.value, v.value


def periodogram(t, x, f_min: float, df: float, Nf: int,
                ks: Optional[np.ndarray] = None, nthreads: int = 0,
                return_threads: bool = False):
    """P[k] for the grid f_k = f_min + k*df (eqs (1)+(2)).

    ks=None evaluates k = 0..Nf-1; otherwise only the listed grid indices (used for
    the strided subsets and dense windows at the large configs).  Returns float64.
    """
    t = np.ascontiguousarray(t, dtype=np.float64)
    x = np.ascontiguousarray(x, dtype=np.float32)
    assert t.ndim == 1 and t.shape == x.shape and t.size >= 2
    if ks is None:
        nk, ks_ptr = int(Nf), None
    else:
        ks = np.ascontiguousarray(ks, dtype=np.int64)
        assert ks.size == 0 or (ks.min() >= 0 and ks.max() < Nf)
        nk, ks_ptr = int(ks.size), ks.ctypes.data
    P = np.empty(nk, dtype=np.float64)
    scratch = np.empty(t.size, dtype=np.float64)
    used = _load().lsp_oracle_periodogram(t.ctypes.data, x.ctypes.data, t.size,
                                          float(f_min), float(df), ks_ptr, nk,
                                          P.ctypes.data, scratch.ctypes.data, int(nthreads))
    return (P, used) if return_threads else P


def periodogram_gls(t, x, f_min: float, df: float, Nf: int,
                    ks: Optional[np.ndarray] = None, nthreads: int = 0) -> np.ndarray:
    """Generalised (floating-mean) periodogram on the grid f_k = f_min + k*df, same normalisation as
    `periodogram` (definition by a 3-parameter least-squares fit, see lsp_oracle.c)."""
    t = np.ascontiguousarray(t, dtype=np.float64)
    x = np.ascontiguousarray(x, dtype=np.float32)
    assert t.ndim == 1 and t.shape == x.shape and t.size >= 4
    if ks is None:
        nk, ks_ptr = int(Nf), None
    else:
        ks = np.ascontiguousarray(ks, dtype=np.int64)
        nk, ks_ptr = int(ks.size), ks.ctypes.data
    P = np.empty(nk, dtype=np.float64)
    scratch = np.empty(t.size, dtype=np.float64)
    _load().lsp_oracle_gls(t.ctypes.data, x.ctypes.data, t.size, float(f_min), float(df), ks_ptr, nk,
                           P.ctypes.data, scratch.ctypes.data, int(nthreads))
    return P


def periodogram_gls_weighted(t, x, w, f_min: float, df: float, Nf: int,
                             ks: Optional[np.ndarray] = None, nthreads: int = 0) -> np.ndarray:
    """Weighted generalised periodogram (per-sample weights w_j >= 0): the weighted
    3-parameter least-squares fit, P = (Nt - 1)/2 * (chi0^2 - chi^2_min)/chi0^2 (reading G14; see lsp_oracle.c)."""
    t = np.ascontiguousarray(t, dtype=np.float64)
    x = np.ascontiguousarray(x, dtype=np.float32)
    w = np.ascontiguousarray(w, dtype=np.float32)
    assert t.ndim == 1 and t.shape == x.shape == w.shape and t.size >= 4
    assert np.all(np.isfinite(w)) and np.all(w >= 0) and w.sum() > 0
    if ks is None:
        nk, ks_ptr = int(Nf), None
    else:
        ks = np.ascontiguousarray(ks, dtype=np.int64)
        nk, ks_ptr = int(ks.size), ks.ctypes.data
    P = np.empty(nk, dtype=np.float64)
    s1 = np.empty(t.size, dtype=np.float64)
    s2 = np.empty(t.size, dtype=np.float64)
    _load().lsp_oracle_gls_weighted(t.ctypes.data, x.ctypes.data, w.ctypes.data, t.size, float(f_min), float(df),
                                    ks_ptr, nk, P.ctypes.data, s1.ctypes.data, s2.ctypes.data, int(nthreads))
    return P


def periodogram_gls_numpy(t, x, freqs) -> np.ndarray:
    """Numpy twin of lsp_oracle_gls: the chi^2 reduction of the fit x ~ a cos + b sin + c by numpy.linalg.lstsq
    (SVD; a different solver from the C normal equations), over 2 var."""
    t = np.asarray(t, dtype=np.float64)
    X = np.asarray(x, dtype=np.float32).astype(np.float64)
    Nt = t.size
    X = X - X.sum() / Nt
    chi0 = (X * X).sum()
    var = chi0 / (Nt - 1)
    out = np.empty(len(freqs))
    for i, f in enumerate(np.asarray(freqs, dtype=np.float64)):
        w = 2.0 * np.pi * f
        A = np.stack([np.cos(w * t), np.sin(w * t), np.ones(Nt)], axis=1)
        beta, _, rank, _ = np.linalg.lstsq(A, X, rcond=None)
        out[i] = 0.0 if rank < 3 else (chi0 - ((X - A @ beta) ** 2).sum()) / (2.0 * var)
    return out


def periodogram_batched(t, x, f_min: float, df: float, Nf: int, nthreads: int = 0):
    """B independent series on one shared grid: P[B,Nf], peak index, peak value."""
    t = np.asarray(t, dtype=np.float64)
    x = np.asarray(x, dtype=np.float32)
    B = x.shape[0]
    P = np.empty((B, Nf), dtype=np.float64)
    for b in range(B):
        tb = t[b] if t.ndim == 2 else t
        P[b] = periodogram(tb, x[b], f_min, df, Nf, nthreads=nthreads)
    idx = np.array([argmax(P[b]) for b in range(B)], dtype=np.int64)
    return P, idx, P[np.arange(B), idx]


def argmax(P: np.ndarray) -> int:
    """Lowest index among equal maxima (reading G9)."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    return int(_load().lsp_oracle_argmax(P.ctypes.data, P.size))


def periodogram_numpy(t, x, freqs) -> np.ndarray:
    """Numpy twin of lsp_oracle.c: eqs (1)+(2), same readings G1, G5, G7."""
    t = np.asarray(t, dtype=np.float64)
    X = np.asarray(x, dtype=np.float32).astype(np.float64)
    Nt = t.size
    X = X - X.sum() / Nt
    var = (X * X).sum() / (Nt - 1)                             # G1
    out = np.empty(len(freqs))
    for i, f in enumerate(np.asarray(freqs, dtype=np.float64)):
        w = 2.0 * np.pi * f
        if w == 0.0:
            out[i] = X.sum() ** 2 / Nt / (2.0 * var)
            continue
        tau = np.arctan2(np.sin(2 * w * t).sum(), np.cos(2 * w * t).sum()) / (2 * w)   # eq. (2)
        c = np.cos(w * (t - tau))
        s = np.sin(w * (t - tau))
        CC, SS = (c * c).sum(), (s * s).sum()
        p = 0.0
        if CC > 1e-12 * Nt:
            p += (X * c).sum() ** 2 / CC                       # eq. (1), first term
        if SS > 1e-12 * Nt:
            p += (X * s).sum() ** 2 / SS                       # eq. (1), second term
        out[i] = p / (2.0 * var)
    return out


def false_alarm_probability(P, Nt: int, Nf_ind: float) -> np.ndarray:
    """Eq. (3): Q = 1 - [1 - (1 - p)^((Nt-3)/2)]^Nf, p the normalised power in [0, 1]
    (Nf -> N_f,ind).

    Reading G13: the paper writes p = 2 P_n / N_t, which is the beta variable of the cited law
    (Schwarzenberg-Czerny 1998) when "unit variance" means sum X^2 / N_t = 1.  This library scales with the
    sample variance sum X^2 / (N_t - 1) (reading G1), for which the SAME variable is p = 2 P / (N_t - 1): P 2 var is the
    chi^2 reduction of the two-parameter fit and (N_t - 1) var the total, so p ~ Beta(1, (N_t - 3)/2) and the single-trial
    survival is (1 - p)^((N_t - 3)/2), reaching 0 exactly at P_max = (N_t - 1)/2.  Pinned by scipy's incomplete beta
    function and by Monte-Carlo exceedance counts at N_t = 12 (tests/test_oracle_pins.py::test_fap_*)."""
    P = np.asarray(P, dtype=np.float64)
    base = np.clip(1.0 - 2.0 * P / (Nt - 1.0), 0.0, 1.0)
    single = base ** ((Nt - 3) / 2.0)
    return 1.0 - (1.0 - single) ** Nf_ind
