"""ctypes access to the CPU oracle (oracle/oracle_fredec.c).  TEST INFRASTRUCTURE ONLY:
imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference legs,
never by the product package."""
from __future__ import annotations

import ctypes as C
import numpy as np

from .build import build as _build

_lib = None
_f64p = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_i64p = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        for sfx in ("", "_ld"):
            f = getattr(L, "oracle_scan" + sfx)
            f.restype = C.c_int
            f.argtypes = [_f64p, _f64p, _f64p, C.c_int64, C.c_void_p, C.c_int32,
                          C.c_double, C.c_double, C.c_int64, _f64p]
            f = getattr(L, "oracle_chi2_base" + sfx)
            f.restype = C.c_int
            f.argtypes = [_f64p, _f64p, _f64p, C.c_int64, C.c_void_p, C.c_int32, _f64p]
            f = getattr(L, "oracle_trig_averages" + sfx)
            f.restype = C.c_int
            f.argtypes = [_f64p, _f64p, _f64p, C.c_int64, _f64p, C.c_int64, _f64p]
        L.oracle_topk.restype = C.c_int
        L.oracle_topk.argtypes = [_f64p, C.c_int64, C.c_int32, _i64p]
        L.oracle_num_threads.restype = C.c_int
        L.oracle_set_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


def _prep(t, x, w, base_funcs):
    t = np.ascontiguousarray(t, dtype=np.float64)
    x = np.ascontiguousarray(x, dtype=np.float64)
    w = np.ascontiguousarray(w, dtype=np.float64)
    N = t.shape[0]
    if base_funcs is None:
        base = np.zeros((0, N))
    else:
        base = np.ascontiguousarray(base_funcs, dtype=np.float64).reshape(-1, N)
    d = base.shape[0]
    bp = base.ctypes.data_as(C.c_void_p) if d > 0 else None
    return t, x, w, N, base, d, bp


def scan(t, x, w, base_funcs, f0, df, K, threads: int = 1, long_double: bool = False):
    """z[k] = chi-square reduction at f0 + k*df.  Raises on an oracle error code."""
    L = lib()
    t, x, w, N, base, d, bp = _prep(t, x, w, base_funcs)
    z = np.empty(int(K), dtype=np.float64)
    L.oracle_set_threads(int(threads) if threads > 0 else L.oracle_num_threads())
    fn = L.oracle_scan_ld if long_double else L.oracle_scan
    rc = fn(t, x, w, N, bp, d, float(f0), float(df), int(K), z)
    if rc != 0:
        raise RuntimeError(f"oracle_scan failed with code {rc}")
    return z


def scan_batched(t, x, w, base_funcs, f0, df, K, threads: int = 1):
    B = t.shape[0]
    return np.stack([scan(t[b], x[b], w[b], base_funcs[b], f0, df, K, threads) for b in range(B)])


def chi2_base(t, x, w, base_funcs, long_double: bool = False):
    L = lib()
    t, x, w, N, base, d, bp = _prep(t, x, w, base_funcs)
    out = np.empty(1, dtype=np.float64)
    fn = L.oracle_chi2_base_ld if long_double else L.oracle_chi2_base
    rc = fn(t, x, w, N, bp, d, out)
    if rc != 0:
        raise RuntimeError(f"oracle_chi2_base failed with code {rc}")
    return float(out[0])


def trig_averages(t, x, w, freqs, long_double: bool = False):
    """[M][10] trigonometric averages of PAPER.md:242-262, systems (19) and (20), at the given
    frequencies (cycles per unit of t); column order in oracle_fredec.c."""
    L = lib()
    t, x, w = (np.ascontiguousarray(a, dtype=np.float64) for a in (t, x, w))
    freqs = np.ascontiguousarray(freqs, dtype=np.float64)
    out = np.empty((freqs.shape[0], 10), dtype=np.float64)
    fn = L.oracle_trig_averages_ld if long_double else L.oracle_trig_averages
    rc = fn(t, x, w, t.shape[0], freqs, freqs.shape[0], out)
    if rc != 0:
        raise RuntimeError(f"oracle_trig_averages failed with code {rc}")
    return out


def topk(z, k):
    """Indices of the k highest peaks (S7), -1 padded; returns (idx[k], count)."""
    L = lib()
    z = np.ascontiguousarray(z, dtype=np.float64)
    idx = np.empty(int(k), dtype=np.int64)
    rc = L.oracle_topk(z, z.shape[0], int(k), idx)
    if rc < 0:
        raise RuntimeError(f"oracle_topk failed with code {rc}")
    return idx, rc


def topk_batched(z, k):
    return np.stack([topk(z[b], k)[0] for b in range(z.shape[0])])


def num_threads() -> int:
    return int(lib().oracle_num_threads())
