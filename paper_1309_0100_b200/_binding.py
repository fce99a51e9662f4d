"""Thin ctypes binding of libfredec_b200.so (include/fredec.h): argument marshalling only.

Every step of the scan runs in the CUDA kernels behind the C-ABI; nothing here computes.
Arrays may be numpy arrays (host buffers, staged by the library) or torch tensors (CPU,
pinned or CUDA; CUDA tensors are used in place).  There is no CPU fallback: a missing
library or a failing CUDA call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# FREDEC_LIB: a measurement build of the same library (paper_1309_0100_b200/build.py --variant), for A/B timings
LIB_PATH = os.environ.get("FREDEC_LIB") or os.path.join(_HERE, "libfredec_b200.so")

FREDEC_OK, FREDEC_EINVAL, FREDEC_EDATA, FREDEC_ESINGULAR, FREDEC_ECUDA, FREDEC_ELIMIT = 0, -1, -2, -3, -4, -5
FREDEC_D_MAX, FREDEC_TOPK_MAX, FREDEC_TOPK_NOALLOC_K_MAX = 64, 1024, 128

# name -> (restype, argtypes); must list every symbol include/fredec.h declares
_P, _I64, _I32, _F64 = C.c_void_p, C.c_int64, C.c_int32, C.c_double
SIGNATURES = {
    "fredec_scan": (C.c_int, [_P, _P, _P, _I64, _P, _I32, _F64, _F64, _I64, _P]),
    "fredec_scan_batched": (C.c_int, [_P, _P, _P, _I64, _I64, _P, _I32, _F64, _F64, _I64, _P]),
    "fredec_scan_topk": (C.c_int, [_P, _P, _P, _I64, _P, _I32, _F64, _F64, _I64, _P, _I32, _P]),
    "fredec_scan_topk_batched": (C.c_int, [_P, _P, _P, _I64, _I64, _P, _I32, _F64, _F64, _I64, _P, _I32, _P]),
    "fredec_chi2_base": (C.c_int, [_P, _P, _P, _I64, _P, _I32, _P]),
    "fredec_chi2_base_batched": (C.c_int, [_P, _P, _P, _I64, _I64, _P, _I32, _P]),
    "fredec_topk": (C.c_int, [_P, _I64, _I32, _P]),
    "fredec_topk_batched": (C.c_int, [_P, _I64, _I64, _I32, _P]),
    "fredec_topk_noalloc": (C.c_int, [_P, _I64, _I32, _P, _P, _P]),
    "fredec_topk_noalloc_cuda_error": (C.c_int, []),
    "fredec_topk_noalloc_scratch_bytes": (C.c_int64, []),
    "fredec_zstat": (C.c_int, [_P, _I64, _F64, _F64, _P]),
    "fredec_fap1": (C.c_int, [_P, _I64, _F64, _F64, _P]),
    "fredec_bandwidth": (C.c_int, [_P, _P, _I64, _F64, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "fredec_phase1": (C.c_int, [_P, _P, _P, _I64, _F64, _F64, _I64, _F64, _F64, _F64, _I32, _I32,
                                _P, _P, _P, _I32, _P, C.POINTER(C.c_int32)]),
    "fredec_phase1_refined": (C.c_int, [_P, _P, _P, _I64, _F64, _F64, _I64, _F64, _F64, _F64, _I32, _I32, _I32, _F64,
                                        _P, _P, _P, _I32, _P, _P, C.POINTER(C.c_int32)]),
    "fredec_trig_averages": (C.c_int, [_P, _P, _P, _I64, _P, _I64, _P]),
    "fredec_subset_fits": (C.c_int, [_P, _P, _P, _I64, _P, _I32, _P]),
    "fredec_refine": (C.c_int, [_P, _P, _P, _I64, _P, _I32, _I32, _F64, C.POINTER(C.c_double),
                                C.POINTER(C.c_int32)]),
    "fredec_refine_batched": (C.c_int, [_P, _P, _P, _I64, _P, _I32, _P, _I64, _I32, _F64, _P, _P, _P, _P]),
    "fredec_set_stream": (C.c_int, [_P]),
    "fredec_set_async": (C.c_int, [_I32]),
    "fredec_set_timing": (C.c_int, [_I32]),
    "fredec_last_status": (C.c_int, [C.POINTER(C.c_int32)]),
    "fredec_pending": (C.c_int, []),
    "fredec_last_timing": (C.c_int, [C.POINTER(C.c_double)]),
    "fredec_last_launches": (C.c_int, []),
    "fredec_shutdown": (C.c_int, []),
    "fredec_strerror": (C.c_char_p, [C.c_int]),
    "fredec_last_cuda_error": (C.c_int, []),
    "fredec_version": (C.c_int, []),
}

# include/fredec_bench.h: the FP64 roofline probes live in a library of their own (bench.py only)
BENCH_LIB_PATH = os.path.join(_HERE, "libfredec_bench.so")
BENCH_SIGNATURES = {
    "fredec_bench_fp64": (C.c_int, [_I32, _I64, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "fredec_bench_fp64_name": (C.c_char_p, [_I32]),
}

_lib = None
_bench_lib = None


class FredecError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        super().__init__(f"{where} failed: {code} ({detail})")


def lib():
    """Loads libfredec_b200.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1309_0100_b200.build` "
                "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def bench_lib():
    """Loads libfredec_bench.so (measurement probes); raises if it has not been built."""
    global _bench_lib
    if _bench_lib is None:
        if not os.path.exists(BENCH_LIB_PATH):
            raise RuntimeError(f"{BENCH_LIB_PATH} is missing: build it with `python -m paper_1309_0100_b200.build`")
        L = C.CDLL(BENCH_LIB_PATH)
        for name, (res, args) in BENCH_SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _bench_lib = L
    return _bench_lib


def _check(rc: int, where: str) -> int:
    if rc < 0:
        L = lib()
        detail = L.fredec_strerror(rc).decode()
        if rc == FREDEC_ECUDA:
            detail += f", cudaError {L.fredec_last_cuda_error()}"
        raise FredecError(rc, where, detail)
    return rc


def _is_torch(a) -> bool:
    return type(a).__module__.startswith("torch")


def _ptr(a, dtype=np.float64):
    """(address, keep-alive) of a contiguous float64/int64 numpy array or torch tensor."""
    if a is None:
        return None, None
    if _is_torch(a):
        import torch
        want = torch.float64 if dtype == np.float64 else torch.int64
        if a.dtype != want or not a.is_contiguous():
            raise TypeError(f"need a contiguous {want} tensor")
        return a.data_ptr(), a
    arr = np.ascontiguousarray(a, dtype=dtype)
    return arr.ctypes.data, arr


def _empty_like_kind(ref, shape, dtype=np.float64):
    if _is_torch(ref):
        import torch
        return torch.empty(shape, dtype=torch.float64 if dtype == np.float64 else torch.int64,
                           device=ref.device)
    return np.empty(shape, dtype=dtype)


def fredec_set_stream(stream=None) -> None:
    """stream: None (default stream), an int cudaStream_t, or a torch.cuda.Stream."""
    handle = 0 if stream is None else getattr(stream, "cuda_stream", stream)
    _check(lib().fredec_set_stream(C.c_void_p(int(handle))), "fredec_set_stream")


def fredec_set_async(enable: bool) -> None:
    """Asynchronous form for scan / top-k calls on device pointers; see include/fredec.h."""
    _check(lib().fredec_set_async(1 if enable else 0), "fredec_set_async")


def fredec_set_timing(enable: bool) -> None:
    """Per-stage CUDA-event timing of the scan / top-k calls (fredec_last_timing) on or off."""
    _check(lib().fredec_set_timing(1 if enable else 0), "fredec_set_timing")


def fredec_last_status() -> int:
    """Resolves the pending asynchronous call: raises on a data error, else returns the peak count."""
    count = C.c_int32(0)
    _check(lib().fredec_last_status(C.byref(count)), "fredec_last_status")
    return count.value


def fredec_scan(t, x, w, base_funcs, f0, df, K, z_out=None):
    """z[k] = chi-square reduction at f0 + k*df; see include/fredec.h."""
    N = int(t.shape[-1])
    d = 0 if base_funcs is None else int(base_funcs.shape[0]) if base_funcs.ndim == 2 else 1
    if d == 0:
        base_funcs = None
    z = _empty_like_kind(t, (int(K),)) if z_out is None else z_out
    (pt, kt), (px, kx), (pw, kw), (pb, kb), (pz, kz) = map(_ptr, (t, x, w, base_funcs, z))
    _check(lib().fredec_scan(pt, px, pw, N, pb, d, float(f0), float(df), int(K), pz), "fredec_scan")
    return z if z_out is None or kz is z else kz


def fredec_scan_batched(t, x, w, base_funcs, f0, df, K, z_out=None):
    B, N = int(t.shape[0]), int(t.shape[1])
    d = 0 if base_funcs is None else int(base_funcs.shape[1])
    if d == 0:
        base_funcs = None
    z = _empty_like_kind(t, (B, int(K))) if z_out is None else z_out
    (pt, kt), (px, kx), (pw, kw), (pb, kb), (pz, kz) = map(_ptr, (t, x, w, base_funcs, z))
    _check(lib().fredec_scan_batched(pt, px, pw, B, N, pb, d, float(f0), float(df), int(K), pz),
           "fredec_scan_batched")
    return z


def fredec_scan_topk(t, x, w, base_funcs, f0, df, K, k, z_out=None, idx_out=None, want_z=True):
    """Scan + peaks in one call.  Returns (z or None, idx[k], count); count is None when the call was only
    enqueued (fredec_set_async): fredec_last_status() then delivers it."""
    N = int(t.shape[-1])
    d = 0 if base_funcs is None else int(base_funcs.shape[0])
    if d == 0:
        base_funcs = None
    z = (_empty_like_kind(t, (int(K),)) if z_out is None else z_out) if want_z else None
    idx = _empty_like_kind(t, (int(k),), np.int64) if idx_out is None else idx_out
    (pt, kt), (px, kx), (pw, kw), (pb, kb), (pz, kz) = map(_ptr, (t, x, w, base_funcs, z))
    pi, ki = _ptr(idx, np.int64)
    count = _check(lib().fredec_scan_topk(pt, px, pw, N, pb, d, float(f0), float(df), int(K), pz,
                                          int(k), pi), "fredec_scan_topk")
    return z, idx, (None if lib().fredec_pending() else count)   # asynchronous: the count is fredec_last_status()


def fredec_scan_topk_batched(t, x, w, base_funcs, f0, df, K, k, z_out=None, idx_out=None, want_z=True):
    B, N = int(t.shape[0]), int(t.shape[1])
    d = 0 if base_funcs is None else int(base_funcs.shape[1])
    if d == 0:
        base_funcs = None
    z = (_empty_like_kind(t, (B, int(K))) if z_out is None else z_out) if want_z else None
    idx = _empty_like_kind(t, (B, int(k)), np.int64) if idx_out is None else idx_out
    (pt, kt), (px, kx), (pw, kw), (pb, kb), (pz, kz) = map(_ptr, (t, x, w, base_funcs, z))
    pi, ki = _ptr(idx, np.int64)
    _check(lib().fredec_scan_topk_batched(pt, px, pw, B, N, pb, d, float(f0), float(df), int(K), pz,
                                          int(k), pi), "fredec_scan_topk_batched")
    return z, idx


def fredec_chi2_base(t, x, w, base_funcs) -> float:
    N = int(t.shape[-1])
    d = 0 if base_funcs is None else int(base_funcs.shape[0])
    if d == 0:
        base_funcs = None
    out = np.empty(1)
    (pt, kt), (px, kx), (pw, kw), (pb, kb) = map(_ptr, (t, x, w, base_funcs))
    _check(lib().fredec_chi2_base(pt, px, pw, N, pb, d, out.ctypes.data), "fredec_chi2_base")
    return float(out[0])


def fredec_chi2_base_batched(t, x, w, base_funcs):
    B, N = int(t.shape[0]), int(t.shape[1])
    d = 0 if base_funcs is None else int(base_funcs.shape[1])
    if d == 0:
        base_funcs = None
    out = np.empty(B)
    (pt, kt), (px, kx), (pw, kw), (pb, kb) = map(_ptr, (t, x, w, base_funcs))
    _check(lib().fredec_chi2_base_batched(pt, px, pw, B, N, pb, d, out.ctypes.data),
           "fredec_chi2_base_batched")
    return out


def fredec_topk(z, k, idx_out=None):
    """Returns (idx[k], count): indices of the k highest peaks, -1 padded."""
    K = int(z.shape[-1])
    idx = _empty_like_kind(z, (int(k),), np.int64) if idx_out is None else idx_out
    pz, kz = _ptr(z)
    pi, ki = _ptr(idx, np.int64)
    count = _check(lib().fredec_topk(pz, K, int(k), pi), "fredec_topk")
    return idx, (None if lib().fredec_pending() else count)      # asynchronous: the count is fredec_last_status()


def fredec_topk_noalloc(z, k, idx_out, count_out, stream=None):
    """fredec_topk for callers that may not allocate device memory (include/fredec.h): the library's only
    scratch is an array built into it, so nothing here or below calls cudaMalloc.  z, idx_out (int64 [k]) and
    count_out (int32 [1]) are CUDA tensors that the CALLER provides -- this wrapper creates none; stream is
    None (default stream), an int cudaStream_t or a torch.cuda.Stream.  Returns as soon as the work is
    enqueued: synchronise with the stream before reading idx_out / count_out.  Calls that may overlap on
    the GPU race on the shared array; k <= FREDEC_TOPK_NOALLOC_K_MAX."""
    import torch
    if not (_is_torch(z) and _is_torch(idx_out) and _is_torch(count_out)):
        raise TypeError("fredec_topk_noalloc takes caller-provided CUDA tensors only")
    if count_out.dtype != torch.int32 or count_out.numel() < 1 or not count_out.is_contiguous():
        raise TypeError("count_out: contiguous int32 tensor with one element")
    if idx_out.numel() < int(k):
        raise ValueError("idx_out is shorter than k")
    pz, kz = _ptr(z)
    pi, ki = _ptr(idx_out, np.int64)
    h = 0 if stream is None else int(getattr(stream, "cuda_stream", stream))
    rc = lib().fredec_topk_noalloc(pz, int(z.shape[-1]), int(k), pi, count_out.data_ptr(), h or None)
    if rc == FREDEC_ECUDA:
        raise FredecError(rc, "fredec_topk_noalloc", f"cudaError {lib().fredec_topk_noalloc_cuda_error()}")
    _check(rc, "fredec_topk_noalloc")


def fredec_topk_noalloc_scratch_bytes() -> int:
    return int(lib().fredec_topk_noalloc_scratch_bytes())


def fredec_topk_batched(z, k, idx_out=None):
    B, K = int(z.shape[0]), int(z.shape[1])
    idx = _empty_like_kind(z, (B, int(k)), np.int64) if idx_out is None else idx_out
    pz, kz = _ptr(z)
    pi, ki = _ptr(idx, np.int64)
    _check(lib().fredec_topk_batched(pz, B, K, int(k), pi), "fredec_topk_batched")
    return idx


def fredec_zstat(dchi2, chi2_base, N_H, z_out=None):
    """The paper's statistic z = (N_H/2) ln(chi2_base / (chi2_base - dchi2)); see include/fredec.h."""
    K = int(dchi2.shape[-1])
    z = _empty_like_kind(dchi2, (K,)) if z_out is None else z_out
    (pi, ki), (po, ko) = _ptr(dchi2), _ptr(z)
    _check(lib().fredec_zstat(pi, K, float(chi2_base), float(N_H), po), "fredec_zstat")
    return z if z_out is None or ko is z else ko


def fredec_fap1(z, W, A1=1.0, fap_out=None):
    """Single-frequency FAP bound min(1, A1 W exp(-z) sqrt z); see include/fredec.h."""
    K = int(z.shape[-1])
    fap = _empty_like_kind(z, (K,)) if fap_out is None else fap_out
    (pi, ki), (po, ko) = _ptr(z), _ptr(fap)
    _check(lib().fredec_fap1(pi, K, float(W), float(A1), po), "fredec_fap1")
    return fap if fap_out is None or ko is fap else ko


def fredec_bandwidth(t, w, f_max):
    """(T_eff, W) = (sqrt(4 pi Var_w t), f_max T_eff)."""
    N = int(t.shape[-1])
    te, W = C.c_double(), C.c_double()
    (pt, kt), (pw, kw) = _ptr(t), _ptr(w)
    _check(lib().fredec_bandwidth(pt, pw, N, float(f_max), C.byref(te), C.byref(W)), "fredec_bandwidth")
    return te.value, W.value


def fredec_phase1(t, x, w, f0, df, K, fap0=0.05, fap1=0.1, A1=1.0, max_base=10, k_peaks=32, pool_cap=None,
                  refine_base=False, refine_iter=20, refine_tol=1e-9):
    """Phase 1 of FREDEC (preliminary scan): returns a dict with the candidate pool (grid indices,
    statistic, FAP; sorted by FAP) and the base frequencies' grid indices in the order found.
    refine_base: fredec_phase1_refined (the base frequencies are refitted after every addition); the dict
    then also holds base_freqs, the frequencies the base ends with."""
    N = int(t.shape[-1])
    pool_cap = max(1, N // 10) if pool_cap is None else int(pool_cap)
    pool_idx = np.empty(pool_cap, dtype=np.int64)
    pool_z, pool_fap = np.empty(pool_cap), np.empty(pool_cap)
    base_idx = np.empty(int(max_base), dtype=np.int64)
    base_freq = np.empty(int(max_base))
    n_base = C.c_int32(0)
    (pt, kt), (px, kx), (pw, kw) = map(_ptr, (t, x, w))
    if refine_base:
        n = _check(lib().fredec_phase1_refined(
            pt, px, pw, N, float(f0), float(df), int(K), float(fap0), float(fap1), float(A1), int(max_base),
            int(k_peaks), int(refine_iter), float(refine_tol), pool_idx.ctypes.data, pool_z.ctypes.data,
            pool_fap.ctypes.data, pool_cap, base_idx.ctypes.data, base_freq.ctypes.data, C.byref(n_base)),
            "fredec_phase1_refined")
    else:
        n = _check(lib().fredec_phase1(pt, px, pw, N, float(f0), float(df), int(K), float(fap0), float(fap1),
                                       float(A1), int(max_base), int(k_peaks), pool_idx.ctypes.data,
                                       pool_z.ctypes.data, pool_fap.ctypes.data, pool_cap, base_idx.ctypes.data,
                                       C.byref(n_base)), "fredec_phase1")
    out = {"pool_idx": pool_idx[:n].copy(), "pool_z": pool_z[:n].copy(), "pool_fap": pool_fap[:n].copy(),
           "base_idx": base_idx[:n_base.value].copy()}
    if refine_base:
        out["base_freqs"] = base_freq[:n_base.value].copy()
    return out


def fredec_trig_averages(t, x, w, freqs, out=None):
    """[M][10] trigonometric averages of the paper's systems (19) and (20); see include/fredec.h."""
    N, M = int(t.shape[-1]), int(freqs.shape[-1])
    res = _empty_like_kind(t, (M, 10)) if out is None else out
    (pt, kt), (px, kx), (pw, kw), (pf, kf), (po, ko) = map(_ptr, (t, x, w, freqs, res))
    _check(lib().fredec_trig_averages(pt, px, pw, N, pf, M, po), "fredec_trig_averages")
    return res if out is None or ko is res else ko


def fredec_subset_fits(t, x, w, freqs, l_out=None):
    """l[mask] = min chi2 of constant + sinusoids at the frequencies selected by mask, for all
    2^n subsets of freqs; see include/fredec.h."""
    N, n = int(t.shape[-1]), int(freqs.shape[-1])
    res = _empty_like_kind(t, (1 << n,)) if l_out is None else l_out
    (pt, kt), (px, kx), (pw, kw), (pf, kf), (po, ko) = map(_ptr, (t, x, w, freqs, res))
    _check(lib().fredec_subset_fits(pt, px, pw, N, pf, n, po), "fredec_subset_fits")
    return res if l_out is None or ko is res else ko


def fredec_refine(t, x, w, freqs, max_iter=20, tol=1e-9):
    """Local multifrequency fit: returns (refined freqs [n] as numpy, l = min chi2, iterations)."""
    N = int(t.shape[-1])
    f = np.array(freqs.cpu().numpy() if _is_torch(freqs) else freqs, dtype=np.float64, copy=True)
    l, it = C.c_double(), C.c_int32()
    (pt, kt), (px, kx), (pw, kw) = map(_ptr, (t, x, w))
    _check(lib().fredec_refine(pt, px, pw, N, f.ctypes.data, int(f.shape[0]), int(max_iter), float(tol),
                               C.byref(l), C.byref(it)), "fredec_refine")
    return f, l.value, it.value


def fredec_refine_batched(t, x, w, pool_freqs, masks=None, max_iter=20, tol=1e-9, T=None):
    """Local multifrequency fits of many tuples of one pool (bit j of masks[i] selects pool_freqs[j];
    masks=None with T: T copies of the whole pool).  Returns (freqs [T][n_pool], l [T], iters [T] int32,
    status [T] int32) as numpy arrays."""
    N, n_pool = int(t.shape[-1]), int(pool_freqs.shape[-1])
    pm = None
    if masks is not None and _is_torch(masks) and masks.is_cuda:
        pm, km = _ptr(masks, np.int64)                       # device masks: used in place
        T = int(masks.shape[0])
    elif masks is not None:
        masks = np.ascontiguousarray(masks.cpu().numpy() if _is_torch(masks) else masks, dtype=np.int64)
        T = int(masks.shape[0])
        pm = masks.ctypes.data
    T = 1 if T is None else int(T)
    freqs = np.empty((T, n_pool))
    l = np.empty(T)
    iters, status = np.empty(T, dtype=np.int32), np.empty(T, dtype=np.int32)
    (pt, kt), (px, kx), (pw, kw), (pp, kp) = map(_ptr, (t, x, w, pool_freqs))
    _check(lib().fredec_refine_batched(pt, px, pw, N, pp, n_pool, pm, T,
                                       int(max_iter), float(tol), freqs.ctypes.data, l.ctypes.data,
                                       iters.ctypes.data, status.ctypes.data), "fredec_refine_batched")
    return freqs, l, iters, status


def fredec_last_timing() -> dict:
    out = (C.c_double * 4)()
    _check(lib().fredec_last_timing(out), "fredec_last_timing")
    return {"prep_ms": out[0], "scan_ms": out[1], "topk_ms": out[2], "total_ms": out[3]}


def fredec_last_launches() -> int:
    return int(lib().fredec_last_launches())


def fredec_bench_fp64(mode: int = 0, iters: int = 1 << 16):
    """(TFLOP/s, ms) of an FP64 roofline probe (include/fredec_bench.h): mode 0 = DFMA only (the FP64
    FMA peak), modes >= 1 = DMMA loops, see fredec_bench_fp64_name."""
    tf, ms = C.c_double(), C.c_double()
    _check(bench_lib().fredec_bench_fp64(int(mode), int(iters), C.byref(tf), C.byref(ms)), "fredec_bench_fp64")
    return tf.value, ms.value


def fredec_bench_fp64_name(mode: int):
    name = bench_lib().fredec_bench_fp64_name(int(mode))
    return None if name is None else name.decode()


def fredec_shutdown() -> None:
    _check(lib().fredec_shutdown(), "fredec_shutdown")


def fredec_version() -> int:
    return int(lib().fredec_version())
