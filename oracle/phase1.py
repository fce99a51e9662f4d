"""CPU oracle of the statistic, the single-frequency FAP and phase 1 of FREDEC (numpy + the C
oracle's scan / topk).  TEST INFRASTRUCTURE ONLY (see oracle/__init__.py); shares no code with the
CUDA path.  Each function follows the passage it cites, in the paper's order and notation.

Pins (tests/test_phase1_pins.py; subset_fits: tests/test_subset_pins.py; refine:
tests/test_refine_pins.py): zstat against (N_H/2) ln(l_base/l_alt) with both l from QR fits;
T_eff against the closed form for evenly spaced, equally weighted times; fap1 against hand values;
phase 1 on constructed series whose outcome the rules fix (with refine_base: two OFF-grid sinusoids must
give a base of exactly two frequencies, each at the true value).  The coefficient A~_1 of eq. 13 and the
readings P1-P4 are not fixed by the paper: parity unpinned for those.
"""
from __future__ import annotations

import numpy as np

from . import chi2_base as _chi2_base, scan as _scan, topk as _topk


def zstat(dchi2, chi2_base: float, N_H: float):
    """PAPER.md:89-95 (eq. 8) / :106 (eq. 10), reading G1: z = (N_H/2) ln(l_base / l_alt),
    l_alt = l_base - dchi2."""
    dchi2 = np.asarray(dchi2, dtype=np.float64)
    l_alt = chi2_base - dchi2
    with np.errstate(divide="ignore"):
        return 0.5 * N_H * np.log(chi2_base / np.maximum(l_alt, 0.0))


def fap1(z, W: float, A1: float = 1.0):
    """PAPER.md:143 (eq. 13) with n = 1: FAP <~ A~_1 W e^{-z} z^{1/2}, capped at 1 (a probability)."""
    z = np.asarray(z, dtype=np.float64)
    zz = np.maximum(z, 0.0)
    return np.where(z > 0.0, np.minimum(1.0, A1 * W * np.exp(-zz) * np.sqrt(zz)), 1.0)


def bandwidth(t, w, f_max: float):
    """T_eff = sqrt(4 pi Var(t_i)) with the weighted variance of t_i; W = f_max T_eff."""
    t = np.asarray(t, dtype=np.float64)
    w = np.asarray(w, dtype=np.float64)
    mean = np.sum(w * t) / np.sum(w)
    var = np.sum(w * (t - mean) ** 2) / np.sum(w)
    T_eff = float(np.sqrt(4.0 * np.pi * var))
    return T_eff, f_max * T_eff


def sinusoid_base(t, freqs):
    """PAPER.md:56 (eq. 2) with fixed frequencies: rows 1, cos 2 pi f_j t, sin 2 pi f_j t."""
    t = np.asarray(t, dtype=np.float64)
    rows = [np.ones_like(t)]
    for f in freqs:
        # the rounded product alone would lose the low bits of large phases: reduce exactly
        hi = f * t
        lo = np.array([_fma_residual(float(f), float(ti), float(h)) for ti, h in zip(t, hi)])
        ph = 2.0 * np.pi * ((hi - np.rint(hi)) + lo)
        rows.append(np.cos(ph))
        rows.append(np.sin(ph))
    return np.stack(rows)


def _fma_residual(a: float, b: float, hi: float) -> float:
    """a*b - hi exactly, in rational arithmetic (Python floats have no fma before 3.13)."""
    from fractions import Fraction
    return float(Fraction(a) * Fraction(b) - Fraction(hi))


def _grid_frequency(f0: float, df: float, k: int) -> float:
    """The double nearest f0 + k df (reading S1), as the C oracle's fma(k, df, f0)."""
    from fractions import Fraction
    return float(Fraction(k) * Fraction(df) + Fraction(f0))


def phase1(t, x, w, f0, df, K, fap0=0.05, fap1_thr=0.1, A1=1.0, max_base=10, k_peaks=32, pool_cap=None,
           threads: int = 0, refine_base: bool = False, refine_iter: int = 20, refine_tol: float = 1e-9):
    """PAPER.md:199-210 (section 4.2).  Returns dict(pool_idx, pool_z, pool_fap, base_idx, base_freqs).

    refine_base (reading P5): "adding to the base model the frequency corresponding to
    the largest peak" taken as the paper's own fit of such a model -- after the peak's grid
    frequency has joined the base, ALL base frequencies are refitted together by the local multifrequency
    fit of eq. 17 (`refine` below), and the next residual periodogram uses the refitted,
    off-grid frequencies.  Without it a signal up to df/2 off the grid leaves a residue that re-enters the
    base at the neighbouring grid point.  base_idx stays the grid index of each iteration's top peak;
    base_freqs are the frequencies the base ends with.  If the local fit fails (singular normal equations)
    the unrefined frequencies are kept for that iteration."""
    t = np.asarray(t, dtype=np.float64)
    N = t.shape[0]
    pool_cap = max(1, N // 10) if pool_cap is None else pool_cap
    f_max = f0 + df * (K - 1)
    _, W = bandwidth(t, w, f_max)
    base_f, base_idx, pool = [], [], {}
    for m in range(max_base):
        d = 2 * m + 1
        N_H = N - 3 * (m + 1) - 1
        if N_H <= 0 or N < d + 3:
            break
        base = sinusoid_base(t, base_f)
        dchi2 = _scan(t, x, w, base, f0, df, K, threads=threads)  # "single-frequency residual periodogram"
        l_base = _chi2_base(t, x, w, base)
        idx, count = _topk(dchi2, k_peaks)
        if count == 0 or not l_base > 0.0:
            break
        z = zstat(dchi2[idx[:count]], l_base, N_H)
        fap = fap1(z, W, A1)
        if fap[0] > fap0:
            break
        for j in range(count):
            if j == 0 or (fap[j] < fap1_thr and z[j] >= 0.5 * z[0]):
                i = int(idx[j])
                if i not in pool or fap[j] < pool[i][1]:
                    pool[i] = (float(z[j]), float(fap[j]))
        base_idx.append(int(idx[0]))                            # "adding to the base model the frequency
        base_f.append(_grid_frequency(f0, df, int(idx[0])))     #  corresponding to the largest peak"
        if refine_base and N >= 3 * len(base_f) + 2:
            try:
                base_f = [float(f) for f in refine(t, x, w, base_f, max_iter=refine_iter, tol=refine_tol)[0]]
            except np.linalg.LinAlgError:
                pass
    entries = sorted(pool.items(), key=lambda kv: (kv[1][1], kv[0]))
    entries = entries[:min(N // 10, pool_cap)]
    return {"pool_idx": np.array([e[0] for e in entries], dtype=np.int64),
            "pool_z": np.array([e[1][0] for e in entries]), "pool_fap": np.array([e[1][1] for e in entries]),
            "base_idx": np.array(base_idx, dtype=np.int64), "base_freqs": np.array(base_f, dtype=np.float64)}


def subset_fits(t, x, w, freqs, tau: float = 1e-10, masks=None, return_pivots: bool = False):
    """PAPER.md:158-175 (section 3) for every subset of the pool `freqs` (the 2^n - 1
    fits of phase 2, here with the frequencies held fixed: l_m(f') of eq. 7):
    g and Q of eqs. 15-16 summed directly, Cholesky Q = L L^T, a = L^{-1} g by forward substitution,
    l = D - |a|^2 (reading G2).  A column whose pivot^2 <= tau * (its diagonal) is dropped (reading S6).
    Returns l[mask], mask = 0 .. 2^n - 1, bit j selecting freqs[j] (or only for the given masks); with
    return_pivots also the smallest relative pivot^2 / diagonal of each fit (0 when a column was dropped):
    a diagnostic of the conditioning, about eps / pivot of D is lost to rounding on any FP64 path."""
    t, x, w = (np.asarray(a, dtype=np.float64) for a in (t, x, w))
    n = len(freqs)
    Phi = sinusoid_base(t, freqs)                       # rows 1, cos w_1 t, sin w_1 t, ...
    Q = np.array([[np.sum(w * Phi[a] * Phi[b]) for b in range(2 * n + 1)] for a in range(2 * n + 1)])
    g = np.array([np.sum(w * x * Phi[a]) for a in range(2 * n + 1)])
    D = np.sum(w * x * x)
    masks = range(1 << n) if masks is None else [int(m) for m in masks]
    out = np.empty(len(masks))
    pmin = np.ones(len(masks))
    for pos, mask in enumerate(masks):
        idx = [0] + [c for j in range(n) if (mask >> j) & 1 for c in (2 * j + 1, 2 * j + 2)]
        m = len(idx)
        L = np.zeros((m, m))
        a = np.zeros(m)
        for i in range(m):                              # row i of L and entry i of a = L^{-1} g
            for k in range(i):
                if L[k, k] > 0.0:
                    L[i, k] = (Q[idx[i], idx[k]] - L[i, :k] @ L[k, :k]) / L[k, k]
            piv2 = Q[idx[i], idx[i]] - L[i, :i] @ L[i, :i]
            if piv2 > tau * Q[idx[i], idx[i]]:
                L[i, i] = np.sqrt(piv2)
                a[i] = (g[idx[i]] - L[i, :i] @ a[:i]) / L[i, i]
                pmin[pos] = min(pmin[pos], piv2 / Q[idx[i], idx[i]])
            else:
                pmin[pos] = 0.0
        out[pos] = max(D - a @ a, 0.0)
    return (out, pmin) if return_pivots else out


def refine(t, x, w, freqs, max_iter: int = 20, tol: float = 1e-9):
    """PAPER.md:177-185 (section 3, eq. 17): the local multifrequency fit.  Each iteration: exact linear
    fit of theta at the current frequencies (eq. 14: Q = L L^T, a = L^{-1} g, theta = L^{-T} a), then the
    quadratic model of chi2 in xi = (theta, f) around (theta*, f): gradient g_f = <(x - mu) J> (its theta
    part is zero), matrix Q_f = <J J^T> with J = (model functions, d mu/d f_k) (its leading block is Q),
    step Q_f^{-1} g_f, frequencies updated; a last linear fit gives l_{n,loc}.  Times centred on their
    weighted mean.  Readings R1, R2: |step| <= 0.5 / T_eff; stop when
    max |step| T_eff <= tol.  Returns (freqs, l, iterations)."""
    t, x, w = (np.asarray(a, dtype=np.float64) for a in (t, x, w))
    f = np.array(freqs, dtype=np.float64, copy=True)
    n = f.size
    t0 = np.sum(w * t) / np.sum(w)
    tc = t - t0
    T_eff, _ = bandwidth(t, w, 1.0)
    D = np.sum(w * x * x)
    iters, converged = 0, max_iter == 0
    while True:
        Phi = sinusoid_base(tc, f)
        Q = (Phi * w) @ Phi.T
        g = (Phi * w) @ x
        L = np.linalg.cholesky(Q)
        a = _forward(L, g)
        theta = _forward(L.T[::-1, ::-1], a[::-1])[::-1]          # back substitution
        l = D - a @ a
        if converged or iters == max_iter:
            return f, max(float(l), 0.0), iters
        dmu = np.stack([2.0 * np.pi * tc * (-theta[2 * k + 1] * Phi[2 * k + 2] + theta[2 * k + 2] * Phi[2 * k + 1])
                        for k in range(n)])
        J = np.vstack([Phi, dmu])
        Qf = (J * w) @ J.T
        gf = (J * w) @ (x - theta @ Phi)
        Lf = np.linalg.cholesky(Qf)
        af = _forward(Lf, gf)
        step = _forward(Lf.T[::-1, ::-1], af[::-1])[::-1]
        df = np.clip(step[2 * n + 1:], -0.5 / T_eff, 0.5 / T_eff)
        f = f + df
        iters += 1
        converged = np.max(np.abs(df)) * T_eff <= tol


def _forward(L, b):
    """Solves L y = b for lower-triangular L by forward substitution."""
    y = np.zeros_like(b, dtype=np.float64)
    for i in range(b.size):
        y[i] = (b[i] - L[i, :i] @ y[:i]) / L[i, i]
    return y
