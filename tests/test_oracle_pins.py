"""Pins for the CPU oracle (oracle/oracle_fredec.c): it is checked against what the paper
and the mathematics fix, never against itself or the CUDA path.

Pin                                   | catches
--------------------------------------+-------------------------------------------------
QR least squares on tiny inputs       | wrong definition of z (G1, G2, S4), dropped term
FFT closed form (even spacing)        | sums, normalisation, factor 2, frequency units
scipy.signal.lombscargle (d = 0, 1)   | weights, floating mean, cos/sin cross term
mpmath 50 digits, large phases        | range reduction, rounding budget
invariants (i)-(viii), SURVEY 8(c)    | sign/index/transposition errors, singular rule
alias example of PAPER.md:294         | qualitative behaviour the paper prints
"""
import numpy as np
import pytest

from paper_1309_0100_b200 import inputs

TWO_PI = 2.0 * np.pi


def lstsq_chi2_drop(t, x, w, base, freqs):
    """Definition of z written with Householder-QR/SVD least squares (numpy.linalg.lstsq)
    on sqrt(w)-scaled design matrices: chi2_min(base) - chi2_min(base + cos + sin).
    PAPER.md:67 (eq. 4), :72 (eq. 5), :106 (eq. 10, n = 1)."""
    sw = np.sqrt(w)
    A0 = (base * sw).T if base is not None and base.shape[0] else np.zeros((t.size, 0))

    def chi2_min(A):
        if A.shape[1] == 0:
            return float(np.sum(w * x * x))
        theta = np.linalg.lstsq(A, sw * x, rcond=None)[0]
        r = sw * x - A @ theta
        return float(r @ r)

    base_chi2 = chi2_min(A0)
    out = np.empty(len(freqs))
    for j, f in enumerate(freqs):
        A1 = np.column_stack([A0, sw * np.cos(TWO_PI * f * t), sw * np.sin(TWO_PI * f * t)])
        out[j] = base_chi2 - chi2_min(A1)
    return out, base_chi2


def grid_frequencies(f0, df, K):
    """S1: the grid frequency is the double nearest to the real number f0 + k*df (one
    rounding, what fma(k, df, f0) returns); computed here with exact rationals."""
    from fractions import Fraction
    return np.array([float(Fraction(k) * Fraction(float(df)) + Fraction(float(f0))) for k in range(K)])


# ------------------------------------------------------------------ brute force (QR)
@pytest.mark.parametrize("d", [0, 1, 2, 5])
@pytest.mark.parametrize("N", [12, 50])
def test_z_is_qr_chi2_drop(oracle_mod, d, N):
    t, x, w, base = inputs.random_series(100 + 10 * d + N, N, d)
    f0, df, K = 0.013, 0.0037, 100
    z = oracle_mod.scan(t, x, w, base, f0, df, K)
    f = f0 + df * np.arange(K)
    zb, chi2b = lstsq_chi2_drop(t, x, w, base, f)
    assert np.max(np.abs(z - zb)) <= 1e-12 * chi2b
    assert abs(oracle_mod.chi2_base(t, x, w, base) - chi2b) <= 1e-12 * chi2b


def test_z_is_qr_chi2_drop_sinusoid_base(oracle_mod):
    """Base = offset + two accepted sinusoids (the residual periodogram of PAPER.md:201)."""
    rng = np.random.Generator(np.random.PCG64(7))
    N = 60
    t = np.sort(rng.uniform(0, 50, N))
    w = 1.0 / rng.uniform(0.5, 2, N) ** 2
    x = 3 * np.cos(TWO_PI * t / 4.1) + np.sin(TWO_PI * t / 9.7) + rng.normal(0, 1, N)
    base = inputs.base_offset_sinusoids(t, [4.1, 9.7])
    f0, df, K = 0.0113, 0.0071, 80   # never closer than ~1e-3 cycles/span to a base frequency
    z = oracle_mod.scan(t, x, w, base, f0, df, K)
    zb, chi2b = lstsq_chi2_drop(t, x, w, base, f0 + df * np.arange(K))
    assert np.max(np.abs(z - zb)) <= 1e-11 * chi2b


# ------------------------------------------------------------------ FFT closed form
@pytest.mark.parametrize("N", [64, 101])
def test_even_spacing_fourier_frequencies(oracle_mod, N):
    """Unit weights, evenly spaced times, base = offset, Fourier frequencies m/(N dt),
    0 < m < N/2: cos, sin and 1 are mutually orthogonal with <cos^2> = <sin^2> = N/2, so
    z = (2/N) |FFT(x)_m|^2  (Schuster periodogram)."""
    rng = np.random.Generator(np.random.PCG64(N))
    dt = 0.25
    t = dt * np.arange(N)
    x = rng.normal(0, 1, N) + 0.5 * np.cos(TWO_PI * 3 * t / (N * dt))
    w = np.ones(N)
    df = 1.0 / (N * dt)
    K = (N - 1) // 2
    z = oracle_mod.scan(t, x, w, inputs.base_offset(t), df, df, K)   # f = m*df, m = 1..K
    X = np.fft.fft(x)
    expect = (2.0 / N) * np.abs(X[1:K + 1]) ** 2
    assert np.max(np.abs(z - expect)) <= 1e-12 * np.max(expect)


def test_even_spacing_alias_symmetry(oracle_mod):
    """(viii) evenly spaced times: z(f) = z(1/dt - f)."""
    rng = np.random.Generator(np.random.PCG64(5))
    N, dt = 80, 0.5
    t = dt * np.arange(N)
    x = rng.normal(0, 1, N)
    w = 1.0 / rng.uniform(0.5, 2, N) ** 2
    base = inputs.base_offset(t)
    f = 0.013 + 0.009 * np.arange(60)
    za = np.array([oracle_mod.scan(t, x, w, base, ff, 1.0, 1)[0] for ff in f])
    zb = np.array([oracle_mod.scan(t, x, w, base, 1.0 / dt - ff, 1.0, 1)[0] for ff in f])
    assert np.max(np.abs(za - zb)) <= 1e-11 * np.max(za)


# ------------------------------------------------------------------ installed library
@pytest.mark.parametrize("d", [0, 1])
def test_against_scipy_lombscargle(oracle_mod, d):
    """d = 0 / d = 1 with arbitrary times and weights is the (floating-mean) weighted
    Lomb-Scargle periodogram: scipy's normalised power = z / chi2_base."""
    from scipy.signal import lombscargle
    t, x, w, base = inputs.random_series(42 + d, 300, 1)
    base = base if d else None
    f0, df, K = 0.002, 0.0011, 400
    z = oracle_mod.scan(t, x, w, base, f0, df, K)
    chi2b = oracle_mod.chi2_base(t, x, w, base)
    f = f0 + df * np.arange(K)
    p = lombscargle(t, x, TWO_PI * f, weights=w, floating_mean=bool(d), normalize="normalize")
    assert np.max(np.abs(z / chi2b - p)) <= 1e-12


# ------------------------------------------------------------------ exact value (mpmath)
def _mp_chi2_drop(t, x, w, base, freqs, digits=50):
    import mpmath as mp
    mp.mp.dps = digits
    N = len(t)
    tt = [mp.mpf(float(v)) for v in t]
    xx = [mp.mpf(float(v)) for v in x]
    ww = [mp.mpf(float(v)) for v in w]
    cols0 = [[mp.mpf(float(v)) for v in row] for row in base]

    def chi2_min(cols):
        if not cols:
            return mp.fsum(ww[i] * xx[i] ** 2 for i in range(N))
        n = len(cols)
        Q = mp.matrix(n, n)
        g = mp.matrix(n, 1)
        for a in range(n):
            g[a] = mp.fsum(ww[i] * xx[i] * cols[a][i] for i in range(N))
            for b in range(n):
                Q[a, b] = mp.fsum(ww[i] * cols[a][i] * cols[b][i] for i in range(N))
        theta = mp.lu_solve(Q, g)
        return mp.fsum(ww[i] * (xx[i] - mp.fsum(theta[a] * cols[a][i] for a in range(n))) ** 2
                       for i in range(N))

    c0 = chi2_min(cols0)
    out = []
    for f in freqs:
        ff = mp.mpf(float(f))
        c = [mp.cos(2 * mp.pi * ff * tt[i]) for i in range(N)]
        s = [mp.sin(2 * mp.pi * ff * tt[i]) for i in range(N)]
        out.append(float(c0 - chi2_min(cols0 + [c, s])))
    return np.array(out), float(c0)


@pytest.mark.parametrize("d,t_span,f0,df", [(1, 30.0, 0.05, 0.013), (2, 1.0e4, 4.3, 0.0137)])
def test_against_mpmath_50_digits(oracle_mod, d, t_span, f0, df):
    """Bounds the oracle's absolute error, including large phases (t up to 1e4, f ~ 5:
    5e4 turns, where a naive sin(2 pi f t) already loses ~1e-11)."""
    N, K = 18, 40
    t, x, w, base = inputs.random_series(900 + d, N, d, t_span=t_span)
    z = oracle_mod.scan(t, x, w, base, f0, df, K)
    f = grid_frequencies(f0, df, K)
    zmp, chi2b = _mp_chi2_drop(t, x, w, base, f)
    assert np.max(np.abs(z - zmp)) <= 1e-12 * chi2b
    zl = oracle_mod.scan(t, x, w, base, f0, df, K, long_double=True)
    assert np.max(np.abs(z - zl)) <= 1e-12 * chi2b


def test_long_double_build_agrees_on_tiny_config(oracle_mod):
    wl = inputs.config(1, K=2000)
    t, x, w, base = wl.series(0)
    z = oracle_mod.scan(t, x, w, base, wl.f0, wl.df, wl.K)
    zl = oracle_mod.scan(t, x, w, base, wl.f0, wl.df, wl.K, long_double=True)
    assert np.max(np.abs(z - zl)) <= 1e-12 * np.max(zl)


# ------------------------------------------------------------------ invariants
def test_noiseless_sinusoid_peaks_at_true_frequency(oracle_mod):
    """(i) x = c0 + A cos(2 pi f* t + phi), f* on the grid, base contains the constant:
    the alternative model fits exactly, so z(f*) = chi2_base and argmax = index of f*."""
    rng = np.random.Generator(np.random.PCG64(11))
    N = 150
    t = np.sort(rng.uniform(0, 200, N))
    w = 1.0 / rng.uniform(0.5, 2, N) ** 2
    f0, df, K, kstar = 0.01, 0.0005, 400, 137
    fstar = float(np.float64(kstar) * df + f0)
    x = 1.7 + 2.5 * np.cos(TWO_PI * fstar * t + 0.9)
    base = inputs.base_offset(t)
    z = oracle_mod.scan(t, x, w, base, f0, df, K)
    chi2b = oracle_mod.chi2_base(t, x, w, base)
    assert int(np.argmax(z)) == kstar
    assert abs(z[kstar] - chi2b) <= 1e-9 * chi2b     # limited by fl(f*) vs fma rounding
    idx, cnt = oracle_mod.topk(z, 3)
    assert idx[0] == kstar


@pytest.mark.parametrize("cfg,kw", [(1, dict(K=3000)), (2, dict(K=3000)), (3, dict(K=1500))])
def test_bounds_0_le_z_le_chi2_base(oracle_mod, cfg, kw):
    """(ii) 0 <= z <= chi2_base (nested models)."""
    wl = inputs.config(cfg, **kw)
    t, x, w, base = wl.series(0)
    z = oracle_mod.scan(t, x, w, base, wl.f0, wl.df, wl.K)
    chi2b = oracle_mod.chi2_base(t, x, w, base)
    assert np.all(np.isfinite(z)) and z.min() >= 0.0 and z.max() <= chi2b * (1 + 1e-12)


def test_time_origin_invariance(oracle_mod):
    """(iii) t -> t + t0 with the base re-evaluated leaves z unchanged (S10; the paper
    itself shifts to <t> = 0)."""
    t, x, w, _ = inputs.random_series(3, 200, 0)
    f0, df, K = 0.01, 0.002, 300
    t0 = 12345.678
    za = oracle_mod.scan(t, x, w, inputs.base_offset_trend(t), f0, df, K)
    zb = oracle_mod.scan(t + t0, x, w, inputs.base_offset_trend(t + t0), f0, df, K)
    assert np.max(np.abs(za - zb)) <= 1e-10 * np.max(za)


def test_base_reparametrisation_invariance(oracle_mod):
    """(iv) base_funcs -> M base_funcs with M invertible spans the same model."""
    t, x, w, base = inputs.random_series(4, 120, 3)
    M = np.array([[2.0, 0.3, -1.0], [0.0, -1.5, 0.4], [0.7, 0.0, 1.1]])
    f0, df, K = 0.02, 0.003, 200
    za = oracle_mod.scan(t, x, w, base, f0, df, K)
    zb = oracle_mod.scan(t, x, w, M @ base, f0, df, K)
    assert np.max(np.abs(za - zb)) <= 1e-11 * np.max(za)


def test_scale_covariance(oracle_mod):
    """(v) x -> alpha x gives z -> alpha^2 z; w -> beta w gives z -> beta z (S5)."""
    t, x, w, base = inputs.random_series(5, 100, 2)
    f0, df, K = 0.02, 0.003, 150
    z = oracle_mod.scan(t, x, w, base, f0, df, K)
    assert np.allclose(oracle_mod.scan(t, 4.0 * x, w, base, f0, df, K), 16.0 * z, rtol=1e-12, atol=0)
    assert np.allclose(oracle_mod.scan(t, x, 8.0 * w, base, f0, df, K), 8.0 * z, rtol=1e-12, atol=0)


def test_pure_cos_pure_sin_split(oracle_mod):
    """(vi)-like check on the quadratic part: with d = 0 and x = cos(2 pi f t) exactly on a
    grid point, the fit is exact: z = <x^2> (uses <cos^2> + <sin^2> = <1>)."""
    rng = np.random.Generator(np.random.PCG64(2))
    t = np.sort(rng.uniform(0, 40, 90))
    w = rng.uniform(0.5, 2, 90)
    f = 0.375
    for phase in (0.0, np.pi / 2, 1.0):
        x = np.cos(TWO_PI * f * t + phase)
        z = oracle_mod.scan(t, x, w, None, f, 1.0, 1)[0]
        assert abs(z - np.sum(w * x * x)) <= 1e-12 * np.sum(w)


def test_trial_frequency_in_base_gives_zero(oracle_mod):
    """(vii) S6: a trial frequency equal to a base frequency (or f = 0 with a constant in
    the base) adds nothing: z = 0, never NaN."""
    t, x, w, _ = inputs.random_series(6, 80, 0)
    P = 8.0
    base = inputs.base_offset_sinusoids(t, [P])
    z = oracle_mod.scan(t, x, w, base, 1.0 / P, 1.0, 1)
    assert z[0] == 0.0
    z = oracle_mod.scan(t, x, w, inputs.base_offset(t), 0.0, 0.01, 5)
    assert z[0] == 0.0 and np.all(np.isfinite(z)) and np.all(z[1:] > 0)
    # d = 0, f = 0: cos = 1 is a legitimate regressor, sin = 0 is dropped
    z = oracle_mod.scan(t, x, w, None, 0.0, 0.01, 2)
    assert abs(z[0] - np.sum(w * x) ** 2 / np.sum(w)) <= 1e-12 * np.sum(w * x * x)


def test_zero_weights_and_duplicates_allowed(oracle_mod):
    """S11: w_i = 0 rows drop out; duplicated times are fine."""
    t, x, w, base = inputs.random_series(8, 60, 1)
    t2 = np.concatenate([t, t[:5], [1e3, 2e3]])
    x2 = np.concatenate([x, x[:5], [1e6, -1e6]])
    w2 = np.concatenate([w, np.zeros(5), [0.0, 0.0]])
    za = oracle_mod.scan(t, x, w, base, 0.01, 0.004, 100)
    zb = oracle_mod.scan(t2, x2, w2, inputs.base_offset(t2), 0.01, 0.004, 100)
    assert np.max(np.abs(za - zb)) <= 1e-12 * np.max(za)


def test_singular_base_is_an_error(oracle_mod):
    t, x, w, _ = inputs.random_series(9, 30, 0)
    base = np.stack([np.ones_like(t), 2.0 * np.ones_like(t)])
    with pytest.raises(RuntimeError):
        oracle_mod.scan(t, x, w, base, 0.01, 0.01, 4)


def test_openmp_is_bit_identical_to_serial(oracle_mod):
    wl = inputs.config(3, K=400)
    t, x, w, base = wl.series(0)
    za = oracle_mod.scan(t, x, w, base, wl.f0, wl.df, wl.K, threads=1)
    zb = oracle_mod.scan(t, x, w, base, wl.f0, wl.df, wl.K, threads=0)
    assert np.array_equal(za, zb)


# ------------------------------------------------------------------ the paper's example
def test_alias_example_of_section_7_1(oracle_mod):
    """PAPER.md:294 (section 7.1): two equal sinusoids at 0.9 and 1.1 Hz observed with
    periodic gaps that alias at 0.1 Hz put the single-frequency maximum at the WRONG
    frequency 1.0 Hz, the true ones looking like side aliases, peaks at 1.0 +- 0.1 k.
    The Paper-I series itself is not available; tests/golden/alias_example.txt states the
    construction used here (own synthetic series of the same kind)."""
    import os
    cfg = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "alias_example.txt")) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                k, v = line.split("=")
                cfg[k.strip()] = float(v)
    period, window, dt = cfg["gap_period"], cfg["window"], cfg["dt"]
    n_per = int(round(window / dt))
    t = np.concatenate([m * period + dt * np.arange(n_per) for m in range(int(cfg["n_windows"]))])
    x = np.cos(TWO_PI * cfg["f_a"] * t) + np.cos(TWO_PI * cfg["f_b"] * t)
    w = np.ones_like(t)
    f0, df, K = 0.5, 0.001, 1001                       # 0.5 .. 1.5
    z = oracle_mod.scan(t, x, w, inputs.base_offset(t), f0, df, K)
    kmax = int(np.argmax(z))
    assert abs((f0 + df * kmax) - cfg["expected_argmax"]) <= 2 * df
    idx, cnt = oracle_mod.topk(z, 9)
    peaks = np.sort(f0 + df * idx[:cnt])
    for fa in (cfg["f_a"], cfg["f_b"]):                # the true frequencies are side peaks
        assert np.min(np.abs(peaks - fa)) <= 0.01
        assert z[int(round((fa - f0) / df))] < z[kmax]


# ------------------------------------------------------------------ top-k (S7)
@pytest.mark.parametrize("z,k,expect,count", [
    ([0, 1, 0, 3, 0, 2, 0], 3, [3, 5, 1], 3),                    # plain peaks, by height
    ([0, 1, 0, 3, 0, 2, 0], 5, [3, 5, 1, -1, -1], 3),            # fewer peaks than k
    ([5, 1, 0, 1, 7], 2, [4, 0], 2),                             # both edges eligible
    ([0, 2, 2, 2, 0, 2, 0], 4, [1, 5, -1, -1], 2),               # plateau -> lowest index; tie -> index asc
    ([1, 2, 3, 4, 5], 2, [4, -1], 1),                            # monotone up: right edge
    ([5, 4, 3, 2, 1], 2, [0, -1], 1),                            # monotone down: left edge
    ([3, 3, 3, 3], 2, [0, -1], 1),                               # all equal: plateau from the edge
    ([0, 4, 0, 4, 0, 4], 3, [1, 3, 5], 3),                       # exact ties ranked by index
    ([7], 1, [0], 1),                                            # K = 1
    ([0, float("nan"), 0, 1, 0], 2, [3, 0], 2),                  # NaN ranks as -inf, so z[0] = 0 is a (low) peak
])
def test_topk_hand_cases(oracle_mod, z, k, expect, count):
    idx, cnt = oracle_mod.topk(np.array(z, dtype=np.float64), k)
    assert cnt == count
    assert idx.tolist() == expect


def test_topk_config1_sanity(oracle_mod):
    """config 1's two strongest peaks sit at the injected periods 17.3 d and
    91 d, i.e. k ~ (1/17.3 - 1e-3)/1e-4 = 568 and k ~ (1/91 - 1e-3)/1e-4 = 100."""
    wl = inputs.config(1)
    z = oracle_mod.scan(*wl.series(0), wl.f0, wl.df, wl.K)
    idx, cnt = oracle_mod.topk(z, 10)
    assert cnt == 10 and abs(idx[0] - 568) <= 1 and abs(idx[1] - 100) <= 1
    assert np.all(np.diff(z[idx]) <= 0)


@pytest.mark.parametrize("seed,K", [(1, 3000), (2, 257), (3, 20_000)])
def test_topk_against_scipy_find_peaks(oracle_mod, seed, K):
    """oracle_topk against a library peak finder it shares nothing with: on an array without ties the peaks of
    reading S7 (z[i] > z[i-1] and z[i] >= z[i+1], outside = -infinity) are scipy.signal.find_peaks' strict
    interior maxima plus an end point that tops its one neighbour; the order is z descending; a k below the
    number of peaks keeps the k highest."""
    from scipy.signal import find_peaks
    rng = np.random.Generator(np.random.PCG64(1000 + seed))
    z = rng.standard_normal(K).cumsum() * 0.05 + rng.standard_normal(K)
    ref = set(find_peaks(z)[0].tolist())
    if z[0] >= z[1]:
        ref.add(0)
    if z[-1] > z[-2]:
        ref.add(K - 1)
    idx, cnt = oracle_mod.topk(z, K)
    got = idx[:cnt]
    assert cnt == len(ref) and set(got.tolist()) == ref and np.all(idx[cnt:] == -1)
    assert np.all(np.diff(z[got]) <= 0.0)
    k = max(1, cnt // 7)
    idx_k, cnt_k = oracle_mod.topk(z, k)
    assert cnt_k == k and idx_k.tolist() == got[:k].tolist()
    # ties: S7 takes the first point of a flat stretch reached by an ascent -- of a plateau that tops both sides
    # (find_peaks reports its middle) and, by the letter of the rule, also of a shelf on an ascending slope
    zp = np.round(z, 1)
    mid, props = find_peaks(zp, plateau_size=1)
    idx_p, cnt_p = oracle_mod.topk(zp, K)
    got_p = set(idx_p[:cnt_p].tolist())
    assert set(props["left_edges"].tolist()) <= got_p
    for i in got_p - set(props["left_edges"].tolist()) - {0, K - 1}:
        j = i
        while j + 1 < K and zp[j + 1] == zp[i]:
            j += 1
        assert zp[i - 1] < zp[i] and j > i and (j + 1 == K or zp[j + 1] > zp[i]), i   # a shelf, or a final plateau
    assert oracle_mod.topk(np.array([1.0, 2.0, 2.0, 3.0, 0.0]), 5)[0].tolist() == [3, 1, -1, -1, -1]
