"""Pins for oracle/phase1.py (statistic, FAP, bandwidth, phase-1 driver): checked against what
the paper and the mathematics fix, never against the CUDA path.

Pin                                         | catches
--------------------------------------------+-----------------------------------------------
(N_H/2) ln(l_base/l_alt) from two QR fits   | wrong ratio / sign / N_H in the statistic (G1)
closed-form T_eff for even spacing          | variance normalisation, factor 4 pi, weights
hand values of W e^-z sqrt z                | exponent sign, power of z, cap at 1
constructed series for phase 1              | stop rule, base order, half-height rule, N/10 cap
off-grid sinusoids, refine_base             | a refit that is skipped, applied to the wrong entry, or not fed back
"""
import numpy as np
import pytest

from paper_1309_0100_b200 import inputs

TWO_PI = 2.0 * np.pi


@pytest.fixture(scope="module")
def p1(oracle_mod):
    from oracle import phase1
    return phase1


def _lstsq_min(A, y):
    theta = np.linalg.lstsq(A, y, rcond=None)[0]
    r = y - A @ theta
    return float(r @ r)


def test_zstat_is_the_log_likelihood_ratio(oracle_mod, p1):
    """z = (N_H/2) ln(l_base/l_alt), both minima from Householder-QR fits."""
    t, x, w, base = inputs.random_series(11, 40, 3)
    f0, df, K = 0.013, 0.011, 25
    N, d = t.size, base.shape[0]
    N_H = N - d - 3
    sw = np.sqrt(w)
    A0 = (base * sw).T
    l_base = _lstsq_min(A0, sw * x)
    z_def = np.empty(K)
    for k in range(K):
        f = f0 + k * df
        A1 = np.column_stack([A0, sw * np.cos(TWO_PI * f * t), sw * np.sin(TWO_PI * f * t)])
        z_def[k] = 0.5 * N_H * np.log(l_base / _lstsq_min(A1, sw * x))
    dchi2 = oracle_mod.scan(t, x, w, base, f0, df, K)
    z = p1.zstat(dchi2, oracle_mod.chi2_base(t, x, w, base), N_H)
    assert np.max(np.abs(z - z_def)) <= 1e-10 * np.max(z_def)
    assert np.all(np.diff(p1.zstat(np.linspace(0.0, 0.99, 50), 1.0, 7.0)) > 0)   # monotone in dchi2
    assert p1.zstat(np.array([0.0]), 3.0, 9.0)[0] == 0.0


def test_bandwidth_closed_form(p1):
    """evenly spaced, equally weighted times t_i = i*Delta have variance
    Delta^2 (N^2 - 1)/12, so T_eff = Delta sqrt(pi (N^2 - 1)/3); f_max scales W linearly."""
    N, delta = 101, 0.37
    t = 5.0 + delta * np.arange(N)
    T_eff, W = p1.bandwidth(t, np.full(N, 2.5), 3.0)
    assert abs(T_eff - delta * np.sqrt(np.pi * (N * N - 1) / 3.0)) <= 1e-12 * T_eff
    assert abs(W - 3.0 * T_eff) <= 1e-15 * W
    # a weight of 2 is the same as observing that epoch twice
    rng = np.random.Generator(np.random.PCG64(3))
    tt = rng.uniform(0, 50, 30)
    ww = np.ones(30)
    ww[[3, 17]] = 2.0
    T_a, _ = p1.bandwidth(tt, ww, 1.0)
    T_b, _ = p1.bandwidth(np.concatenate([tt, tt[[3, 17]]]), np.ones(32), 1.0)
    assert abs(T_a - T_b) <= 1e-13 * T_a
    # dense uniform coverage of [0, T]: T_eff -> T sqrt(pi/3)
    T_c, _ = p1.bandwidth(np.linspace(0.0, 10.0, 200001), np.ones(200001), 1.0)
    assert abs(T_c / 10.0 - np.sqrt(np.pi / 3.0)) < 1e-5


def test_fap1_hand_values(p1):
    """PAPER.md:143 (eq. 13), n = 1: A W e^-z z^(1/2)."""
    fap = p1.fap1(np.array([1.0, 4.0, 9.0, 0.25, 0.0, -1.0]), 10.0, 1.0)
    assert abs(fap[1] - 10.0 * np.exp(-4.0) * 2.0) < 1e-15
    assert abs(fap[2] - 10.0 * np.exp(-9.0) * 3.0) < 1e-17
    assert fap[0] == 1.0 and fap[3] == 1.0          # 10 e^-1 = 3.68 and 10 e^-.25 / 2 = 3.89 are capped
    assert fap[4] == 1.0 and fap[5] == 1.0          # no improvement: no significance
    assert abs(p1.fap1(np.array([1.0]), 1.0, 1.0)[0] - np.exp(-1.0)) < 1e-16
    assert abs(p1.fap1(np.array([4.0]), 10.0, 0.5)[0] - 0.5 * fap[1]) < 1e-16
    z = np.linspace(0.6, 30, 200)
    assert np.all(np.diff(p1.fap1(z, 1.0)) < 0)     # decreasing beyond the maximum at z = 1/2


def _two_sinusoids(N=120, K=4000, noise=0.05, seed=5):
    rng = np.random.Generator(np.random.PCG64(seed))
    t = np.sort(rng.uniform(0.0, 200.0, N))
    f0, df = 0.002, 0.00025
    k1, k2 = 1213, 2790                              # grid frequencies 0.30525 and 0.6995
    x = (3.0 * np.sin(TWO_PI * (f0 + k1 * df) * t + 0.3) + 1.2 * np.cos(TWO_PI * (f0 + k2 * df) * t)
         + 0.7 + noise * rng.standard_normal(N))
    return t, x, np.full(N, 1.0 / noise ** 2), f0, df, K, k1, k2


def test_phase1_finds_two_grid_sinusoids_then_stops(p1):
    """the strongest variation first, then the next, then the residual
    periodogram is noise and its top FAP exceeds FAP_0.  With the signals ON the grid the base
    model removes them exactly, so the outcome is fixed by the rules."""
    t, x, w, f0, df, K, k1, k2 = _two_sinusoids()
    r = p1.phase1(t, x, w, f0, df, K, fap0=0.01, fap1_thr=0.02, max_base=6, k_peaks=20)
    assert r["base_idx"].tolist() == [k1, k2]
    assert set([k1, k2]) <= set(r["pool_idx"].tolist())
    assert np.all(np.diff(r["pool_fap"]) >= 0)                       # sorted by FAP
    assert np.all(r["pool_fap"] < 0.02)
    assert len(r["pool_idx"]) <= t.size // 10
    # max_base cuts the SLICK loop short
    r1 = p1.phase1(t, x, w, f0, df, K, fap0=0.01, fap1_thr=0.02, max_base=1, k_peaks=20)
    assert r1["base_idx"].tolist() == [k1]


def _two_off_grid_sinusoids(N=150, K=4000, noise=1e-7, seed=8):
    rng = np.random.Generator(np.random.PCG64(seed))
    t = np.sort(rng.uniform(0.0, 200.0, N))
    f0, df = 0.002, 0.00025
    fa, fb = f0 + 1213.41 * df, f0 + 2790.47 * df    # 0.41 and 0.47 of a grid step off the grid
    x = (3.0 * np.sin(TWO_PI * fa * t + 0.3) + 1.2 * np.cos(TWO_PI * fb * t) + 0.7
         + noise * rng.standard_normal(N))
    return t, x, np.full(N, 1.0 / noise ** 2), f0, df, K, fa, fb


def test_phase1_refined_base_holds_each_off_grid_signal_once(p1):
    """PAPER.md:201 + :177-185 (reading P5): two sinusoids BETWEEN grid points, almost no noise.  With the
    base refitted after every addition the base ends with exactly the two true frequencies (to 1e-6 / T; the
    noise allows ~1e-8 / T) and the third periodogram is noise.  The grid-only mode, on the same series, keeps
    finding the residue the mis-tuned base leaves behind -- which is why the refit matters."""
    t, x, w, f0, df, K, fa, fb = _two_off_grid_sinusoids()
    T = t.max() - t.min()
    r = p1.phase1(t, x, w, f0, df, K, fap0=0.01, fap1_thr=0.02, max_base=6, k_peaks=20, refine_base=True)
    assert r["base_idx"].tolist() == [1213, 2790]                 # the peaks' grid points, strongest first
    assert r["base_freqs"].shape == (2,)
    assert np.max(np.abs(r["base_freqs"] - np.array([fa, fb]))) <= 1e-6 / T
    assert {1213, 2790} <= set(r["pool_idx"].tolist())
    grid_only = p1.phase1(t, x, w, f0, df, K, fap0=0.01, fap1_thr=0.02, max_base=6, k_peaks=20)
    assert len(grid_only["base_idx"]) > 2
    assert np.array_equal(grid_only["base_freqs"], f0 + df * grid_only["base_idx"])
    # one iteration only: the refit of a single frequency against the second, unmodelled signal
    r1 = p1.phase1(t, x, w, f0, df, K, fap0=0.01, fap1_thr=0.02, max_base=1, k_peaks=20, refine_base=True)
    assert r1["base_idx"].tolist() == [1213] and abs(r1["base_freqs"][0] - fa) <= 0.05 / T


def test_phase1_refined_on_the_rv_like_series(p1):
    """The config-2 series carries five sinusoids (inputs.RV_PERIODS).  Grid-only phase 1 enters two of them
    twice, at neighbouring grid points; with the refit the base holds five frequencies, no two of them
    adjacent on the grid, each within a tenth of a cycle over the span of an injected one."""
    wl = inputs.config(2)
    t, x, w, _ = wl.series(0)
    T = t.max() - t.min()
    r = p1.phase1(t, x, w, wl.f0, wl.df, wl.K, max_base=10, k_peaks=32, refine_base=True)
    bi = np.sort(r["base_idx"])
    assert len(bi) == 5 and np.all(np.diff(bi) > 1)
    true_f = 1.0 / np.array(inputs.RV_PERIODS)
    for f in r["base_freqs"]:
        assert np.min(np.abs(true_f - f)) <= 0.1 / T
    grid_only = p1.phase1(t, x, w, wl.f0, wl.df, wl.K, max_base=10, k_peaks=32)
    assert np.any(np.diff(np.sort(grid_only["base_idx"])) == 1)   # the duplicates the refit removes


def test_phase1_half_height_rule_and_pool_cap(p1):
    """side peaks below half of the highest do not enter the pool even when their
    FAP is tiny; the pool keeps at most N/10 entries, those of smallest FAP."""
    t, x, w, f0, df, K, k1, k2 = _two_sinusoids(noise=0.01)
    r = p1.phase1(t, x, w, f0, df, K, fap0=0.01, fap1_thr=0.02, max_base=1, k_peaks=50)
    # one periodogram only: the second sinusoid (amplitude 1.2 vs 3: a sixth of the power) is hugely
    # significant but far below half of the top peak's statistic, so it must be absent
    assert k2 not in r["pool_idx"].tolist() and r["pool_idx"][0] == k1
    full = p1.phase1(t, x, w, f0, df, K, fap0=0.01, fap1_thr=0.02, max_base=6, k_peaks=50)
    cut = p1.phase1(t[:40], x[:40], w[:40], f0, df, K, fap0=0.01, fap1_thr=0.02, max_base=6, k_peaks=50)
    assert len(cut["pool_idx"]) <= 4 and len(full["pool_idx"]) <= 12
    capped = p1.phase1(t, x, w, f0, df, K, fap0=0.01, fap1_thr=0.02, max_base=6, k_peaks=50, pool_cap=1)
    assert capped["pool_idx"].tolist() == full["pool_idx"][:1].tolist()


def test_phase1_white_noise_has_empty_pool(p1):
    """when even the highest peak is not significant nothing is collected."""
    rng = np.random.Generator(np.random.PCG64(12))
    t = np.sort(rng.uniform(0.0, 100.0, 80))
    x = rng.standard_normal(80)
    r = p1.phase1(t, x, np.ones(80), 0.005, 0.001, 2000, fap0=0.01, fap1_thr=0.02)
    assert r["base_idx"].size == 0 and r["pool_idx"].size == 0
