"""GPU parity of the statistic, FAP, bandwidth and phase-1 entry points
against oracle/phase1.py, through the C-ABI binding.  Integer results (grid indices, counts)
must be identical; floating point within 1e-12 relative (element-wise maps: a handful of
correctly rounded operations) and 1e-9 relative for statistics derived from a scan."""
import os

import numpy as np
import pytest

from paper_1309_0100_b200 import inputs

pytestmark = pytest.mark.gpu
TWO_PI = 2.0 * np.pi


@pytest.fixture(scope="module")
def fr():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1309_0100_b200 import build
    build.build()
    import paper_1309_0100_b200 as fr
    fr.lib()
    return fr


@pytest.fixture(scope="module")
def p1(oracle_mod):
    from oracle import phase1
    return phase1


@pytest.mark.parametrize("K", [1, 7, 1000, 300_001])
def test_zstat_and_fap1_elementwise(fr, p1, K):
    import torch
    rng = np.random.Generator(np.random.PCG64(K))
    chi2 = 123.456
    dchi2 = chi2 * rng.uniform(0.0, 0.999, K)
    dchi2[0] = 0.0
    z_ref = p1.zstat(dchi2, chi2, 57.0)
    z = fr.fredec_zstat(dchi2, chi2, 57.0)                               # host pointers
    assert np.max(np.abs(z - z_ref)) <= 1e-12 * np.max(z_ref) + 1e-300
    zd = fr.fredec_zstat(torch.from_numpy(dchi2).cuda(), chi2, 57.0)     # device pointers
    assert np.array_equal(zd.cpu().numpy(), z)
    fap_ref = p1.fap1(z, 35.5, 0.8)                                     # the same z on both sides
    fap = fr.fredec_fap1(z, 35.5, 0.8)
    assert np.all(np.abs(fap - fap_ref) <= 1e-13 * fap_ref + 1e-300)       # exp, sqrt: a few ulp
    assert fap[0] == 1.0 and np.all(fap <= 1.0) and np.all(fap >= 0.0)


def test_zstat_perfect_fit_is_inf(fr):
    z = fr.fredec_zstat(np.array([5.0, 2.5]), 5.0, 10.0)
    assert np.isinf(z[0]) and z[0] > 0 and abs(z[1] - 5.0 * np.log(2.0)) < 1e-14


def test_bandwidth_parity(fr, p1):
    for cfg in (1, 2, 4):
        wl = inputs.config(cfg)
        t, x, w, _ = wl.series(0)
        f_max = wl.f0 + wl.df * (wl.K - 1)
        T_ref, W_ref = p1.bandwidth(t, w, f_max)
        T, W = fr.fredec_bandwidth(t, w, f_max)
        assert abs(T - T_ref) <= 1e-12 * T_ref and abs(W - W_ref) <= 1e-12 * W_ref


def _assert_phase1_equal(r, ref):
    assert r["base_idx"].tolist() == ref["base_idx"].tolist()
    assert r["pool_idx"].tolist() == ref["pool_idx"].tolist()
    assert np.all(np.abs(r["pool_z"] - ref["pool_z"]) <= 1e-9 * np.abs(ref["pool_z"]))
    assert np.all(np.abs(r["pool_fap"] - ref["pool_fap"]) <= 1e-7 * ref["pool_fap"] + 1e-300)


def test_phase1_rv_like_series(fr, p1):
    """Config-2 shaped series (seasonal gaps, five sinusoids): several SLICK iterations with alias
    side peaks; pool and base frequencies identical to the oracle's."""
    wl = inputs.config(2, N=400, K=40_000)
    t, x, w, _ = wl.series(0)
    kw = dict(fap0=0.05, fap1=0.1, A1=1.0, max_base=8, k_peaks=24)
    ref = p1.phase1(t, x, w, wl.f0, wl.df, wl.K, fap0=0.05, fap1_thr=0.1, A1=1.0, max_base=8, k_peaks=24)
    r = fr.fredec_phase1(t, x, w, wl.f0, wl.df, wl.K, **kw)
    assert len(ref["base_idx"]) >= 2
    _assert_phase1_equal(r, ref)
    import torch
    rd = fr.fredec_phase1(*[torch.from_numpy(a).cuda() for a in (t, x, w)], wl.f0, wl.df, wl.K, **kw)
    _assert_phase1_equal(rd, r)


def _assert_refined_equal(r, ref, T_eff, tol):
    """Both sides stop their Gauss-Newton when the last step is below tol cycles over T_eff, so the refitted
    frequencies agree to a few tol; the periodograms that follow depend smoothly on them: the discrete
    outcome (which peaks, in which order) must be identical, the statistics agree to 1e-7 relative and the
    FAPs, proportional to e^-z, to 1e-7 z."""
    assert r["base_idx"].tolist() == ref["base_idx"].tolist()
    assert r["pool_idx"].tolist() == ref["pool_idx"].tolist()
    assert np.max(np.abs(r["base_freqs"] - ref["base_freqs"])) * T_eff <= 10 * tol
    assert np.all(np.abs(r["pool_z"] - ref["pool_z"]) <= 1e-7 * np.abs(ref["pool_z"]))
    assert np.all(np.abs(r["pool_fap"] - ref["pool_fap"]) <= (1e-7 * (1.0 + ref["pool_z"])) * ref["pool_fap"] + 1e-300)


def test_phase1_refined_two_off_grid_sinusoids(fr, p1):
    """fredec_phase1_refined (PAPER.md:201 with the fit of PAPER.md:177-185): two sinusoids between grid points
    and almost no noise -- the base ends with exactly the two true frequencies, as the oracle's does, and
    the grid-only mode on the same series does not."""
    rng = np.random.Generator(np.random.PCG64(8))
    N, K, f0, df, noise = 150, 4000, 0.002, 0.00025, 1e-7
    t = np.sort(rng.uniform(0.0, 200.0, N))
    fa, fb = f0 + 1213.41 * df, f0 + 2790.47 * df
    x = 3.0 * np.sin(TWO_PI * fa * t + 0.3) + 1.2 * np.cos(TWO_PI * fb * t) + 0.7 + noise * rng.standard_normal(N)
    w = np.full(N, 1.0 / noise ** 2)
    T_eff, _ = p1.bandwidth(t, w, 1.0)
    tol = 1e-11
    ref = p1.phase1(t, x, w, f0, df, K, fap0=0.01, fap1_thr=0.02, max_base=6, k_peaks=20, refine_base=True,
                    refine_iter=30, refine_tol=tol)
    r = fr.fredec_phase1(t, x, w, f0, df, K, fap0=0.01, fap1=0.02, max_base=6, k_peaks=20, refine_base=True,
                         refine_iter=30, refine_tol=tol)
    assert r["base_idx"].tolist() == [1213, 2790]
    assert np.max(np.abs(r["base_freqs"] - np.array([fa, fb]))) <= 1e-6 / (t.max() - t.min())
    _assert_refined_equal(r, ref, T_eff, tol)
    grid_only = fr.fredec_phase1(t, x, w, f0, df, K, fap0=0.01, fap1=0.02, max_base=6, k_peaks=20)
    assert len(grid_only["base_idx"]) > 2 and "base_freqs" not in grid_only


def test_phase1_refined_rv_like_series_full_config2(fr, p1):
    """Config 2 in full (N = 1000, K = 80 000): with the refit the base holds the five injected signals once
    each (the grid-only mode enters two of them twice, at neighbouring grid points); pool, base and refitted
    frequencies equal the oracle's; host and device pointers agree bit for bit."""
    import torch
    wl = inputs.config(2)
    t, x, w, _ = wl.series(0)
    T_eff, _ = p1.bandwidth(t, w, 1.0)
    tol = 1e-11
    ref = p1.phase1(t, x, w, wl.f0, wl.df, wl.K, max_base=10, k_peaks=32, refine_base=True, refine_iter=30,
                    refine_tol=tol)
    r = fr.fredec_phase1(t, x, w, wl.f0, wl.df, wl.K, max_base=10, k_peaks=32, refine_base=True, refine_iter=30,
                         refine_tol=tol)
    _assert_refined_equal(r, ref, T_eff, tol)
    bi = np.sort(r["base_idx"])
    assert len(bi) == 5 and np.all(np.diff(bi) > 1)
    true_f = 1.0 / np.array(inputs.RV_PERIODS)
    assert all(np.min(np.abs(true_f - f)) <= 0.1 / (t.max() - t.min()) for f in r["base_freqs"])
    rd = fr.fredec_phase1(*[torch.from_numpy(a).cuda() for a in (t, x, w)], wl.f0, wl.df, wl.K, max_base=10,
                          k_peaks=32, refine_base=True, refine_iter=30, refine_tol=tol)
    for key in ("base_idx", "pool_idx", "base_freqs", "pool_z", "pool_fap"):
        assert np.array_equal(rd[key], r[key]), key
    grid_only = fr.fredec_phase1(t, x, w, wl.f0, wl.df, wl.K, max_base=10, k_peaks=32)
    assert np.any(np.diff(np.sort(grid_only["base_idx"])) == 1)
    # max_base cuts the loop; a refit needs N >= 3 m + 2 observations and max_base <= 25
    r2 = fr.fredec_phase1(t, x, w, wl.f0, wl.df, wl.K, max_base=2, k_peaks=32, refine_base=True)
    assert r2["base_idx"].tolist() == r["base_idx"][:2].tolist() and r2["base_freqs"].shape == (2,)
    for bad in (dict(max_base=26), dict(refine_tol=0.0), dict(refine_iter=-1)):
        with pytest.raises(fr.FredecError) as e:
            fr.fredec_phase1(t, x, w, wl.f0, wl.df, wl.K, refine_base=True, **bad)
        assert e.value.code == fr.FREDEC_EINVAL


def test_phase1_tiny_config_and_noise(fr, p1):
    wl = inputs.config(1)
    t, x, w, _ = wl.series(0)
    ref = p1.phase1(t, x, w, wl.f0, wl.df, wl.K, max_base=5, k_peaks=10)
    r = fr.fredec_phase1(t, x, w, wl.f0, wl.df, wl.K, max_base=5, k_peaks=10)
    _assert_phase1_equal(r, ref)
    assert abs(1.0 / (wl.f0 + r["base_idx"][0] * wl.df) - 17.3) < 0.1      # the generator's main period
    rng = np.random.Generator(np.random.PCG64(12))
    tn = np.sort(rng.uniform(0.0, 100.0, 80))
    xn = rng.standard_normal(80)
    rn = fr.fredec_phase1(tn, xn, np.ones(80), 0.005, 0.001, 2000, fap0=0.01, fap1=0.02)
    assert rn["base_idx"].size == 0 and rn["pool_idx"].size == 0


def test_phase1_argument_errors(fr):
    t, x, w, _ = inputs.random_series(1, 50, 0)
    with pytest.raises(fr.FredecError) as e:
        fr.fredec_phase1(t, x, w, 0.01, 0.001, 100, fap0=0.2, fap1=0.1)      # FAP_1 >= FAP_0
    assert e.value.code == fr.FREDEC_EINVAL
    with pytest.raises(fr.FredecError):
        fr.fredec_phase1(t, x, w, 0.01, 0.001, 100, max_base=40)            # 2*40+1 > FREDEC_D_MAX
    with pytest.raises(fr.FredecError):
        fr.fredec_zstat(np.ones(4), -1.0, 10.0)
    with pytest.raises(fr.FredecError):
        fr.fredec_fap1(np.ones(4), 1.0, 0.0)


@pytest.mark.parametrize("N,M", [(1, 1), (37, 5), (1000, 300), (10_000, 25)])
def test_trig_averages_parity(fr, oracle_mod, N, M):
    """Systems (19), (20) of PAPER.md:242-262 at an arbitrary frequency list.  Tolerance: every term
    carries a few ulp (sincos, products) and the N-term sums differ in order: 4 N eps x sum |term|."""
    import torch
    rng = np.random.Generator(np.random.PCG64(1000 * N + M))
    t = np.sort(rng.uniform(-1500.0, 1500.0, N))
    x = rng.standard_normal(N) * 3.0 + 1.0
    w = rng.uniform(0.25, 4.0, N)
    freqs = rng.uniform(0.0, 3.0, M)
    freqs[0] = 0.0
    ref = oracle_mod.trig_averages(t, x, w, freqs)
    got = fr.fredec_trig_averages(t, x, w, freqs)
    s1, st, sx, sxt, st2 = (np.sum(w * a) for a in (1.0 + 0 * t, abs(t), abs(x), abs(x * t), t * t))
    scale = np.array([s1, s1, st, st, sx, sx, sxt, sxt, st2, st2])
    assert np.all(np.abs(got - ref) <= 4 * N * np.finfo(float).eps * scale + 1e-300)
    gd = fr.fredec_trig_averages(*[torch.from_numpy(a).cuda() for a in (t, x, w, freqs)])
    assert np.array_equal(gd.cpu().numpy(), got)


@pytest.mark.parametrize("n,N", [(1, 4), (3, 40), (6, 200), (10, 1000)])
def test_subset_fits_parity(fr, p1, n, N):
    """Every subset's linear fit.  Tolerance: l is a Schur complement of
    numbers of size D = <x^2>, so errors are relative to D: 1e-10 D (conditioning of a pool with
    well separated frequencies times a few hundred roundings)."""
    import torch
    rng = np.random.Generator(np.random.PCG64(77 * n + N))
    t = np.sort(rng.uniform(0.0, 500.0, N))
    freqs = np.sort(rng.uniform(0.01, 0.9, n))
    x = rng.standard_normal(N) + sum(rng.uniform(0.5, 2.0) * np.sin(2 * np.pi * f * t + rng.uniform(0, 6))
                                     for f in freqs[: max(1, n // 2)])
    w = rng.uniform(0.5, 2.0, N)
    ref = p1.subset_fits(t, x, w, freqs)
    got = fr.fredec_subset_fits(t, x, w, freqs)
    D = float(np.sum(w * x * x))
    assert got.shape == ref.shape and np.all(np.abs(got - ref) <= 1e-10 * D)
    gd = fr.fredec_subset_fits(*[torch.from_numpy(a).cuda() for a in (t, x, w, freqs)])
    assert np.array_equal(gd.cpu().numpy(), got)


@pytest.mark.parametrize("n", [13, 17])
def test_subset_fits_large_pool_sampled(fr, p1, n):
    """Pools beyond one depth-first task (n > 11: a prefix of n - 6 frequencies per warp, then a walk
    over 64 extensions): sampled subsets, the empty and the full one, against the oracle."""
    rng = np.random.Generator(np.random.PCG64(n))
    N = 600
    t = np.sort(rng.uniform(0.0, 800.0, N))
    freqs = np.sort(rng.uniform(0.01, 0.9, n))
    x = rng.standard_normal(N) + sum(1.5 * np.cos(2 * np.pi * f * t + j) for j, f in enumerate(freqs[::3]))
    w = rng.uniform(0.5, 2.0, N)
    got = fr.fredec_subset_fits(t, x, w, freqs)
    masks = np.unique(np.concatenate([[0, (1 << n) - 1, 1, 1 << (n - 1)], rng.integers(0, 1 << n, 300)]))
    ref = p1.subset_fits(t, x, w, freqs, masks=masks)
    D = float(np.sum(w * x * x))
    assert np.all(np.abs(got[masks] - ref) <= 1e-10 * D)
    assert np.all(got >= 0.0) and np.all(got <= got[0] * (1 + 1e-12))


@pytest.mark.parametrize("n", [20, 22, 25])
def test_subset_fits_largest_pools_sampled(fr, p1, n):
    """The pool sizes the paper calls long-but-feasible and "the limit" (15-20, 25-27;
    55 Cnc needed n = 25): 2^n fits in one call, sampled masks (+ empty, full, single bits) against
    the oracle's from-scratch Cholesky."""
    rng = np.random.Generator(np.random.PCG64(100 + n))
    N = 800
    t = np.sort(rng.uniform(0.0, 900.0, N))
    freqs = np.sort(rng.uniform(0.01, 0.9, n))
    x = rng.standard_normal(N) + sum(1.2 * np.cos(2 * np.pi * f * t + j) for j, f in enumerate(freqs[::4]))
    w = rng.uniform(0.5, 2.0, N)
    got = fr.fredec_subset_fits(t, x, w, freqs)
    masks = np.unique(np.concatenate([[0, (1 << n) - 1], 1 << np.arange(n), rng.integers(0, 1 << n, 200),
                                      ((1 << n) - 1) ^ (1 << np.arange(0, n, 5))]))
    ref = p1.subset_fits(t, x, w, freqs, masks=masks)
    D = float(np.sum(w * x * x))
    assert got.shape == (1 << n,)
    assert np.max(np.abs(got[masks] - ref)) <= 1e-10 * D
    assert np.all(got >= 0.0) and np.all(got <= got[0] * (1 + 1e-12))


def _alias_example_series():
    """The own series of tests/golden/alias_example.txt (0.9 and 1.1 Hz, gaps aliasing at 0.1 Hz)."""
    import os
    cfg = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "alias_example.txt")) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                k, v = line.split("=")
                cfg[k.strip()] = float(v)
    n_per = int(round(cfg["window"] / cfg["dt"]))
    t = np.concatenate([m * cfg["gap_period"] + cfg["dt"] * np.arange(n_per) for m in range(int(cfg["n_windows"]))])
    rng = np.random.Generator(np.random.PCG64(294))
    x = np.cos(2 * np.pi * cfg["f_a"] * t) + np.cos(2 * np.pi * cfg["f_b"] * t + 1.0) + 0.1 * rng.standard_normal(t.size)
    return t, x, np.ones_like(t)


@pytest.mark.parametrize("which", ["rv_like_pool", "alias_comb", "near_duplicates"])
def test_subset_fits_aliased_pools(fr, p1, which, report):
    """Pools as phase 1 really produces them ("will likely contain some aliases"): Q of a
    subset that holds a frequency and its aliases is badly conditioned, which is where the walk's
    incrementally updated L^{-1} loses digits.  Pools: (a) the pool the ORACLE's phase 1 finds on the
    config-2 series (seasonal gaps: yearly alias families); (b) the 0.6 ... 1.4 Hz comb of the alias
    example; (c) constructed near-duplicates 0.1/T, 1e-3/T and exactly 0 apart.
    Tolerance as for the benign pools, 1e-10 D (D = <x^2>), wherever the fit is conditioned well enough
    for the oracle itself to be that accurate (smallest relative pivot >= 1e-4; measured against 40-digit
    arithmetic the FP64 oracle is off by up to 1.7e-5 D on the full comb, whose Q has condition 3e16).
    Below that both sides lose eps / pivot of D: bound 1e3 eps D / pivot down to pivot 1e-8; inside the
    S6 band only validity (finite, 0 <= l <= l of the constant alone).  The worst cases per class go to
    the `report` fixture (tables subset_alias_*)."""
    rng = np.random.Generator(np.random.PCG64(7))
    if which == "rv_like_pool":
        wl = inputs.config(2)
        t, x, w, _ = wl.series(0)
        ref1 = p1.phase1(t, x, w, wl.f0, wl.df, wl.K, max_base=10, k_peaks=32)
        idx = ref1["pool_idx"][:18]
        assert idx.size >= 8, "phase 1 should find a pool with aliases on the RV-like series"
        freqs = wl.f0 + wl.df * idx
    elif which == "alias_comb":
        t, x, w = _alias_example_series()
        freqs = np.array([0.6, 0.7, 0.8, 0.9, 1.0, 1.1, 1.2, 1.3, 1.4])
    else:
        t, x, w, _ = inputs.random_series(31, 500, 0, t_span=300.0)
        T = t.max() - t.min()
        freqs = np.array([0.05, 0.05 + 0.1 / T, 0.11, 0.11 + 1e-3 / T, 0.2, 0.2, 0.31, 0.31 + 0.03 / T, 0.4])
    n = freqs.size
    got = fr.fredec_subset_fits(t, x, w, freqs)
    masks = np.arange(1 << n) if n <= 10 else np.unique(np.concatenate(
        [[0, (1 << n) - 1], 1 << np.arange(n), rng.integers(0, 1 << n, 600)]))
    ref, pmin = p1.subset_fits(t, x, w, freqs, masks=masks, return_pivots=True)
    D = float(np.sum(w * x * x))
    err = np.abs(got[masks] - ref)
    well = pmin >= 1e-4                       # class A: the oracle itself is good to ~1e-12 D
    band = (pmin >= 1e-8) & ~well             # class B: eps / pivot of D is lost on either side
    for name, sel in (("pivot>=1e-4", well), ("1e-8<=pivot<1e-4", band), ("pivot<1e-8 or dropped", ~well & ~band)):
        if sel.any():
            report(f"subset_alias_{which}",
                   f"n={n} {name}: masks={int(sel.sum())} max|dl|/D={err[sel].max() / D:.3e} "
                   f"max|dl|*pivot/(eps D)={np.max(err[sel] * np.maximum(pmin[sel], 1e-300)) / (2.2e-16 * D):.3e}")
    assert np.all(np.isfinite(got)) and np.all(got >= 0.0) and np.all(got <= got[0] * (1 + 1e-12))
    assert well.sum() >= masks.size // 8
    assert err[well].max() <= 1e-10 * D, f"max |dl| / D = {err[well].max() / D:.3e}"
    if band.any():
        assert np.all(err[band] <= 1e3 * 2.2e-16 * D / pmin[band])


def test_subset_fits_duplicate_frequency_and_errors(fr, p1):
    t, x, w, _ = inputs.random_series(3, 60, 0)
    freqs = np.array([0.2, 0.2, 0.31])
    ref = p1.subset_fits(t, x, w, freqs)
    got = fr.fredec_subset_fits(t, x, w, freqs)
    assert np.all(np.isfinite(got)) and np.all(np.abs(got - ref) <= 1e-9 * ref[0])
    with pytest.raises(fr.FredecError):
        fr.fredec_subset_fits(t, x, w, np.linspace(0.1, 0.9, 26))           # n > 25
    with pytest.raises(fr.FredecError):
        fr.fredec_subset_fits(t[:5], x[:5], w[:5], np.array([0.1, 0.2]))    # N < 2n + 2


@pytest.mark.parametrize("noise,n", [(0.0, 2), (0.3, 2), (0.5, 4)])
def test_refine_parity(fr, p1, noise, n):
    """Local multifrequency fit.  Both sides stop on the same criterion
    (max |step| T_eff <= tol), so the frequencies agree to a few tol / T_eff and l to rounding of a
    Schur complement of size D: 1e-9 D (the iteration count may differ by one at the threshold)."""
    rng = np.random.Generator(np.random.PCG64(90 + n))
    N = 400
    t = np.sort(rng.uniform(50.0, 650.0, N))
    f_true = np.sort(rng.uniform(0.02, 0.4, n))
    x = 0.3 + sum((2.5 - 0.4 * k) * np.cos(2 * np.pi * f * t + k) for k, f in enumerate(f_true)) \
        + noise * rng.standard_normal(N)
    w = rng.uniform(0.5, 2.0, N)
    T = t.max() - t.min()
    start = f_true + rng.uniform(-0.25, 0.25, n) / T
    tol = 1e-9
    f_ref, l_ref, it_ref = p1.refine(t, x, w, start, max_iter=30, tol=tol)
    f, l, it = fr.fredec_refine(t, x, w, start, max_iter=30, tol=tol)
    T_eff, _ = p1.bandwidth(t, w, 1.0)
    D = float(np.sum(w * x * x))
    assert np.max(np.abs(f - f_ref)) * T_eff <= 10 * tol
    assert abs(l - l_ref) <= 1e-9 * D and abs(it - it_ref) <= 1
    if noise == 0.0:
        assert np.max(np.abs(f - f_true)) * T < 1e-7 and l <= 1e-12 * D
    # device pointers; and no iterations = the linear fit at the start
    import torch
    fd, ld, _ = fr.fredec_refine(*[torch.from_numpy(a).cuda() for a in (t, x, w)], start, max_iter=30, tol=tol)
    assert np.array_equal(fd, f) and ld == l
    f0, l0, it0 = fr.fredec_refine(t, x, w, start, max_iter=0)
    _, l0_ref, _ = p1.refine(t, x, w, start, max_iter=0)
    assert it0 == 0 and np.array_equal(f0, start) and abs(l0 - l0_ref) <= 1e-9 * D


def test_refine_batched_parity_1000_tuples(fr, p1, oracle_mod, report):
    """PAPER.md:214 / :266: the local fits l_{m,loc} of many subsets of one pool in one call (one CTA per
    tuple, every iteration on the device) against the oracle's refine() looped over the tuples.  Pool: 12
    frequencies near 12 sinusoids of the series (start values up to 0.2 / T off); 1000 random subsets of
    1..6 of them + the empty and the full tuple.  Bars: frequencies within 10 tol / T_eff, l within
    1e-9 D, iteration counts within one (both sides stop on max |step| T_eff <= tol)."""
    rng = np.random.Generator(np.random.PCG64(2140))
    N, n_pool = 600, 12
    t = np.sort(rng.uniform(0.0, 400.0, N))
    T = t.max() - t.min()
    f_true = 0.02 + 0.035 * np.arange(n_pool) + rng.uniform(-0.005, 0.005, n_pool)
    x = 0.4 + sum((3.0 - 0.15 * k) * np.cos(2 * np.pi * f * t + 0.7 * k) for k, f in enumerate(f_true)) \
        + 0.5 * rng.standard_normal(N)
    w = rng.uniform(0.5, 2.0, N)
    pool = f_true + rng.uniform(-0.2, 0.2, n_pool) / T
    masks = [0, (1 << n_pool) - 1]
    while len(masks) < 1002:
        size = int(rng.integers(1, 7))
        masks.append(int(sum(1 << int(j) for j in rng.choice(n_pool, size=size, replace=False))))
    masks = np.array(masks, dtype=np.int64)
    tol = 1e-9
    freqs, l, iters, status = fr.fredec_refine_batched(t, x, w, pool, masks, max_iter=30, tol=tol)
    assert np.all(status == 0)
    T_eff, _ = p1.bandwidth(t, w, 1.0)
    D = float(np.sum(w * x * x))
    worst_f = worst_l = 0.0
    for i, mask in enumerate(masks):
        sel = [j for j in range(n_pool) if (mask >> j) & 1]
        if not sel:                        # the empty tuple: the constant alone, nothing to iterate
            assert iters[i] == 0 and abs(l[i] - oracle_mod.chi2_base(t, x, w, np.ones((1, N)))) <= 1e-12 * D
            continue
        f_ref, l_ref, it_ref = p1.refine(t, x, w, pool[sel], max_iter=30, tol=tol)
        assert abs(int(iters[i]) - it_ref) <= 1, (i, mask, iters[i], it_ref)
        if sel:
            worst_f = max(worst_f, float(np.max(np.abs(freqs[i, sel] - f_ref))) * T_eff)
        worst_l = max(worst_l, abs(l[i] - l_ref))
        unsel = [j for j in range(n_pool) if not (mask >> j) & 1]
        assert np.array_equal(freqs[i, unsel], pool[unsel])
    assert worst_f <= 10 * tol, worst_f
    assert worst_l <= 1e-9 * D, worst_l / D
    # the single-tuple call is the batched one with T = 1; device pointers give the same bits
    import torch
    f1, l1, it1 = fr.fredec_refine(t, x, w, pool[[1, 4, 7]], max_iter=30, tol=tol)
    i147 = fr.fredec_refine_batched(t, x, w, pool, np.array([0b10010010]), max_iter=30, tol=tol)
    assert np.max(np.abs(f1 - i147[0][0, [1, 4, 7]])) * T_eff <= 10 * tol and abs(l1 - i147[1][0]) <= 1e-9 * D
    fd, ld, _, _ = fr.fredec_refine_batched(*[torch.from_numpy(a).cuda() for a in (t, x, w, pool)], masks[:50],
                                             max_iter=30, tol=tol)
    assert np.array_equal(fd, freqs[:50]) and np.array_equal(ld, l[:50])
    report("refine_batched", f"tuples=50 kernel_ms={fr.fredec_last_timing()['scan_ms']:.3f}")
    fr.fredec_refine_batched(t, x, w, pool, masks, max_iter=30, tol=tol)
    tm = fr.fredec_last_timing()
    report("refine_batched", f"tuples={masks.size} N={N} sizes 1..6 (+ empty, full 12): kernel_ms={tm['scan_ms']:.3f} "
                             f"tuples_per_s={masks.size / (tm['scan_ms'] * 1e-3):.3e}")


def test_refine_batched_singular_tuple_and_errors(fr):
    t, x, w, _ = inputs.random_series(2, 80, 0)
    pool = np.array([0.2, 0.2, 0.31])
    freqs, l, iters, status = fr.fredec_refine_batched(t, x, w, pool, np.array([0b011, 0b101, 0b100]))
    assert status.tolist() == [fr.FREDEC_ESINGULAR, 0, 0] and l[0] == 0.0 and l[1] > 0.0
    with pytest.raises(fr.FredecError):
        fr.fredec_refine_batched(t, x, w, pool, np.array([8]))                 # bit beyond the pool
    with pytest.raises(fr.FredecError):
        fr.fredec_refine_batched(t[:10], x[:10], w[:10], pool, np.array([7]))    # N < 3 m + 2
    with pytest.raises(fr.FredecError):
        fr.fredec_refine_batched(t, x, w, np.linspace(0.1, 0.9, 26))           # pool > 25


def test_refine_batched_device_masks(fr):
    """Masks in device memory are measured and range-checked by a small kernel: same fits as host masks, a bit
    beyond the pool is FREDEC_EINVAL, and N only has to cover the largest tuple actually present."""
    import torch
    t, x, w, _ = inputs.random_series(2, 40, 0)
    pool = np.linspace(0.11, 0.47, 20)                       # N = 40 < 3 * 20 + 2: only small tuples fit
    masks = np.array([0b11, 0b101, 1 << 19, 0, 0b1110000], dtype=np.int64)
    ref = fr.fredec_refine_batched(t, x, w, pool, masks)
    dev = fr.fredec_refine_batched(t, x, w, pool, torch.from_numpy(masks).cuda())
    for a, b in zip(ref, dev):
        assert np.array_equal(a, b)
    for bad in ([0b11, 1 << 20], [-1, 0b11]):
        with pytest.raises(fr.FredecError) as e:
            fr.fredec_refine_batched(t, x, w, pool, torch.tensor(bad, dtype=torch.int64, device="cuda"))
        assert e.value.code == fr.FREDEC_EINVAL
    with pytest.raises(fr.FredecError) as e:                 # a tuple of 13 needs N >= 41
        fr.fredec_refine_batched(t, x, w, pool, torch.tensor([(1 << 13) - 1], dtype=torch.int64, device="cuda"))
    assert e.value.code == fr.FREDEC_EINVAL


def test_non_finite_frequencies_are_data_errors(fr):
    """freqs must be finite (include/fredec.h): FREDEC_EDATA from host and from device pointers."""
    import torch
    t, x, w, _ = inputs.random_series(2, 60, 0)
    bad = np.array([0.1, np.nan, 0.3])
    for conv in (lambda a: a, lambda a: torch.from_numpy(a).cuda()):
        args = [conv(a) for a in (t, x, w)]
        for fn in (lambda: fr.fredec_trig_averages(*args, conv(bad)),
                   lambda: fr.fredec_subset_fits(*args, conv(bad)),
                   lambda: fr.fredec_refine(*args, bad),
                   lambda: fr.fredec_trig_averages(*args, conv(np.array([np.inf])))):
            with pytest.raises(fr.FredecError) as e:
                fn()
            assert e.value.code == fr.FREDEC_EDATA
    assert np.all(np.isfinite(fr.fredec_trig_averages(t, x, w, np.array([0.1, 0.2]))))


def test_refine_errors(fr):
    t, x, w, _ = inputs.random_series(2, 60, 0)
    with pytest.raises(fr.FredecError) as e:
        fr.fredec_refine(t, x, w, np.array([0.2, 0.2]))           # equal frequencies: singular
    assert e.value.code == fr.FREDEC_ESINGULAR
    with pytest.raises(fr.FredecError):
        fr.fredec_refine(t[:7], x[:7], w[:7], np.array([0.1, 0.2]))   # N < 3n + 2
    with pytest.raises(fr.FredecError):
        fr.fredec_refine(t, x, w, np.array([0.1]), tol=0.0)
