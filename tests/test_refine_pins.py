"""Pins for oracle.phase1.refine: exact recovery on noiseless off-grid sinusoids,
stationarity of the profile chi-square, agreement with scipy's general non-linear least squares, and
the step clamp (reading R1)."""
import numpy as np
import pytest

TWO_PI = 2.0 * np.pi


@pytest.fixture(scope="module")
def p1(oracle_mod):
    from oracle import phase1
    return phase1


def _series(noise, seed=4, N=150):
    rng = np.random.Generator(np.random.PCG64(seed))
    t = np.sort(rng.uniform(100.0, 400.0, N))
    f_true = np.array([0.0371234, 0.1129876])
    x = (0.4 + 2.0 * np.cos(TWO_PI * f_true[0] * t + 0.7) + 1.1 * np.sin(TWO_PI * f_true[1] * t - 0.2)
         + noise * rng.standard_normal(N))
    w = rng.uniform(0.5, 2.0, N)
    return t, x, w, f_true


def test_refine_recovers_noiseless_frequencies(p1):
    t, x, w, f_true = _series(0.0)
    T = t.max() - t.min()
    start = f_true + np.array([0.3, -0.25]) / T
    f, l, iters = p1.refine(t, x, w, start, max_iter=30, tol=1e-11)
    assert np.max(np.abs(f - f_true)) * T < 1e-8 and l <= 1e-13 * np.sum(w * x * x)    # D - |a|^2 cancels to rounding
    assert 2 <= iters <= 15
    # no iterations: the linear fit at the start frequencies (l_m of eq. 7), larger than the local minimum
    f0, l0, it0 = p1.refine(t, x, w, start, max_iter=0)
    assert it0 == 0 and np.array_equal(f0, start) and abs(l0 - p1.subset_fits(t, x, w, start, masks=[3])[0]) <= 1e-9 * l0
    assert l0 > 1e-3 * np.sum(w * x * x)


def test_refine_is_stationary_and_matches_scipy(p1):
    from scipy.optimize import least_squares
    t, x, w, f_true = _series(0.3)
    T = t.max() - t.min()
    start = f_true + np.array([-0.2, 0.15]) / T
    f, l, iters = p1.refine(t, x, w, start, max_iter=40, tol=1e-10)
    # profile chi2(f) = min over theta: central differences vanish at the local fit
    prof = lambda ff: p1.subset_fits(t, x, w, ff, masks=[3])[0]
    h = 1e-5 / T
    for k in range(2):
        e = np.zeros(2)
        e[k] = h
        slope = (prof(f + e) - prof(f - e)) / (2 * h)
        curv = (prof(f + e) - 2 * prof(f) + prof(f - e)) / h ** 2
        assert abs(slope) <= 1e-4 * abs(curv) / T and curv > 0          # at a minimum
    assert abs(l - prof(f)) <= 1e-9 * l
    # the general-purpose solver started at the same point lands on the same minimum
    sw = np.sqrt(w)
    t0 = np.sum(w * t) / np.sum(w)

    def resid(p):
        mu = p[0] + sum(p[1 + 2 * k] * np.cos(TWO_PI * p[5 + k] * (t - t0)) + p[2 + 2 * k] * np.sin(TWO_PI * p[5 + k] * (t - t0))
                        for k in range(2))
        return sw * (x - mu)
    p0 = np.concatenate([[0.0, 1.0, 1.0, 1.0, 1.0], start])
    # give scipy the linear part at the start
    A = np.column_stack([sw] + [sw * fn(TWO_PI * fk * (t - t0)) for fk in start for fn in (np.cos, np.sin)])
    p0[:5] = np.linalg.lstsq(A, sw * x, rcond=None)[0]
    sol = least_squares(resid, p0, xtol=1e-15, ftol=1e-15, gtol=1e-15, x_scale="jac")
    assert np.max(np.abs(sol.x[5:] - f)) * T < 1e-6
    assert abs(2 * sol.cost - l) <= 1e-9 * l


def test_refine_step_clamp(p1):
    """Reading R1: one update moves a frequency by at most 0.5 / T_eff."""
    t, x, w, f_true = _series(0.0)
    T_eff, _ = p1.bandwidth(t, w, 1.0)
    start = f_true + np.array([0.45, 0.0]) / (t.max() - t.min())
    f1, _, it = p1.refine(t, x, w, start, max_iter=1)
    assert it == 1 and np.all(np.abs(f1 - start) <= 0.5 / T_eff * (1 + 1e-12))
