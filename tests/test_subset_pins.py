"""Pins for oracle.phase1.subset_fits (PAPER.md:158-175 for every subset of a pool):
the definition by QR least squares, nesting, and exactness on noiseless sinusoids."""
import numpy as np
import pytest

from paper_1309_0100_b200 import inputs

TWO_PI = 2.0 * np.pi


@pytest.fixture(scope="module")
def p1(oracle_mod):
    from oracle import phase1
    return phase1


def _lstsq_l(t, x, w, fs):
    sw = np.sqrt(w)
    cols = [sw] + [sw * fn(TWO_PI * f * t) for f in fs for fn in (np.cos, np.sin)]
    A = np.column_stack(cols)
    theta = np.linalg.lstsq(A, sw * x, rcond=None)[0]
    r = sw * x - A @ theta
    return float(r @ r)


def test_subset_fits_are_the_least_squares_minima(p1, oracle_mod):
    t, x, w, _ = inputs.random_series(31, 60, 0, t_span=40.0)
    freqs = np.array([0.051, 0.173, 0.3, 0.42])
    l = p1.subset_fits(t, x, w, freqs)
    for mask in range(16):
        fs = [freqs[j] for j in range(4) if (mask >> j) & 1]
        assert abs(l[mask] - _lstsq_l(t, x, w, fs)) <= 1e-11 * l[0], mask
    assert abs(l[0] - oracle_mod.chi2_base(t, x, w, inputs.base_offset(t))) <= 1e-12 * l[0]
    # nesting: a larger model never fits worse (the smaller Q is a leading block)
    for mask in range(16):
        for j in range(4):
            assert l[mask | (1 << j)] <= l[mask] * (1 + 1e-12)
    # consistency with the scan: dropping chi2 by scan(base = subset model) at a pool frequency
    base = p1.sinusoid_base(t, freqs[[0, 2]])
    dz = oracle_mod.scan(t, x, w, base, freqs[1], 1.0, 1)[0]
    assert abs((l[0b0101] - l[0b0111]) - dz) <= 1e-10 * l[0]


def test_subset_fits_noiseless_and_duplicate_frequency(p1):
    rng = np.random.Generator(np.random.PCG64(2))
    t = np.sort(rng.uniform(0, 30, 50))
    freqs = np.array([0.11, 0.29, 0.47])
    x = 1.5 + 2.0 * np.cos(TWO_PI * 0.11 * t + 0.4) + 0.7 * np.sin(TWO_PI * 0.47 * t)
    w = rng.uniform(0.5, 2.0, 50)
    l = p1.subset_fits(t, x, w, freqs)
    assert l[0b101] <= 1e-12 * l[0]                                      # the true model fits exactly
    assert l[0b111] <= 1e-12 * l[0]
    assert l[0b001] > 1e-3 * l[0] and l[0b100] > 1e-3 * l[0]             # either signal alone does not
    # a duplicated frequency adds nothing and does not break the factorisation (S6)
    ld = p1.subset_fits(t, x, w, np.array([0.11, 0.11]))
    assert np.isfinite(ld).all() and abs(ld[0b11] - ld[0b01]) <= 1e-9 * ld[0] and abs(ld[0b10] - ld[0b01]) <= 1e-12 * ld[0]
