"""Pins for oracle.trig_averages (systems (19), (20) of PAPER.md:242-262): against the definition in
50-digit arithmetic, a closed form, derivative identities and column-swap identities."""
import numpy as np

from paper_1309_0100_b200 import inputs

TWO_PI = 2.0 * np.pi


def test_trig_averages_against_mpmath(oracle_mod):
    import mpmath as mp
    mp.mp.dps = 50
    rng = np.random.Generator(np.random.PCG64(8))
    N = 12
    t = rng.uniform(-3e4, 3e4, N)          # phases of ~1e5 turns
    x = rng.standard_normal(N)
    w = rng.uniform(0.5, 2.0, N)
    freqs = np.array([0.0137, 1.7, 4.99])
    got = oracle_mod.trig_averages(t, x, w, freqs)
    for j, f in enumerate(freqs):
        ref = [mp.mpf(0)] * 10
        for i in range(N):
            ti, xi, wi = mp.mpf(float(t[i])), mp.mpf(float(x[i])), mp.mpf(float(w[i]))
            c, s = mp.cos(2 * mp.pi * mp.mpf(float(f)) * ti), mp.sin(2 * mp.pi * mp.mpf(float(f)) * ti)
            terms = [wi * c, wi * s, wi * ti * c, wi * ti * s, wi * xi * c, wi * xi * s,
                     wi * xi * ti * c, wi * xi * ti * s, wi * ti * ti * c, wi * ti * ti * s]
            ref = [a + b for a, b in zip(ref, terms)]
        scale = [np.sum(w), np.sum(w), np.sum(w * abs(t)), np.sum(w * abs(t)), np.sum(w * abs(x)), np.sum(w * abs(x)),
                 np.sum(w * abs(x * t)), np.sum(w * abs(x * t)), np.sum(w * t * t), np.sum(w * t * t)]
        for q in range(10):
            assert abs(got[j, q] - float(ref[q])) <= 1e-14 * scale[q], (j, q)


def test_trig_averages_even_spacing_closed_form(oracle_mod):
    """sum_{i<N} exp(i w D i) = (1 - exp(i w D N)) / (1 - exp(i w D)) for unit weights."""
    N, D = 64, 0.75
    t = D * np.arange(N)
    freqs = np.array([0.031, 0.2, 0.61])
    got = oracle_mod.trig_averages(t, np.ones(N), np.ones(N), freqs)
    for j, f in enumerate(freqs):
        q = np.exp(1j * TWO_PI * f * D)
        geo = (1 - q ** N) / (1 - q)
        assert abs(got[j, 0] - geo.real) < 1e-12 and abs(got[j, 1] - geo.imag) < 1e-12


def test_trig_averages_derivative_and_column_identities(oracle_mod):
    """d/dw <sin wt> = <t cos wt>, d/dw <cos wt> = -<t sin wt>, d/dw <t sin wt> = <t^2 cos wt>,
    d/dw <t cos wt> = -<t^2 sin wt> (the t multipliers ARE frequency derivatives);
    x = 1 maps the x columns onto the plain ones, x = t onto the next moment."""
    t, x, w, _ = inputs.random_series(21, 50, 0, t_span=20.0)
    f, h = 0.173, 1e-5
    A = oracle_mod.trig_averages(t, x, w, np.array([f - h, f, f + h]))
    dA = (A[2] - A[0]) / (2 * h) / TWO_PI          # d/d omega
    tol = 1e-6 * np.sum(w * np.abs(t) ** 3)        # O(h^2) truncation of the central difference
    assert abs(dA[1] - A[1, 2]) < tol and abs(dA[0] + A[1, 3]) < tol
    assert abs(dA[3] - A[1, 8]) < tol * 20 and abs(dA[2] + A[1, 9]) < tol * 20
    assert abs(dA[5] - A[1, 6]) < tol * 5 and abs(dA[4] + A[1, 7]) < tol * 5
    one = oracle_mod.trig_averages(t, np.ones_like(t), w, np.array([f]))[0]
    assert np.allclose(one[4:8], one[0:4], rtol=0, atol=1e-13 * np.sum(w * np.abs(t)))
    xt = oracle_mod.trig_averages(t, t, w, np.array([f]))[0]
    assert np.allclose(xt[4:6], xt[2:4], rtol=0, atol=1e-13 * np.sum(w * np.abs(t)))
    assert np.allclose(xt[6:8], xt[8:10], rtol=0, atol=1e-13 * np.sum(w * t * t))
