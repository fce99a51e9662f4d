"""The S6 claim about the five BASELINE.json configs (S6; "the generator asserts no
config has one"): no trial frequency of any config's grid lies in the band where the trial cos / sin column is
nearly in the span of the base model, so rule S6 (drop the column) never decides a value that the parity
tests compare.  Measured here with plain numpy, independently of the oracle and of the CUDA path: the
relative Schur pivot of a column is |P c|^2 / |c|^2 with P the weighted projection off everything before it
(the base functions; for the sine also the cosine), from a Householder QR of the base."""
import numpy as np
import pytest

from paper_1309_0100_b200 import inputs

PIVOT_FLOOR = 1e-6      # the band of rule S6 ends far below (kTauTrial = 1e-10 drops, < 1e-6 loses digits)


def min_relative_pivot(t, w, base, freqs, block=4096):
    sw = np.sqrt(w)
    tc = t - np.sum(w * t) / np.sum(w)
    Q = np.linalg.qr((base * sw).T)[0] if base.shape[0] else np.zeros((t.shape[0], 0))
    worst = np.inf
    for i in range(0, freqs.shape[0], block):
        ph = 2.0 * np.pi * np.outer(tc, freqs[i:i + block])
        C, S = sw[:, None] * np.cos(ph), sw[:, None] * np.sin(ph)
        c2, s2 = np.sum(C * C, axis=0), np.sum(S * S, axis=0)
        C -= Q @ (Q.T @ C)
        S -= Q @ (Q.T @ S)
        pc = np.sum(C * C, axis=0)
        S -= C * (np.sum(C * S, axis=0) / pc)
        ps = np.sum(S * S, axis=0)
        worst = min(worst, float(np.min(pc / c2)), float(np.min(ps / s2)))
    return worst


def test_helper_sees_a_column_inside_the_base():
    """The measure itself: a trial frequency equal to a base frequency gives pivot ~ 0, one 0.3 cycles over the
    span away a pivot of order (pi 0.3)^2 / 3."""
    t, x, w, _ = inputs.random_series(5, 300, 0)
    base = inputs.base_offset_sinusoids(t, [1.0 / 0.2])
    T = t.max() - t.min()
    assert min_relative_pivot(t, w, base, np.array([0.2])) < 1e-20
    p = min_relative_pivot(t, w, base, np.array([0.2 + 0.3 / T]))
    assert 0.05 < p < 1.0


@pytest.mark.parametrize("cfg,stride,series_stride", [(1, 1, 1), (2, 1, 1), (3, 1, 1), (4, 128, 1), (5, 32, 64)])
def test_no_config_has_a_grid_point_in_the_s6_band(cfg, stride, series_stride):
    """Configs 1-3 on every grid point; 4 and 5 on a stride of the grid (and of the batch) plus the grid's
    first 2000 points, where f T is smallest and the cosine is closest to the constant."""
    wl = inputs.config(cfg)
    ks = np.unique(np.concatenate([np.arange(0, wl.K, stride), np.arange(min(wl.K, 2000)), [wl.K - 1]]))
    freqs = wl.f0 + wl.df * ks
    worst = min(min_relative_pivot(*(wl.series(b)[i] for i in (0, 2, 3)), freqs)
                for b in range(0, wl.B, series_stride))
    assert worst >= PIVOT_FLOOR, f"config {cfg}: smallest relative pivot {worst:.3e}"
