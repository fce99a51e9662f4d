"""Seeded synthetic inputs for the FREDEC periodogram scan (numpy only).

This module is the ONE thing the CUDA path and the CPU oracle share: it draws the
time series (t, x, w), evaluates the base-model functions on the times and names the
frequency grid.  It holds none of the method's arithmetic (no trigonometric sums, no
least squares, no peak search).

The five workloads are the synthetic stand-ins BASELINE.json:configs names for the
paper's artificial series (section 7.1) and radial-velocity data sets
(sections 7.2-7.4), which are not available.  Recipe: SURVEY.md
section 8(d); readings of the loosely stated items are recorded in DESIGN.md section 4.

All arrays are float64, times sorted ascending, weights w = 1/sigma^2 (PAPER.md:43:
"D eps_i = kappa / w_i").  Random numbers: numpy.random.Generator(PCG64(seed)),
seed = 13090100 + workload number.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

SEED_BASE = 13090100
TWO_PI = 2.0 * np.pi


@dataclass
class Workload:
    """One scan problem: B series of N observations, d base functions, K grid frequencies."""
    name: str
    t: np.ndarray            # [B, N] (B == 1 for single-series workloads)
    x: np.ndarray            # [B, N]
    w: np.ndarray            # [B, N]
    base_funcs: np.ndarray   # [B, d, N]
    f0: float
    df: float
    K: int
    topk: int
    meta: dict = field(default_factory=dict)

    @property
    def B(self) -> int:
        return self.t.shape[0]

    @property
    def N(self) -> int:
        return self.t.shape[1]

    @property
    def d(self) -> int:
        return self.base_funcs.shape[1]

    @property
    def pairs(self) -> int:
        """(frequency x observation) pairs of one scan of the whole workload."""
        return self.B * self.N * self.K

    def series(self, b: int = 0):
        """(t, x, w, base_funcs[d, N]) of series b as contiguous arrays."""
        return (np.ascontiguousarray(self.t[b]), np.ascontiguousarray(self.x[b]),
                np.ascontiguousarray(self.w[b]), np.ascontiguousarray(self.base_funcs[b]))

    def head(self, K: int | None = None, B: int | None = None) -> "Workload":
        """The same workload restricted to its first K grid points / first B series."""
        K = self.K if K is None else min(K, self.K)
        B = self.B if B is None else min(B, self.B)
        return Workload(f"{self.name}[K={K},B={B}]", self.t[:B], self.x[:B], self.w[:B],
                        self.base_funcs[:B], self.f0, self.df, K, self.topk, dict(self.meta))


def _rng(number: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED_BASE + number))


def base_offset(t: np.ndarray) -> np.ndarray:
    """Base model H_0 of PAPER.md:49 (eq. 1): a free constant.  Returns [1, N]."""
    return np.ones((1, t.shape[0]))


def base_offset_trend(t: np.ndarray) -> np.ndarray:
    """Constant + linear trend ("time polynomial").  Returns [2, N]."""
    return np.stack([np.ones_like(t), t])


def base_offset_sinusoids(t: np.ndarray, periods) -> np.ndarray:
    """Constant + cos/sin pairs at fixed, already accepted periods (base model H_m of
    PAPER.md:56 eq. 2 / PAPER.md:106 eq. 10).  Returns [1 + 2 len(periods), N]."""
    rows = [np.ones_like(t)]
    for P in periods:
        rows.append(np.cos(TWO_PI * t / P))
        rows.append(np.sin(TWO_PI * t / P))
    return np.stack(rows)


def _single(name, t, x, w, base, f0, df, K, topk, **meta) -> Workload:
    return Workload(name, t[None, :], x[None, :], w[None, :], base[None, :, :],
                    float(f0), float(df), int(K), int(topk), meta)


# --------------------------------------------------------------------------- config 1
def tiny(N: int = 200, K: int = 10_000) -> Workload:
    rng = _rng(1)
    t = np.sort(rng.uniform(0.0, 1000.0, N))
    sigma = rng.uniform(1.0, 3.0, N)
    x = (5.0 * np.sin(TWO_PI * t / 17.3 + 0.4) + 3.0 * np.cos(TWO_PI * t / 91.0)
         + rng.normal(0.0, 1.0, N) * sigma)
    return _single("tiny", t, x, 1.0 / sigma**2, base_offset(t), 1e-3, 1e-4, K, 10,
                   signal_periods=[17.3, 91.0])


# ----------------------------------------------------------------------- configs 2, 3
RV_PERIODS = (2.8, 14.6, 44.0, 260.0, 5000.0)
RV_AMPLITUDES = (70.0, 10.0, 12.0, 5.0, 45.0)


def _rv_series(rng: np.random.Generator, N: int):
    """Seasonal sampling: observable 240 d of every 365 d over 8000 d, uniform inside."""
    starts = np.arange(0.0, 8000.0, 365.0)
    ends = np.minimum(starts + 240.0, 8000.0)
    lengths = ends - starts
    season = rng.choice(len(starts), size=N, p=lengths / lengths.sum())
    t = np.sort(starts[season] + rng.uniform(0.0, 1.0, N) * lengths[season])
    sigma = np.exp(rng.normal(np.log(3.0), 0.3, N))
    phases = rng.uniform(0.0, TWO_PI, len(RV_PERIODS))
    x = np.zeros(N)
    for P, A, ph in zip(RV_PERIODS, RV_AMPLITUDES, phases):
        x += A * np.cos(TWO_PI * t / P + ph)
    x += rng.normal(0.0, 1.0, N) * sigma
    return t, x, 1.0 / sigma**2, phases


def rv_like(N: int = 1000, K: int = 80_000) -> Workload:
    t, x, w, phases = _rv_series(_rng(2), N)
    return _single("rv_like", t, x, w, base_offset(t), 1.0 / 16000.0, 1.0 / 80000.0, K, 10,
                   signal_periods=list(RV_PERIODS), phases=phases.tolist())


def residual(N: int = 2000, K: int = 200_000, n_base: int = 4) -> Workload:
    """n_base accepted sinusoids in the base model (d = 2 n_base + 1): the first four signal periods,
    then -- for the late SLICK iterations of PAPER.md:208-210, whose base reaches d = 51 -- further
    fixed periods 3.7 * 1.31^j d."""
    t, x, w, phases = _rv_series(_rng(3), N)
    periods = list(RV_PERIODS[:4]) + [3.7 * 1.31**j for j in range(max(0, n_base - 4))]
    base = base_offset_sinusoids(t, periods[:n_base])
    return _single("residual", t, x, w, base, 1e-4, 1e-5, K, 10,
                   signal_periods=list(RV_PERIODS), base_periods=periods[:n_base],
                   phases=phases.tolist())


# --------------------------------------------------------------------------- config 4
def survey(N: int = 10_000, K: int = 2_000_000) -> Workload:
    """Regular cadence on [0, 3000] d with a 1-day-wide uniform jitter, 30 % dropouts."""
    rng = _rng(4)
    M = int(np.ceil(N / 0.7))
    nominal = np.linspace(0.0, 3000.0, M)
    jittered = nominal + rng.uniform(-0.5, 0.5, M)
    keep = rng.choice(M, size=N, replace=False)
    t = np.sort(jittered[keep])
    sigma = rng.uniform(0.5, 2.0, N)
    periods = np.exp(rng.uniform(np.log(0.5), np.log(500.0), 3))
    amps = rng.uniform(0.5, 3.0, 3)
    phases = rng.uniform(0.0, TWO_PI, 3)
    x = np.zeros(N)
    for P, A, ph in zip(periods, amps, phases):
        x += A * np.cos(TWO_PI * t / P + ph)
    x += rng.normal(0.0, 1.0, N) * sigma
    return _single("survey", t, x, 1.0 / sigma**2, base_offset_trend(t), 1e-4, 1.5e-6, K, 10,
                   signal_periods=periods.tolist(), amplitudes=amps.tolist())


# --------------------------------------------------------------------------- config 5
def batched(B: int = 4096, N: int = 500, K: int = 100_000) -> Workload:
    rng = _rng(5)
    t = np.sort(rng.uniform(0.0, 2000.0, (B, N)), axis=1)
    sigma = rng.uniform(1.0, 3.0, (B, N))
    n_sig = rng.integers(1, 4, B)
    periods = np.exp(rng.uniform(np.log(1.0), np.log(1000.0), (B, 3)))
    amps = rng.uniform(1.0, 10.0, (B, 3))
    phases = rng.uniform(0.0, TWO_PI, (B, 3))
    x = rng.normal(0.0, 1.0, (B, N)) * sigma
    for j in range(3):
        on = (n_sig > j)[:, None]
        x += on * amps[:, j:j + 1] * np.cos(TWO_PI * t / periods[:, j:j + 1] + phases[:, j:j + 1])
    base = np.ones((B, 1, N))
    return Workload("batched", t, x, 1.0 / sigma**2, base, 5e-4, 5e-5, int(K), 5,
                    {"n_sig": n_sig.tolist()})


CONFIGS = {1: tiny, 2: rv_like, 3: residual, 4: survey, 5: batched}


def config(number: int, **kw) -> Workload:
    """Workload number 1..5 of BASELINE.json:configs (keyword overrides shrink it)."""
    return CONFIGS[number](**kw)


# ------------------------------------------------------------ small cases for the tests
def random_series(seed: int, N: int, d: int, t_span: float = 100.0, noise: float = 1.0):
    """Irregular times, unequal weights, a polynomial base of d functions (d may be 0)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    t = np.sort(rng.uniform(0.0, t_span, N))
    sigma = rng.uniform(0.5, 2.0, N)
    x = (2.0 * np.cos(TWO_PI * t * (7.3 / t_span) + 0.3) + 0.7 * np.sin(TWO_PI * t * (19.1 / t_span))
         + 0.05 * t / t_span + rng.normal(0.0, noise, N) * sigma)
    return t, x, 1.0 / sigma**2, mixed_base(t, d, t_span)


def mixed_base(t: np.ndarray, d: int, t_span: float) -> np.ndarray:
    """A well-conditioned base model of d functions: 1, t, then cos/sin pairs at fixed
    frequencies (2.3137 + 1.7291 m)/t_span (accepted sinusoids), t^2 when d is even
    and > 2; plain polynomials for d <= 3.  Returns [d, N]."""
    N = t.shape[0]
    if d == 0:
        return np.zeros((0, N))
    tc = (t - t.mean()) / t_span
    if d <= 3:
        return np.stack([tc**j for j in range(d)])
    rows = [np.ones_like(tc), tc]
    m = 0
    while len(rows) + 2 <= d:
        nu = 2.3137 + 1.7291 * m
        rows += [np.cos(TWO_PI * nu * tc), np.sin(TWO_PI * nu * tc)]
        m += 1
    if len(rows) < d:
        rows.append(tc**2)
    return np.stack(rows)
