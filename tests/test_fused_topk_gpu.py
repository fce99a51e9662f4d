"""GPU parity of the peak extraction fused into the scan's epilogue (`fredec_scan_topk(_batched)` with
z_out = NULL: no periodogram is written, SURVEY.md 8(a) rows a10/a11 in one kernel) against the CPU oracle's
peaks of the CPU oracle's periodogram, and against the library's own two-kernel path (scan -> z -> top-k),
which must agree bit for bit in the indices."""
import numpy as np
import pytest

from paper_1309_0100_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fr():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1309_0100_b200 import build
    build.build()
    import paper_1309_0100_b200 as fr
    fr.lib()
    return fr


def _dev(*arrays):
    import torch
    return [None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]


def fused_peaks(fr, t, x, w, base, f0, df, K, k):
    dt, dx, dw, db = _dev(t, x, w, base if base is not None and base.shape[0] else None)
    z, idx, count = fr.fredec_scan_topk(dt, dx, dw, db, f0, df, K, k, want_z=False)
    assert z is None
    return idx.cpu().numpy(), count


def two_kernel_peaks(fr, t, x, w, base, f0, df, K, k):
    dt, dx, dw, db = _dev(t, x, w, base if base is not None and base.shape[0] else None)
    z, idx, count = fr.fredec_scan_topk(dt, dx, dw, db, f0, df, K, k)
    return z.cpu().numpy(), idx.cpu().numpy(), count


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_fused_peaks_equal_oracle_configs_1_to_3(fr, oracle_mod, cfg):
    wl = inputs.config(cfg)
    t, x, w, base = wl.series(0)
    z_ref = oracle_mod.scan(t, x, w, base, wl.f0, wl.df, wl.K, threads=0)
    idx_ref, cnt_ref = oracle_mod.topk(z_ref, wl.topk)
    idx, cnt = fused_peaks(fr, t, x, w, base, wl.f0, wl.df, wl.K, wl.topk)
    assert cnt == cnt_ref and idx.tolist() == idx_ref.tolist()
    assert fr.fredec_last_launches() < 6  # prep, table, scan (+ tail solve), merge: no top-k scan kernel


def test_fused_peaks_config4_full_size(fr, oracle_mod):
    """Config 4 as bench.py launches it (one series, left-over rounds shared between CTAs and finished by the
    tail-solve kernel): the fused indices equal the oracle's peaks of the library's own periodogram (whose
    parity with the oracle is test_config4_full_size_sampled)."""
    wl = inputs.config(4)
    t, x, w, base = wl.series(0)
    z, idx2, cnt2 = two_kernel_peaks(fr, t, x, w, base, wl.f0, wl.df, wl.K, wl.topk)
    idx, cnt = fused_peaks(fr, t, x, w, base, wl.f0, wl.df, wl.K, wl.topk)
    idx_ref, cnt_ref = oracle_mod.topk(z, wl.topk)
    assert cnt == cnt_ref == cnt2 and idx.tolist() == idx_ref.tolist() == idx2.tolist()
    # more peaks than any single warp list sees, and k at the fused maximum
    idx, cnt = fused_peaks(fr, t, x, w, base, wl.f0, wl.df, wl.K, 32)
    idx_ref, cnt_ref = oracle_mod.topk(z, 32)
    assert cnt == cnt_ref and idx.tolist() == idx_ref.tolist()


def test_fused_peaks_config5_reduced_batch(fr, oracle_mod):
    wl = inputs.config(5, B=40, K=20_000)
    z_ref = oracle_mod.scan_batched(wl.t, wl.x, wl.w, wl.base_funcs, wl.f0, wl.df, wl.K, threads=0)
    dt, dx, dw, db = _dev(wl.t, wl.x, wl.w, wl.base_funcs)
    z, idx = fr.fredec_scan_topk_batched(dt, dx, dw, db, wl.f0, wl.df, wl.K, wl.topk, want_z=False)
    assert z is None
    idx = idx.cpu().numpy()
    for b in range(wl.B):
        assert idx[b].tolist() == oracle_mod.topk(z_ref[b], wl.topk)[0].tolist(), f"series {b}"


@pytest.mark.slow
def test_fused_peaks_config5_full_size(fr, oracle_mod):
    """4096 x 500 x 100 000 as bench.py launches it: fused indices == the two-kernel path's, all series; and
    == the oracle's peaks of the library periodogram on sampled series."""
    wl = inputs.config(5)
    dt, dx, dw, db = _dev(wl.t, wl.x, wl.w, wl.base_funcs)
    _, idx = fr.fredec_scan_topk_batched(dt, dx, dw, db, wl.f0, wl.df, wl.K, wl.topk, want_z=False)
    idx = idx.cpu().numpy()
    z, idx2 = fr.fredec_scan_topk_batched(dt, dx, dw, db, wl.f0, wl.df, wl.K, wl.topk)
    assert np.array_equal(idx, idx2.cpu().numpy())
    for b in (0, 1, 777, 2048, 4095):
        assert idx[b].tolist() == oracle_mod.topk(z[b].cpu().numpy(), wl.topk)[0].tolist()


@pytest.mark.parametrize("d", [0, 1, 2, 3, 4, 5, 6, 7, 8, 9])
@pytest.mark.parametrize("K,k", [(1, 1), (2, 1), (5, 3), (97, 10), (1000, 32), (4097, 7), (30_011, 20)])
def test_fused_peaks_every_tile_shape_and_ragged_grids(fr, oracle_mod, d, K, k):
    """Every kernel instantiation (run lengths 96 ... 16), grids shorter than a run, a unit, a round, and with
    ragged ends; k larger than the number of peaks (-1 padding) and at the fused maximum."""
    k = min(k, K)
    t, x, w, base = inputs.random_series(700 + d, 157, d)
    f0, df = 0.013, 0.0037
    z_ref = oracle_mod.scan(t, x, w, base, f0, df, K, threads=0)
    idx_ref, cnt_ref = oracle_mod.topk(z_ref, k)
    idx, cnt = fused_peaks(fr, t, x, w, base, f0, df, K, k)
    z, idx2, cnt2 = two_kernel_peaks(fr, t, x, w, base, f0, df, K, k)
    assert idx.tolist() == idx2.tolist() and cnt == cnt2
    assert cnt == cnt_ref and idx.tolist() == idx_ref.tolist()


def test_fused_peaks_many_short_series(fr, oracle_mod):
    """Series boundaries inside a CTA's range and CTA boundaries inside a series: rounds of 1, 2, 4 units with
    the observation split, several (series, CTA) pairs per series."""
    rng = np.random.Generator(np.random.PCG64(4242))
    for B, N, K, d, k in [(300, 40, 700, 1, 4), (7, 90, 9000, 2, 12), (1500, 24, 130, 0, 3), (150, 64, 2100, 9, 5)]:
        ts, xs, ws, bs = [], [], [], []
        for b in range(B):
            t, x, w, base = inputs.random_series(int(rng.integers(1 << 30)), N, d, t_span=50.0)
            ts.append(t); xs.append(x); ws.append(w); bs.append(base)
        t, x, w = np.stack(ts), np.stack(xs), np.stack(ws)
        base = np.stack(bs) if d else None
        dt, dx, dw, db = _dev(t, x, w, base)
        f0, df = 0.02, 0.0011
        _, idx = fr.fredec_scan_topk_batched(dt, dx, dw, db, f0, df, K, k, want_z=False)
        z, idx2 = fr.fredec_scan_topk_batched(dt, dx, dw, db, f0, df, K, k)
        idx, idx2, z = idx.cpu().numpy(), idx2.cpu().numpy(), z.cpu().numpy()
        assert np.array_equal(idx, idx2), (B, N, K, d)
        for b in range(0, B, max(1, B // 25)):
            z_ref = oracle_mod.scan(t[b], x[b], w[b], bs[b], f0, df, K, threads=0)
            assert idx[b].tolist() == oracle_mod.topk(z_ref, k)[0].tolist(), (B, N, K, d, b)


def test_fused_falls_back_beyond_its_limits(fr, oracle_mod):
    """k > 32 or more than one pass (d > 9): z_out = NULL still works, through a library-owned periodogram."""
    t, x, w, base = inputs.random_series(91, 300, 13)
    f0, df, K = 0.01, 0.002, 5000
    z_ref = oracle_mod.scan(t, x, w, base, f0, df, K, threads=0)
    idx, cnt = fused_peaks(fr, t, x, w, base, f0, df, K, 10)
    assert idx.tolist() == oracle_mod.topk(z_ref, 10)[0].tolist()
    t, x, w, base = inputs.random_series(92, 300, 2)
    z_ref = oracle_mod.scan(t, x, w, base, f0, df, K, threads=0)
    idx, cnt = fused_peaks(fr, t, x, w, base, f0, df, K, 100)
    assert idx.tolist() == oracle_mod.topk(z_ref, 100)[0].tolist()


def test_fused_peaks_host_pointers_and_repeatability(fr):
    wl = inputs.config(2)
    t, x, w, base = wl.series(0)
    z, idx_h, cnt_h = fr.fredec_scan_topk(t, x, w, base, wl.f0, wl.df, wl.K, wl.topk, want_z=False)
    assert z is None
    runs = [fused_peaks(fr, t, x, w, base, wl.f0, wl.df, wl.K, wl.topk)[0].tolist() for _ in range(3)]
    assert runs[0] == runs[1] == runs[2] == np.asarray(idx_h).tolist()
