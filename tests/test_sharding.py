"""Host logic of the multi-GPU path (frequency-range sharding + peak-list merge), on CPU with
gloo, world_size 2.  The per-rank periodograms come from the oracle here (no GPU)."""
import os
import socket
import sys

import numpy as np
import pytest

from paper_1309_0100_b200 import inputs, sharding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_grid_covers_grid_exactly():
    for K, world in [(10, 1), (10, 3), (7, 8), (2_000_000, 8), (100_003, 4)]:
        seen = []
        for r in range(world):
            s = sharding.shard_grid(1e-4, 1.5e-6, K, world, r)
            seen += list(range(s.k_lo, s.k_hi)) if K < 1000 else [(s.k_lo, s.k_hi)]
            assert s.K == (s.k_hi - s.k_lo) + s.halo_lo + s.halo_hi
            if s.k_hi > s.k_lo:
                assert s.f0 == sharding.grid_frequency(1e-4, 1.5e-6, s.k_lo - s.halo_lo)
        if K < 1000:
            assert seen == list(range(K))
        else:
            assert seen[0][0] == 0 and seen[-1][1] == K
            assert all(a[1] == b[0] for a, b in zip(seen, seen[1:]))


def test_weak_grid_ranges():
    s0 = sharding.weak_grid(0.01, 0.001, 100, 2, 0)
    s1 = sharding.weak_grid(0.01, 0.001, 100, 2, 1)
    assert (s0.k_lo, s0.k_hi, s0.halo_lo, s0.halo_hi, s0.K) == (0, 100, 0, 1, 101)
    assert (s1.k_lo, s1.k_hi, s1.halo_lo, s1.halo_hi, s1.K) == (100, 200, 1, 0, 101)


def test_merge_matches_single_range_peaks(oracle_mod):
    """Sharded top-k (with halos) == top-k of the whole periodogram, incl. a peak on a boundary."""
    wl = inputs.config(1, K=4000)
    t, x, w, base = wl.series(0)
    z = oracle_mod.scan(t, x, w, base, wl.f0, wl.df, wl.K)
    k = 10
    want = oracle_mod.topk(z, k)[0].tolist()
    for world in (2, 3, 7):
        per = -(-wl.K // world)
        # move a shard boundary onto the strongest peak to exercise the halo logic
        lists = []
        for r in range(world):
            s = sharding.shard_grid(wl.f0, wl.df, wl.K, world, r)
            zl = z[s.k_lo - s.halo_lo: s.k_hi + s.halo_hi]
            il = oracle_mod.topk(zl, min(k + 2, len(zl)))[0]
            lists.append(sharding.local_candidates(s, zl, il))
        assert sharding.merge_candidates(lists, k) == want
    # boundary exactly at the top peak
    top = want[0]
    for lo, hi in [(0, top), (top, wl.K)], [(0, top + 1), (top + 1, wl.K)]:
        lists = []
        for a, b in (lo, hi):
            s = sharding._with_halo(wl.f0, wl.df, wl.K, a, b)
            zl = z[s.k_lo - s.halo_lo: s.k_hi + s.halo_hi]
            lists.append(sharding.local_candidates(s, zl, oracle_mod.topk(zl, k + 2)[0]))
        assert sharding.merge_candidates(lists, k) == want


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = inputs.config(1, K=3000)
        t, x, w, base = wl.series(0)
        s = sharding.shard_grid(wl.f0, wl.df, wl.K, world, rank)
        zl = oracle.scan(t, x, w, base, s.f0, wl.df, s.K)      # this rank's range (+ halo)
        il = oracle.topk(zl, min(wl.topk + 2, s.K))[0]
        merged = sharding.gather_topk(s, zl, il, wl.topk)
        q.put((rank, merged))
    finally:
        dist.destroy_process_group()


def test_gloo_world2_gather_topk(oracle_mod):
    import torch.multiprocessing as mp
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    results = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl = inputs.config(1, K=3000)
    z = oracle_mod.scan(*wl.series(0), wl.f0, wl.df, wl.K)
    want = oracle_mod.topk(z, wl.topk)[0].tolist()
    # per-rank frequencies start from fl(f0 + k_lo df): same grid up to one rounding (S1)
    assert results[0] == want and results[1] == want
