"""fredec_topk_noalloc against fredec_topk (GPU).

fredec_topk_noalloc serves programs that cannot let this library call cudaMalloc: a pipeline whose own
memory pool already owns the whole GPU (a library-side cudaMalloc then fails although the pool has room), a
service that cannot take the device-wide stall of an allocation, code running where the allocator is off
limits.  Its scratch memory is a fixed array built into libfredec_b200.so, shared by every call and never
cleared wholesale -- so the thing to check is that a call is not disturbed by what the previous call left
in that array.  Each case therefore makes two calls in a row (different inputs, then the first input
again) and compares every one with the allocating path, fredec_topk.  Indices and counts are integers: the
bar is exact equality, as in the other top-k tests.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not
hide the parity tests.  It passes alone in a fresh process (the first call does the per-device set-up) and
after the rest of the suite (the library's allocating workspace already exists by then).
"""
import numpy as np
import pytest

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


def _periodogram_like(K, seed, ties):
    rng = np.random.Generator(np.random.PCG64(seed))
    z = rng.gamma(1.0, 5.0, K)
    if ties:
        z = np.round(z, 1)                                   # coarse values: exact ties and plateaus
        z[rng.integers(0, K, 20)] = z.max() + 1.0            # tied global maxima
    z[rng.integers(0, K, 3)] = np.nan                        # NaN counts as -infinity
    return z


def _noalloc(fr, dz, k, idx, cnt, stream=None):
    import torch
    idx.fill_(-7)
    cnt.fill_(-7)
    fr.fredec_topk_noalloc(dz, k, idx, cnt, stream=stream)
    torch.cuda.synchronize()
    return idx[:k].cpu().numpy(), int(cnt.item())


# K spans one CTA (no scratch traffic), a few CTAs, the full 592-CTA grid and a ragged tail;
# k spans the three list widths (<= 32, <= 64, <= 128)
@pytest.mark.parametrize("K,k", [(3000, 5), (4097, 32), (50_001, 33), (300_000, 64), (1_000_003, 100),
                                 (2_000_000, 10), (5_000_000, 128)])
def test_two_calls_in_a_row_match_the_allocating_path(fr, K, k):
    import torch
    za = _periodogram_like(K, K + k, ties=True)
    zb = _periodogram_like(K, K + k + 1, ties=False)
    da, db = torch.from_numpy(za).cuda(), torch.from_numpy(zb).cuda()
    idx = torch.empty(k, dtype=torch.int64, device="cuda")   # the caller's buffers, reused by every call
    cnt = torch.empty(1, dtype=torch.int32, device="cuda")
    ref = {}
    for name, d in (("a", da), ("b", db)):
        ri, rc = fr.fredec_topk(d, k)
        ref[name] = (ri.cpu().numpy(), rc)
    for name, d in (("a", da), ("b", db), ("a", da)):        # b runs on a's leftovers, a on b's
        got_i, got_c = _noalloc(fr, d, k, idx, cnt)
        assert got_c == ref[name][1], (K, k, name)
        assert np.array_equal(got_i, ref[name][0]), (K, k, name)


def test_back_to_back_on_one_stream_without_sync_between(fr):
    """Two calls enqueued one after the other on a non-default stream, no host synchronisation between
    them: stream order alone must keep the second call's clearing of the ticket behind the first kernel."""
    import torch
    K, k = 1_500_000, 16
    d1 = torch.from_numpy(_periodogram_like(K, 1, ties=True)).cuda()
    d2 = torch.from_numpy(_periodogram_like(K, 2, ties=True)).cuda()
    r1, c1 = fr.fredec_topk(d1, k)
    r2, c2 = fr.fredec_topk(d2, k)
    i1 = torch.full((k,), -7, dtype=torch.int64, device="cuda")
    i2 = torch.full((k,), -7, dtype=torch.int64, device="cuda")
    n1 = torch.full((1,), -7, dtype=torch.int32, device="cuda")
    n2 = torch.full((1,), -7, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    fr.fredec_topk_noalloc(d1, k, i1, n1, stream=s)
    fr.fredec_topk_noalloc(d2, k, i2, n2, stream=s)
    s.synchronize()
    assert int(n1.item()) == c1 and torch.equal(i1, r1)
    assert int(n2.item()) == c2 and torch.equal(i2, r2)


def test_misaligned_input_and_few_peaks(fr):
    """A row that is not 16-byte aligned takes the scalar path; a monotone series has one peak: unused
    slots are -1 and the count says so."""
    import torch
    K, k = 100_001, 8
    buf = torch.from_numpy(_periodogram_like(K + 1, 9, ties=True)).cuda()
    dz = buf[1:]                                            # 8-byte aligned only
    assert dz.data_ptr() % 16 == 8
    ri, rc = fr.fredec_topk(dz.clone(), k)
    idx = torch.empty(k, dtype=torch.int64, device="cuda")
    cnt = torch.empty(1, dtype=torch.int32, device="cuda")
    for _ in range(2):
        got_i, got_c = _noalloc(fr, dz, k, idx, cnt)
        assert got_c == rc and np.array_equal(got_i, ri.cpu().numpy())
    mono = torch.arange(K, dtype=torch.float64, device="cuda")
    for _ in range(2):
        got_i, got_c = _noalloc(fr, mono, k, idx, cnt)
        assert got_c == 1 and got_i.tolist() == [K - 1] + [-1] * (k - 1)


def test_limits_and_argument_errors(fr):
    import torch
    z = torch.zeros(4000, dtype=torch.float64, device="cuda")
    cnt = torch.empty(1, dtype=torch.int32, device="cuda")
    big = torch.empty(fr.FREDEC_TOPK_NOALLOC_K_MAX + 1, dtype=torch.int64, device="cuda")

    def code(fn):
        with pytest.raises(fr.FredecError) as e:
            fn()
        return e.value.code

    assert code(lambda: fr.fredec_topk_noalloc(z, fr.FREDEC_TOPK_NOALLOC_K_MAX + 1, big, cnt)) == fr.FREDEC_ELIMIT
    assert code(lambda: fr.fredec_topk_noalloc(z[:4], 5, big, cnt)) == fr.FREDEC_EINVAL       # k > K
    assert code(lambda: fr.fredec_topk_noalloc(z, 0, big, cnt)) == fr.FREDEC_EINVAL
    host_idx = torch.empty(8, dtype=torch.int64)                                              # a host buffer
    assert code(lambda: fr.fredec_topk_noalloc(z, 8, host_idx, cnt)) == fr.FREDEC_EINVAL
    assert 0 < fr.fredec_topk_noalloc_scratch_bytes() <= 2 * 1024 * 1024                      # "modest"
