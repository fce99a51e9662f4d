// topk_kernel.cu -- step a11: peaks of the periodogram, reading S7.
//
// i is a peak iff z[i] > z[i-1] and z[i] >= z[i+1]; out-of-range neighbours and NaN count as
// -infinity.  Peaks are ranked by the TOTAL order (z descending, index ascending), so the
// top-k set and its order are unique and the result is bit-exact whatever the traversal order.
//
// Each warp streams a contiguous segment of z once (16-byte loads, several in flight) and keeps
// a sorted top-k list spread over its lanes' registers (rank r lives in slot r/32 of lane
// r%32).  A whole step of 64 points is first compared with the list's k-th entry, so almost all
// points cost a comparison and a share of one vote; the rare survivors are tested for being peaks
// and inserted with warp shuffles.  Warp lists are merged
// per CTA through shared memory, CTA lists by a second small kernel.  No atomics.
#include <cmath>
#include <cstdint>
#include "topk_kernel.cuh"
#include "topk_list.cuh"

namespace fredec {

namespace {

#ifndef FREDEC_TOPK_THREADS
#define FREDEC_TOPK_THREADS 256
#endif
constexpr int kTopkThreads = FREDEC_TOPK_THREADS;
constexpr int kTopkWarps = kTopkThreads / 32;
// Merge the CTA's warp lists (smem) into warp 0's list; then write either the final indices
// (last stage) or this CTA's partial list.
template <int SLOTS>
__device__ void cta_merge_and_write(WarpList<SLOTS>& L, const TopkParams& p, int64_t b, int blk, bool final_stage,
                                    double* sz, int64_t* si)
{
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31, k = p.k;
    L.store(sz + wid * k, si + wid * k);
    __syncthreads();
    if (wid != 0) return;
    const int total = kTopkWarps * k;
    for (int e = k + lane; e - lane < total; e += 32) {  // warp 0's own entries are already in L
        const bool valid = e < total;
        L.offer(valid ? sz[e] : -INFINITY, valid ? si[e] : kEmptyIdx, valid && si[valid ? e : 0] != kEmptyIdx);
    }
    if (final_stage) {
        int found = 0;
#pragma unroll
        for (int s = 0; s < SLOTS; ++s) {
            const int r = s * 32 + lane;
            const bool has = r < k && L.id[s] != kEmptyIdx;
            if (r < k) p.idx_out[b * k + r] = has ? L.id[s] : -1;
            found += __popc(__ballot_sync(0xffffffffu, has));
        }
        if (lane == 0) p.count_out[b] = found;
    } else {
        L.store(p.part_z + (b * p.nblk + blk) * k, p.part_i + (b * p.nblk + blk) * k);
    }
}

// 16-byte load of the two grid points [i, i + 1] of a row of K points (i even, the row 16-byte aligned);
// points at or beyond K read as -infinity.
__device__ __forceinline__ double2 load_pair(const double* __restrict__ z, int64_t i, int64_t K)
{
    if (i + 1 < K) return *reinterpret_cast<const double2*>(z + i);
    return make_double2(i < K ? z[i] : -INFINITY, -INFINITY);
}

template <int SLOTS>
__global__ void __launch_bounds__(kTopkThreads) topk_scan_kernel(TopkParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* sz = reinterpret_cast<double*>(smem_raw);
    int64_t* si = reinterpret_cast<int64_t*>(sz + kTopkWarps * p.k);
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t b = blockIdx.y, K = p.K;
    const double* z = p.z + b * K;
    // contiguous chunk of this CTA, cut into one contiguous segment per warp (multiples of 64 points)
    constexpr int64_t kStep = 64;  // points per warp and step: one 16-byte load per lane
    int64_t chunk = (K + p.nblk - 1) / p.nblk;
    chunk = (chunk + kStep * kTopkWarps - 1) / (kStep * kTopkWarps) * (kStep * kTopkWarps);
    const int64_t begin = (int64_t)blockIdx.x * chunk;
    const int64_t end = min(K, begin + chunk);
    const int64_t seg = chunk / kTopkWarps;
    const int64_t s0 = begin + wid * seg, s1 = min(end, s0 + seg);

    WarpList<SLOTS> L;
    L.init(p.k, lane);
    if ((reinterpret_cast<uintptr_t>(z) & 15) == 0) {
        // The warp walks its segment in steps of 64 points, kRing - 1 loads ahead.  A step is looked at
        // closely only if some lane's point could enter the list (z >= the list's k-th entry; until k peaks
        // are known that entry is -infinity and every step is): almost every step costs one load, two
        // comparisons and a vote.  The neighbours of a lane's two points are its own, the adjacent
        // lanes' (shuffles) and, at the warp's edges, the previous / next step's.
        constexpr int kRing = 4;
        double2 ring[kRing];
#pragma unroll
        for (int u = 0; u < kRing - 1; ++u) ring[u] = load_pair(z, s0 + u * kStep + 2 * lane, K);
        double prev_c = s0 > 0 && s0 < K ? z[s0 - 1] : -INFINITY;  // the point before the step (lane 31's view)
        for (int64_t base = s0; base < s1; base += kStep * kRing) {
#pragma unroll
            for (int u = 0; u < kRing; ++u) {
                const int64_t sb = base + u * kStep;  // this step
                if (sb >= s1) break;                  // warp-uniform
                ring[(u + kRing - 1) % kRing] = load_pair(z, sb + (kRing - 1) * kStep + 2 * lane, K);
                const double2 cur = ring[u], nxt = ring[(u + 1) % kRing];
                if (__any_sync(0xffffffffu, cur.x >= L.thr_z || cur.y >= L.thr_z)) {
                    const int64_t i0 = sb + 2 * lane;
                    const double a = sanitize(cur.x), c = sanitize(cur.y);
                    const double up = __shfl_up_sync(0xffffffffu, c, 1), dn = __shfl_down_sync(0xffffffffu, a, 1);
                    const double first_next = sanitize(__shfl_sync(0xffffffffu, nxt.x, 0));
                    const double last_prev = sanitize(__shfl_sync(0xffffffffu, prev_c, 31));
                    const double l = lane == 0 ? last_prev : up;
                    const double r = lane == 31 ? first_next : dn;
                    L.offer(a, i0, i0 < s1 && a > l && a >= c);
                    L.offer(c, i0 + 1, i0 + 1 < s1 && c > a && c >= r);
                }
                prev_c = cur.y;
            }
        }
    } else {
        for (int64_t base = s0 + lane; base - lane < s1; base += 32) {
            const int64_t i = base;
            bool peak = false;
            double v = -INFINITY;
            if (i < s1) {
                v = sanitize(z[i]);
                const double l = i > 0 ? sanitize(z[i - 1]) : -INFINITY;
                const double r = i + 1 < K ? sanitize(z[i + 1]) : -INFINITY;
                peak = v > l && v >= r;
            }
            L.offer(v, i, peak);
        }
    }
    cta_merge_and_write<SLOTS>(L, p, b, blockIdx.x, p.nblk == 1, sz, si);
}

template <int SLOTS>
__global__ void __launch_bounds__(kTopkThreads) topk_merge_kernel(TopkParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* sz = reinterpret_cast<double*>(smem_raw);
    int64_t* si = reinterpret_cast<int64_t*>(sz + kTopkWarps * p.k);
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t b = blockIdx.x;
    const int64_t total = (int64_t)p.nblk * p.k;
    const double* cz = p.part_z + b * total;
    const int64_t* ci = p.part_i + b * total;
    WarpList<SLOTS> L;
    L.init(p.k, lane);
    for (int64_t base = wid * 32; base < total; base += kTopkThreads) {
        const int64_t e = base + lane;
        const bool valid = e < total && ci[e] != kEmptyIdx;
        L.offer(valid ? cz[e] : -INFINITY, valid ? ci[e] : kEmptyIdx, valid);
    }
    cta_merge_and_write<SLOTS>(L, p, b, 0, true, sz, si);
}

// CTA that owns unit g of the scan's contiguous partition [c T / grid, (c + 1) T / grid)
__device__ __forceinline__ int unit_owner(int64_t g, int64_t T, int grid)
{
    int c = (int)(g * grid / T);
    while (c + 1 < grid && (int64_t)(c + 1) * T / grid <= g) ++c;
    while (c > 0 && (int64_t)c * T / grid > g) --c;
    return c;
}

__global__ void __launch_bounds__(kTopkThreads) topk_fused_merge_kernel(FusedMergeParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* sz = reinterpret_cast<double*>(smem_raw);
    int64_t* si = reinterpret_cast<int64_t*>(sz + kTopkWarps * p.k);
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t b = blockIdx.x;
    WarpList<1> L;
    L.init(p.k, lane);
    if (p.info[b].status == 0) {
        // the lists of the groups that hold this series: two ranges [g0, g1) and [h0, h1)
        int64_t g0, g1, h0 = 0, h1 = 0;
        if (p.shared) {
            g0 = 0;
            g1 = p.grid;
            h0 = p.tail_group0;
            h1 = h0 + p.Rt;
        } else {
            g0 = b + unit_owner(b * p.U, p.T, p.grid);
            g1 = b + unit_owner((b + 1) * p.U - 1, p.T, p.grid) + 1;
        }
        const int64_t per = (int64_t)p.nw * p.k;
        const int64_t n1 = (g1 - g0) * per, total = n1 + (h1 - h0) * per;
        for (int64_t base = (int64_t)wid * 32; base < total; base += kTopkThreads) {
            const int64_t e = base + lane;
            bool valid = e < total;
            double zc = -INFINITY;
            int64_t ic = kEmptyIdx;
            if (valid) {
                const int64_t at = e < n1 ? g0 * per + e : h0 * per + (e - n1);
                ic = __ldcg(p.list_i + at);
                valid = ic >= 0 && ic != kEmptyIdx;
                if (valid) zc = __ldcg(p.list_z + at);
            }
            L.offer(zc, ic, valid);
        }
        // unit boundaries: the first point of unit u is a peak iff first_ok and z_first > z_last of unit u - 1;
        // the last point iff last_ok and z_last >= z_first of unit u + 1 (outside the grid: -infinity)
        const double* ed = p.edges + b * p.U * 4;
        for (int64_t base = (int64_t)wid * 32; base < p.U; base += kTopkThreads) {
            const int64_t u = base + lane;
            bool pf = false, pl = false;
            double zf = -INFINITY, zl = -INFINITY;
            if (u < p.U) {
                const double2 f = __ldcg(reinterpret_cast<const double2*>(ed + u * 4));
                const double2 l = __ldcg(reinterpret_cast<const double2*>(ed + u * 4 + 2));
                const double before = u > 0 ? __ldcg(ed + (u - 1) * 4 + 2) : -INFINITY;
                const double after = u + 1 < p.U ? __ldcg(ed + (u + 1) * 4) : -INFINITY;
                zf = f.x;
                zl = l.x;
                pf = f.y != 0.0 && zf > before;
                pl = l.y != 0.0 && zl >= after;
            }
            L.offer(zf, u * p.unit_points, pf);
            L.offer(zl, (u + 1) * p.unit_points - 1, pl);
        }
    }
    TopkParams tp;
    tp.z = nullptr;
    tp.idx_out = p.idx_out;
    tp.count_out = p.count_out;
    tp.part_z = nullptr;
    tp.part_i = nullptr;
    tp.K = p.K;
    tp.k = p.k;
    tp.nblk = 1;
    cta_merge_and_write<1>(L, tp, b, 0, true, sz, si);
}

template <int SLOTS>
cudaError_t launch_slots(const TopkParams& p, int64_t B, cudaStream_t stream, int* launches)
{
    const size_t smem = (size_t)kTopkWarps * p.k * 16;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(topk_scan_kernel<SLOTS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)smem);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(topk_merge_kernel<SLOTS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    topk_scan_kernel<SLOTS><<<dim3((unsigned)p.nblk, (unsigned)B), kTopkThreads, smem, stream>>>(p);
    *launches = 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess || p.nblk == 1) return e;
    topk_merge_kernel<SLOTS><<<(unsigned)B, kTopkThreads, smem, stream>>>(p);
    *launches = 2;
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_fused_merge(const FusedMergeParams& p, int64_t B, cudaStream_t stream)
{
    if (p.k < 1 || p.k > 32) return cudaErrorInvalidValue;
    const size_t smem = (size_t)kTopkWarps * p.k * 16;
    topk_fused_merge_kernel<<<(unsigned)B, kTopkThreads, smem, stream>>>(p);
    return cudaGetLastError();
}

int topk_pick_nblk(int64_t B, int64_t K, int sm_count)
{
    // enough CTAs to cover the chip a few times over, at least ~4096 elements each
    int64_t want = (4 * (int64_t)sm_count + B - 1) / B;
    int64_t most = (K + 4095) / 4096;
    int64_t n = want < most ? want : most;
    if (n < 1) n = 1;
    if (n > 4096) n = 4096;
    return (int)n;
}

cudaError_t launch_topk(const TopkParams& p, int64_t B, cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (p.k <= 32) return launch_slots<1>(p, B, stream, launches);
    if (p.k <= 64) return launch_slots<2>(p, B, stream, launches);
    if (p.k <= 128) return launch_slots<4>(p, B, stream, launches);
    if (p.k <= 256) return launch_slots<8>(p, B, stream, launches);
    if (p.k <= 512) return launch_slots<16>(p, B, stream, launches);
    return launch_slots<32>(p, B, stream, launches);
}

}  // namespace fredec
