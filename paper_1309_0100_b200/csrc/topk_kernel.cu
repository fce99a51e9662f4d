// topk_kernel.cu -- step a11: peaks of the periodogram, reading S7.
//
// i is a peak iff z[i] > z[i-1] and z[i] >= z[i+1]; out-of-range neighbours and NaN count as
// -infinity.  Peaks are ranked by the TOTAL order (z descending, index ascending), so the
// top-k set and its order are unique and the result is bit-exact whatever the traversal order.
//
// Each warp streams its share of z once (coalesced; the +-1 neighbours come from L1) and keeps
// a sorted top-k list spread over its lanes' registers (rank r lives in slot r/32 of lane
// r%32).  A candidate is first compared with the list's k-th entry, so almost all peaks cost
// one comparison; the rare survivors are inserted with warp shuffles.  Warp lists are merged
// per CTA through shared memory, CTA lists by a second small kernel.  No atomics.
#include <cmath>
#include <cstdint>
#include "topk_kernel.cuh"

namespace fredec {

namespace {

#ifndef FREDEC_TOPK_THREADS
#define FREDEC_TOPK_THREADS 256
#endif
#ifndef FREDEC_TOPK_UN
#define FREDEC_TOPK_UN 4
#endif
constexpr int kTopkThreads = FREDEC_TOPK_THREADS;
constexpr int kTopkWarps = kTopkThreads / 32;
constexpr int64_t kEmptyIdx = INT64_MAX;

__device__ __forceinline__ bool beats(double za, int64_t ia, double zb, int64_t ib)
{
    return za > zb || (za == zb && ia < ib);
}
__device__ __forceinline__ double sanitize(double v) { return (v != v) ? -INFINITY : v; }
__device__ __forceinline__ int64_t shfl_i64(int64_t v, int src)
{
    return (int64_t)__shfl_sync(0xffffffffu, (long long)v, src);
}
__device__ __forceinline__ int64_t shfl_up_i64(int64_t v)
{
    return (int64_t)__shfl_up_sync(0xffffffffu, (long long)v, 1);
}

template <int SLOTS>
struct WarpList {
    double z[SLOTS];
    int64_t id[SLOTS];
    double thr_z;  // the k-th entry (rank k-1), broadcast to all lanes
    int64_t thr_i;
    int k, lane;

    __device__ __forceinline__ void init(int k_, int lane_)
    {
        k = k_;
        lane = lane_;
#pragma unroll
        for (int s = 0; s < SLOTS; ++s) {
            z[s] = -INFINITY;
            id[s] = kEmptyIdx;
        }
        thr_z = -INFINITY;
        thr_i = kEmptyIdx;
    }
    // all lanes call with the same candidate
    __device__ __forceinline__ void insert(double zc, int64_t ic)
    {
        if (!beats(zc, ic, thr_z, thr_i)) return;
        double carry_z = 0.0;  // entry of rank 32*s - 1 (lane 31 of the previous slot)
        int64_t carry_i = 0;
        bool carry_b = false;  // does the candidate beat that entry
#pragma unroll
        for (int s = 0; s < SLOTS; ++s) {
            const bool b = beats(zc, ic, z[s], id[s]);
            double pz = __shfl_up_sync(0xffffffffu, z[s], 1);
            int64_t pi = shfl_up_i64(id[s]);
            bool pb = (bool)__shfl_up_sync(0xffffffffu, (int)b, 1);
            if (lane == 0) {
                pz = carry_z;
                pi = carry_i;
                pb = (s == 0) ? false : carry_b;
            }
            carry_z = __shfl_sync(0xffffffffu, z[s], 31);
            carry_i = shfl_i64(id[s], 31);
            carry_b = (bool)__shfl_sync(0xffffffffu, (int)b, 31);
            if (b) {
                z[s] = pb ? pz : zc;
                id[s] = pb ? pi : ic;
            }
        }
        const int rk = k - 1;
        double tz = -INFINITY;
        int64_t ti = kEmptyIdx;
#pragma unroll
        for (int s = 0; s < SLOTS; ++s)
            if (s == rk / 32) {
                tz = __shfl_sync(0xffffffffu, z[s], rk % 32);
                ti = shfl_i64(id[s], rk % 32);
            }
        thr_z = tz;
        thr_i = ti;
    }
    // each lane proposes its own candidate (valid or not)
    __device__ __forceinline__ void offer(double zc, int64_t ic, bool valid)
    {
        unsigned m = __ballot_sync(0xffffffffu, valid && beats(zc, ic, thr_z, thr_i));
        while (m) {
            const int src = __ffs(m) - 1;
            m &= m - 1;
            insert(__shfl_sync(0xffffffffu, zc, src), shfl_i64(ic, src));
        }
    }
    __device__ __forceinline__ void store(double* dz, int64_t* di) const
    {
#pragma unroll
        for (int s = 0; s < SLOTS; ++s) {
            const int r = s * 32 + lane;
            if (r < k) {
                dz[r] = z[s];
                di[r] = id[s];
            }
        }
    }
};

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

template <int SLOTS>
__global__ void __launch_bounds__(kTopkThreads) topk_scan_kernel(TopkParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* sz = reinterpret_cast<double*>(smem_raw);
    int64_t* si = reinterpret_cast<int64_t*>(sz + kTopkWarps * p.k);
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t b = blockIdx.y, K = p.K;
    const double* z = p.z + b * K;
    // contiguous chunk of this CTA, a multiple of what the CTA covers per step
    constexpr int UN = FREDEC_TOPK_UN;                               // 16-byte loads in flight per thread
    constexpr int64_t kStep = kTopkThreads * 2;         // elements per CTA and sub-step
    int64_t chunk = (K + p.nblk - 1) / p.nblk;
    chunk = (chunk + kStep - 1) / kStep * kStep;
    const int64_t begin = (int64_t)blockIdx.x * chunk;
    const int64_t end = min(K, begin + chunk);

    WarpList<SLOTS> L;
    L.init(p.k, lane);
    if ((reinterpret_cast<uintptr_t>(z) & 15) == 0) {
        // each lane owns two adjacent elements per sub-step (one 16-byte load); their outer
        // neighbours come from the adjacent lanes, the warp's two outer neighbours from L1/L2
        for (int64_t base = begin + wid * 64; base < end; base += kStep * UN) {
            double2 v[UN];
            double lft[UN], rgt[UN];
#pragma unroll
            for (int u = 0; u < UN; ++u) {
                const int64_t i0 = base + u * kStep + 2 * lane;
                v[u] = make_double2(-INFINITY, -INFINITY);
                if (i0 + 1 < K) {
                    v[u] = *reinterpret_cast<const double2*>(z + i0);
                } else if (i0 < K) {
                    v[u].x = z[i0];
                }
                lft[u] = (lane == 0 && i0 > 0 && i0 < K) ? z[i0 - 1] : -INFINITY;
                rgt[u] = (lane == 31 && i0 + 2 < K) ? z[i0 + 2] : -INFINITY;
            }
#pragma unroll
            for (int u = 0; u < UN; ++u) {
                const int64_t i0 = base + u * kStep + 2 * lane;
                if (base + u * kStep >= end) break;  // warp-uniform
                const double a = sanitize(v[u].x), c = sanitize(v[u].y);
                const double up = __shfl_up_sync(0xffffffffu, c, 1), dn = __shfl_down_sync(0xffffffffu, a, 1);
                const double l = lane == 0 ? sanitize(lft[u]) : up;
                const double r = lane == 31 ? sanitize(rgt[u]) : dn;
                L.offer(a, i0, i0 < K && a > l && a >= c);
                L.offer(c, i0 + 1, i0 + 1 < K && c > a && c >= r);
            }
        }
    } else {
        for (int64_t base = begin + wid * 32; base < end; base += kTopkThreads) {
            const int64_t i = base + lane;
            bool peak = false;
            double v = -INFINITY;
            if (i < K) {
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
