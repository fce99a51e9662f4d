// topk_list.cuh -- the warp-level sorted top-k list of step a11 (peaks ranked by z descending, index
// ascending: a total order, so the result is unique whatever the order of insertion).  Shared by the
// peak-extraction kernels (topk_kernel.cu) and the scan kernel's fused epilogue (scan_mma_kernel.cu).
#pragma once
#include <cmath>
#include <cstdint>
#include <cuda_runtime.h>

namespace fredec {

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

}  // namespace fredec
