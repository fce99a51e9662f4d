// topk_kernel.cuh -- launch interface of the peak-extraction kernels.
#pragma once
#include "common.cuh"

namespace fredec {

struct TopkParams {
    const double* z;   // [B][K]
    int64_t* idx_out;  // [B][k]
    int* count_out;    // [B] number of peaks found (<= k)
    double* part_z;    // workspace [B][nblk][k]   (unused when nblk == 1)
    int64_t* part_i;   // workspace [B][nblk][k]
    int64_t K;
    int k;
    int nblk;  // CTAs per series in the first kernel
};

// Second stage of the peak extraction fused into the scan (scan_mma_kernel.cuh): per series, merges the MMA
// warps' lists of every (series, CTA) pair and settles the first / last grid point of every unit from the
// edge records.
struct FusedMergeParams {
    const double* list_z;    // [groups][nw][k]
    const int64_t* list_i;   // < 0 or INT64_MAX: empty entry
    const double* edges;     // [B][U][4]
    const SeriesInfo* info;  // [B]
    int64_t* idx_out;        // [B][k]
    int* count_out;          // [B]
    int64_t K, U, T;         // grid points, units per series, total units
    int64_t unit_points;     // grid points per unit
    int k, nw, grid;         // list length, MMA warps per CTA, CTAs of the scan
    int shared, Rt, tail_group0;
};
cudaError_t launch_fused_merge(const FusedMergeParams& p, int64_t B, cudaStream_t stream);

int topk_pick_nblk(int64_t B, int64_t K, int sm_count);
// Launches 1 kernel (nblk == 1) or 2 kernels; *launches receives the number.
cudaError_t launch_topk(const TopkParams& p, int64_t B, cudaStream_t stream, int* launches);

}  // namespace fredec
