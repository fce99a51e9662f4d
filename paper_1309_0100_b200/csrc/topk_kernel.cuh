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

int topk_pick_nblk(int64_t B, int64_t K, int sm_count);
// Launches 1 kernel (nblk == 1) or 2 kernels; *launches receives the number.
cudaError_t launch_topk(const TopkParams& p, int64_t B, cudaStream_t stream, int* launches);

}  // namespace fredec
