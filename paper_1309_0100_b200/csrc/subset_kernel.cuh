// subset_kernel.cuh -- linear multifrequency fits for every subset of a frequency pool: the
// l_m(f') of PAPER.md:81 (eq. 7) / :158-175 (section 3) that phase 2 evaluates for all
// 2^n - 1 subsets, with the frequencies held fixed.
#pragma once
#include "common.cuh"

namespace fredec {

// Augmented Gram matrix A [(M+1)][(M+1)], M = 2n+1 model functions (row-major, symmetric):
//   A[a][b] = <phi_a phi_b>,  A[a][M] = <x phi_a>,  A[M][M] = <x^2> = D   (eqs. 15, 16)
// basis [M][N] = the functions' values (1, cos w_1 t, sin w_1 t, ...).  Fixed-order sums.
cudaError_t launch_gram(const double* basis, const double* x, const double* w, int64_t N, int M, double* A,
                        cudaStream_t stream);

// l_out[mask] = D - |L^{-1} g|^2 for the sub-model {1} + {cos, sin of frequency j : bit j of mask},
// mask = 0 .. 2^n - 1.  Depth-first over the subsets, one warp per subtree, factor rows
// in shared memory.
cudaError_t launch_subset_fits(const double* A, int n, double* l_out, int sm_count, cudaStream_t stream);

}  // namespace fredec
