// refine_kernel.cuh -- local multifrequency fits (section 3, eq. 17): Gauss-Newton
// over the frequencies with the linear coefficients re-fitted exactly at every iteration, for a batch of
// tuples drawn from one pool (phase 2 tabulates l_{m,loc} for the subsets of the pool;
// "many entirely independent instances of the fitting subroutine").
#pragma once
#include "common.cuh"

namespace fredec {

struct RefineParams {
    const double* t;       // [N]
    const double* x;       // [N]
    const double* w;       // [N]
    const double* bw;      // [4] output of launch_bandwidth: T_eff, Var t, weighted mean of t, status
    const double* pool;    // [n_pool] starting frequencies
    const int64_t* masks;  // [T] bit j selects pool[j]; nullptr: every tuple is the whole pool
    double* freqs_out;     // [T][n_pool] refined frequencies (pool[j] where bit j is clear)
    double* l_out;         // [T] min chi2 at the returned frequencies (0 on failure)
    int32_t* iters_out;    // [T] frequency updates made
    int32_t* status_out;   // [T] 0, -3 (singular normal equations) or -2 (bad t / w)
    int64_t N;
    int n_pool, max_iter;
    double tol;
};

// One CTA per tuple; m_max >= the largest number of selected frequencies of any tuple (sizes the shared
// memory).  Model: constant + m sinusoids (eq. 2), times centred on their weighted mean.
// Per iteration: Gram matrix of (1, cos, sin, t' cos, t' sin, x) in one sweep -> exact linear fit by
// Cholesky (eq. 14) -> Q_f, g_f of eq. 17 from the same matrix -> step Q_f^{-1} g_f, its frequency part
// clamped to +-0.5 / T_eff (reading R1) -> stop when max |step| T_eff <= tol (reading R2).
cudaError_t launch_refine_batched(const RefineParams& p, int64_t T, int m_max, cudaStream_t stream);
size_t refine_batched_smem(int m_max);
// Tuple masks that live on the device: out2[0] = the largest tuple size, out2[1] = how many masks are out of
// range (negative, or a bit at or beyond n_pool).  out2: two ints of device memory.
cudaError_t launch_mask_stats(const int64_t* masks, int64_t T, int n_pool, int* out2, cudaStream_t stream);

}  // namespace fredec
