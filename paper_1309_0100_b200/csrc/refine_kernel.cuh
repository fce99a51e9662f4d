// refine_kernel.cuh -- local multifrequency fit (section 3, eq. 17): Gauss-Newton
// over the frequencies with the linear coefficients re-fitted exactly at every iteration.
#pragma once
#include "common.cuh"

namespace fredec {

// rows [3n+1][N] of the model functions at the current frequencies, times centred on t0:
//   row 0 = 1, rows 2k+1 / 2k+2 = cos / sin(2 pi f_k t'), and, when theta != nullptr, rows 2n+1+k =
//   d mu / d f_k = 2 pi t' (-a_k sin + b_k cos) with (a_k, b_k) = theta[2k+1], theta[2k+2]   (eq. 2's derivative)
cudaError_t launch_model_rows(const double* t, int64_t N, double t0, const double* freqs, int n, const double* theta,
                              double* rows, cudaStream_t stream);

// Solves the normal equations held in the augmented Gram matrix A [(m+1)][(m+1)] (last row/column =
// <x phi>, <x^2>) by Cholesky: theta [m] = Q^{-1} g, out2[0] = l = D - |L^{-1} g|^2,
// out2[1] = status (0, or -3 when a pivot^2 <= 1e-12 x its diagonal).  One CTA.  m <= 76.
cudaError_t launch_chol_solve(const double* A, int m, double* theta, double* out2, cudaStream_t stream);

// Gauss-Newton step from the Gram matrix G [(m+1)][(m+1)] of (Phi [2n+1], dmu/df [n], x), m = 3n+1, and
// the linear fit theta: g_f = <(x - mu) J> (its theta part vanishes), Q_f = <J J^T>,
// step = Q_f^{-1} g_f; df_out [n] = its frequency part, clamped to +-max_step.  out2 as above.
cudaError_t launch_gn_step(const double* G, int n, const double* theta, double max_step, double* df_out,
                           double* out2, cudaStream_t stream);

// freqs[k] += df[k]
cudaError_t launch_axpy_small(double* freqs, const double* df, int n, cudaStream_t stream);

}  // namespace fredec
