// stat_kernel.cuh -- the paper-normalised statistic, the single-frequency FAP and the pieces the
// phase-1 driver needs around the scan.
#pragma once
#include "common.cuh"

namespace fredec {

// z[k] = -(N_H / 2) log1p(-dchi2[k] / chi2_base)      (PAPER.md:89-95 eq. 8, :106 eq. 10; reading G1)
cudaError_t launch_zstat(const double* dchi2, int64_t K, double chi2_base, double NH, double* z_out,
                         cudaStream_t stream);

// fap[k] = min(1, A1 W exp(-z[k]) sqrt(z[k]))            (eq. 13 with n = 1)
cudaError_t launch_fap1(const double* z, int64_t K, double W, double A1, double* fap_out, cudaStream_t stream);

// *flag (device int) = 1 if any of v[0..n) is NaN or infinite, else 0
cudaError_t launch_finite_flag(const double* v, int64_t n, int* flag, cudaStream_t stream);

// out[0] = T_eff = sqrt(4 pi Var(t)), out[1] = Var(t) (weighted), out[2] = weighted mean of t
// out[3] = status (0 or FREDEC_EDATA as a double).  One CTA, fixed-order sums.
cudaError_t launch_bandwidth(const double* t, const double* w, int64_t N, double* out4, cudaStream_t stream);

// base [1 + 2m][N]: row 0 = 1, rows 2j+1 / 2j+2 = cos / sin(2 pi f_j t)  (eq. 2 with the
// frequencies fixed), phases reduced exactly before the evaluation.  freqs: m doubles in device memory.
cudaError_t launch_sin_base(const double* t, int64_t N, const double* freqs, int m, double* base_out,
                            cudaStream_t stream);

// For the k peak indices idx[j] (-1 = unused): out[j] = (z, fap) of dchi2[idx[j]], as in zstat / fap1, with
// chi2_base read from the scan's per-series record in device memory (so that no host round trip separates
// the scan from its peak statistics).
cudaError_t launch_peak_stats(const double* dchi2, const int64_t* idx, int k, const SeriesInfo* info, double NH,
                              double W, double A1, double* out2k, cudaStream_t stream);

}  // namespace fredec
