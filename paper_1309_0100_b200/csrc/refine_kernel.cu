// refine_kernel.cu -- see refine_kernel.cuh.  Small latency-sized kernels: the systems have at most
// 3n + 1 <= 76 unknowns; the sums over the observations are formed by gram_kernel (subset_kernel.cu).
#include "refine_kernel.cuh"

namespace fredec {

namespace {

constexpr int kRowsThreads = 256;
constexpr int kSolveThreads = 128;
constexpr int kMaxUnknowns = 76;  // 3 * 25 + 1
constexpr double kTauRefine = 1e-12;

__global__ void __launch_bounds__(kRowsThreads) model_rows_kernel(const double* __restrict__ t, int64_t N, double t0,
                                                                 const double* __restrict__ freqs, int n,
                                                                 const double* __restrict__ theta,
                                                                 double* __restrict__ rows)
{
    const int64_t i = (int64_t)blockIdx.x * kRowsThreads + threadIdx.x;
    if (i >= N) return;
    const double tc = t[i] - t0;
    rows[i] = 1.0;
    for (int k = 0; k < n; ++k) {
        double s, c;
        sincospi(2.0 * frac_prod(freqs[k], tc), &s, &c);
        rows[(int64_t)(2 * k + 1) * N + i] = c;
        rows[(int64_t)(2 * k + 2) * N + i] = s;
        if (theta != nullptr) {
            const double a = theta[2 * k + 1], b = theta[2 * k + 2];
            rows[(int64_t)(2 * n + 1 + k) * N + i] = 6.283185307179586477 * tc * fma(b, c, -(a * s));
        }
    }
}

// In-place Cholesky of the leading m x m block of S (lower triangle, leading dimension LD) with row m
// carried along as a right-hand side: afterwards S[i][j] = L[i][j], S[m][j] = a_j =
// (L^{-1} g)_j and S[m][m] = D - |a|^2.  diag0[j] = the original diagonal.  Returns 0 or -3.
__device__ int chol_with_rhs(double* S, int LD, int m, const double* diag0, int* status_sm)
{
    const int tid = threadIdx.x;
    if (tid == 0) *status_sm = 0;
    __syncthreads();
    for (int j = 0; j < m; ++j) {
        const double piv = S[j * LD + j];
        if (!(piv > kTauRefine * diag0[j])) {  // uniform across the CTA
            if (tid == 0) *status_sm = -3;
            break;
        }
        const double inv = rsqrt(piv);
        __syncthreads();
        for (int i = j + tid; i <= m; i += kSolveThreads) S[i * LD + j] = i == j ? piv * inv : S[i * LD + j] * inv;
        __syncthreads();
        const int rows = m - j;  // rows j+1 .. m
        for (int e = tid; e < rows * rows; e += kSolveThreads) {
            const int i = j + 1 + e / rows, k = j + 1 + e % rows;
            if (k <= i) S[i * LD + k] = fma(-S[i * LD + j], S[k * LD + j], S[i * LD + k]);
        }
        __syncthreads();
    }
    __syncthreads();
    return *status_sm;
}

__global__ void __launch_bounds__(kSolveThreads) chol_solve_kernel(const double* __restrict__ A, int m,
                                                                  double* __restrict__ theta, double* __restrict__ out2)
{
    __shared__ double S[(kMaxUnknowns + 1) * (kMaxUnknowns + 1)];
    __shared__ double diag0[kMaxUnknowns + 1];
    __shared__ int status;
    const int LD = m + 1;
    for (int e = threadIdx.x; e < (m + 1) * (m + 1); e += kSolveThreads) {
        const int i = e / (m + 1), k = e % (m + 1);
        S[i * LD + k] = A[e];
        if (i == k) diag0[i] = A[e];
    }
    __syncthreads();
    const int rc = chol_with_rhs(S, LD, m, diag0, &status);
    if (threadIdx.x == 0) {
        if (rc == 0) {
            // theta = L^{-T} a by back substitution
            for (int j = m - 1; j >= 0; --j) {
                double v = S[m * LD + j];
                for (int i = j + 1; i < m; ++i) v = fma(-S[i * LD + j], theta[i], v);
                theta[j] = v / S[j * LD + j];
            }
        }
        out2[0] = rc == 0 ? fmax(S[m * LD + m], 0.0) : 0.0;
        out2[1] = (double)rc;
    }
}

__global__ void __launch_bounds__(kSolveThreads) gn_step_kernel(const double* __restrict__ G, int n,
                                                               const double* __restrict__ theta, double max_step,
                                                               double* __restrict__ df_out, double* __restrict__ out2)
{
    __shared__ double S[(kMaxUnknowns + 1) * (kMaxUnknowns + 1)];
    __shared__ double diag0[kMaxUnknowns + 1];
    __shared__ double step[kMaxUnknowns];
    __shared__ int status;
    const int m = 3 * n + 1, lin = 2 * n + 1, LDG = m + 1, LD = m + 1;
    // Q_f = <J J^T> (its leading block is Q: "low-top submatrix"); right-hand side
    // g_f = <(x - mu) J> with mu = sum_b theta_b Phi_b
    for (int e = threadIdx.x; e < m * m; e += kSolveThreads) {
        const int i = e / m, k = e % m;
        S[i * LD + k] = G[i * LDG + k];
        if (i == k) diag0[i] = G[i * LDG + k];
    }
    for (int a = threadIdx.x; a < m; a += kSolveThreads) {
        double v = G[a * LDG + m];
        for (int b = 0; b < lin; ++b) v = fma(-theta[b], G[a * LDG + b], v);
        S[m * LD + a] = v;
    }
    if (threadIdx.x == 0) {
        S[m * LD + m] = 0.0;
        diag0[m] = 1.0;
    }
    __syncthreads();
    const int rc = chol_with_rhs(S, LD, m, diag0, &status);
    if (threadIdx.x == 0) {
        if (rc == 0) {
            // only the frequency part of the step is needed: the last n unknowns
            for (int j = m - 1; j >= lin; --j) {
                double v = S[m * LD + j];
                for (int i = j + 1; i < m; ++i) v = fma(-S[i * LD + j], step[i], v);
                step[j] = v / S[j * LD + j];
            }
            for (int k = 0; k < n; ++k) df_out[k] = fmin(fmax(step[lin + k], -max_step), max_step);
        } else {
            for (int k = 0; k < n; ++k) df_out[k] = 0.0;
        }
        out2[0] = 0.0;
        out2[1] = (double)rc;
    }
}

__global__ void axpy_small_kernel(double* freqs, const double* df, int n)
{
    const int k = threadIdx.x;
    if (k < n) freqs[k] += df[k];
}

}  // namespace

cudaError_t launch_model_rows(const double* t, int64_t N, double t0, const double* freqs, int n, const double* theta,
                              double* rows, cudaStream_t stream)
{
    model_rows_kernel<<<(unsigned)((N + kRowsThreads - 1) / kRowsThreads), kRowsThreads, 0, stream>>>(t, N, t0, freqs, n,
                                                                                                    theta, rows);
    return cudaGetLastError();
}

cudaError_t launch_chol_solve(const double* A, int m, double* theta, double* out2, cudaStream_t stream)
{
    if (m < 1 || m > kMaxUnknowns) return cudaErrorInvalidValue;
    chol_solve_kernel<<<1, kSolveThreads, 0, stream>>>(A, m, theta, out2);
    return cudaGetLastError();
}

cudaError_t launch_gn_step(const double* G, int n, const double* theta, double max_step, double* df_out, double* out2,
                           cudaStream_t stream)
{
    if (n < 1 || 3 * n + 1 > kMaxUnknowns) return cudaErrorInvalidValue;
    gn_step_kernel<<<1, kSolveThreads, 0, stream>>>(G, n, theta, max_step, df_out, out2);
    return cudaGetLastError();
}

cudaError_t launch_axpy_small(double* freqs, const double* df, int n, cudaStream_t stream)
{
    axpy_small_kernel<<<1, 32, 0, stream>>>(freqs, df, n);
    return cudaGetLastError();
}

}  // namespace fredec
