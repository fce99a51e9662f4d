// subset_kernel.cu -- see subset_kernel.cuh.
//
// The paper runs "many entirely independent instances of the fitting subroutine" whose arrays
// live in global memory.  Here the full Fisher matrix Q and gradient g of the pool
// are formed ONCE (every subset's Q is a sub-matrix of it: "low-top submatrix"), kept
// in shared memory, and each warp eliminates one subset's augmented matrix [[Q_S, g_S], [g_S^T, D]]
// in its own shared-memory workspace: after the m elimination steps of the Cholesky / LDL^T
// factorisation the last diagonal entry is the Schur complement D - g_S^T Q_S^{-1} g_S = l_S.
#include "subset_kernel.cuh"

namespace fredec {

namespace {

constexpr int kGramThreads = 256;
constexpr int kSubsetWarps = 8;

__global__ void __launch_bounds__(kGramThreads) gram_kernel(const double* __restrict__ basis,
                                                           const double* __restrict__ x,
                                                           const double* __restrict__ w, int64_t N, int M,
                                                           double* __restrict__ A)
{
    __shared__ double red[kGramThreads / 32];
    const int a = blockIdx.x, b = blockIdx.y;
    if (a > b) return;
    const double* pa = a < M ? basis + (int64_t)a * N : x;
    const double* pb = b < M ? basis + (int64_t)b * N : x;
    double acc = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += kGramThreads) acc = fma(w[i] * pa[i], pb[i], acc);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0;
        for (int k = 0; k < kGramThreads / 32; ++k) v += red[k];  // fixed order
        A[a * (M + 1) + b] = v;
        A[b * (M + 1) + a] = v;
    }
}

__global__ void __launch_bounds__(kSubsetWarps * 32) subset_fit_kernel(const double* __restrict__ A, int n,
                                                                      double* __restrict__ l_out)
{
    extern __shared__ double sm[];
    const int M = 2 * n + 1, LD = M + 1;
    double* Afull = sm;                                                 // [LD][LD]
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double* Wk = sm + LD * LD + wid * (LD * LD + LD);                   // this warp's workspace [m+1][LD]
    int* ids = reinterpret_cast<int*>(Wk + LD * LD);                    // [LD] indices into the full model
    for (int e = threadIdx.x; e < LD * LD; e += blockDim.x) Afull[e] = A[e];
    __syncthreads();

    const int64_t total = (int64_t)1 << n;
    for (int64_t mask = (int64_t)blockIdx.x * kSubsetWarps + wid; mask < total;
         mask += (int64_t)gridDim.x * kSubsetWarps) {
        // model functions of the subset: the constant, then (cos, sin) of each chosen frequency; x last
        int m = 1;
        if (lane == 0) {
            ids[0] = 0;
            for (int j = 0; j < n; ++j)
                if ((mask >> j) & 1) {
                    ids[m++] = 2 * j + 1;
                    ids[m++] = 2 * j + 2;
                }
            ids[m] = M;
        }
        m = 1 + 2 * __popcll((unsigned long long)mask);
        __syncwarp();
        for (int e = lane; e < (m + 1) * (m + 1); e += 32) {
            const int i = e / (m + 1), k = e - i * (m + 1);
            if (k <= i) Wk[i * LD + k] = Afull[ids[i] * LD + ids[k]];
        }
        __syncwarp();
        for (int j = 0; j < m; ++j) {
            const double piv = Wk[j * LD + j];
            // a function that the earlier ones already span is dropped (the rule of DESIGN.md S6)
            if (piv > kTauTrial * Afull[ids[j] * LD + ids[j]]) {
                const double inv = 1.0 / piv;
                for (int i = j + 1; i <= m; ++i) {
                    const double fac = Wk[i * LD + j] * inv;
                    for (int k = j + 1 + lane; k <= i; k += 32) Wk[i * LD + k] = fma(-fac, Wk[k * LD + j], Wk[i * LD + k]);
                }
            }
            __syncwarp();
        }
        if (lane == 0) l_out[mask] = fmax(Wk[m * LD + m], 0.0);
        __syncwarp();
    }
}

}  // namespace

cudaError_t launch_gram(const double* basis, const double* x, const double* w, int64_t N, int M, double* A,
                        cudaStream_t stream)
{
    gram_kernel<<<dim3(M + 1, M + 1), kGramThreads, 0, stream>>>(basis, x, w, N, M, A);
    return cudaGetLastError();
}

cudaError_t launch_subset_fits(const double* A, int n, double* l_out, int sm_count, cudaStream_t stream)
{
    const int LD = 2 * n + 2;
    const size_t smem = ((size_t)LD * LD + (size_t)kSubsetWarps * (LD * LD + LD)) * 8;
    cudaError_t e = cudaFuncSetAttribute(subset_fit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int64_t total = (int64_t)1 << n;
    int64_t grid = (total + kSubsetWarps - 1) / kSubsetWarps;
    if (grid > (int64_t)sm_count * 4) grid = (int64_t)sm_count * 4;
    subset_fit_kernel<<<(unsigned)grid, kSubsetWarps * 32, smem, stream>>>(A, n, l_out);
    return cudaGetLastError();
}

}  // namespace fredec
