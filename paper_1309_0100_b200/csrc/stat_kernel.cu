// stat_kernel.cu -- element-wise statistics on the periodogram (HBM-bound: 8 B read + 8 B written
// per grid point) and the small kernels of the phase-1 driver.  See stat_kernel.cuh.
#include "stat_kernel.cuh"

namespace fredec {

namespace {

constexpr int kStatThreads = 256;

__device__ __forceinline__ double zstat_of(double dchi2, double chi2_base, double NH)
{
    // (N_H/2) ln(l_base / l_alt) with l_alt = l_base - dchi2  (reading G1); dchi2 <= l_base
    double r = chi2_base > 0.0 ? dchi2 / chi2_base : 0.0;
    r = fmin(fmax(r, 0.0), 1.0);
    return -0.5 * NH * log1p(-r);  // +inf for a perfect fit (r = 1)
}

__device__ __forceinline__ double fap1_of(double z, double W, double A1)
{
    if (!(z > 0.0)) return 1.0;
    return fmin(1.0, A1 * W * exp(-z) * sqrt(z));
}

__global__ void __launch_bounds__(kStatThreads) zstat_kernel(const double* __restrict__ dchi2, int64_t K,
                                                            double chi2_base, double NH, double* __restrict__ z)
{
    for (int64_t k = (int64_t)blockIdx.x * kStatThreads + threadIdx.x; k < K; k += (int64_t)gridDim.x * kStatThreads)
        z[k] = zstat_of(dchi2[k], chi2_base, NH);
}

__global__ void __launch_bounds__(kStatThreads) fap1_kernel(const double* __restrict__ z, int64_t K, double W, double A1,
                                                           double* __restrict__ fap)
{
    for (int64_t k = (int64_t)blockIdx.x * kStatThreads + threadIdx.x; k < K; k += (int64_t)gridDim.x * kStatThreads)
        fap[k] = fap1_of(z[k], W, A1);
}

// fixed-order block sum (one CTA of kStatThreads threads), result broadcast
__device__ double cta_sum(double v, double* red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) red[wid] = v;
    __syncthreads();
    double r = (lane < (kStatThreads >> 5)) ? red[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
    return r;
}

__global__ void __launch_bounds__(kStatThreads) bandwidth_kernel(const double* __restrict__ t,
                                                                const double* __restrict__ w, int64_t N, double* out4)
{
    __shared__ double red[32];
    double sw = 0.0, swt = 0.0, bad = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += kStatThreads) {
        const double ti = t[i], wi = w[i];
        if (!isfinite(ti) || !isfinite(wi) || wi < 0.0) bad = 1.0;
        sw += wi;
        swt = fma(wi, ti, swt);
    }
    bad = cta_sum(bad, red);
    const double W = cta_sum(sw, red);
    const double mean = cta_sum(swt, red) / W;
    double sv = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += kStatThreads) {
        const double dt = t[i] - mean;
        sv = fma(w[i] * dt, dt, sv);
    }
    const double var = cta_sum(sv, red) / W;  // weighted variance of t_i
    if (threadIdx.x == 0) {
        const bool ok = bad == 0.0 && W > 0.0 && isfinite(W);
        out4[0] = ok ? sqrt(4.0 * 3.14159265358979323846 * var) : 0.0;
        out4[1] = ok ? var : 0.0;
        out4[2] = ok ? mean : 0.0;
        out4[3] = ok ? 0.0 : -2.0;  // FREDEC_EDATA
    }
}

__global__ void __launch_bounds__(kStatThreads) sin_base_kernel(const double* __restrict__ t, int64_t N,
                                                               const double* __restrict__ freqs, int m,
                                                               double* __restrict__ base)
{
    const int64_t i = (int64_t)blockIdx.x * kStatThreads + threadIdx.x;
    if (i >= N) return;
    const double ti = t[i];
    base[i] = 1.0;
    for (int j = 0; j < m; ++j) {
        double s, c;
        sincospi(2.0 * frac_prod(freqs[j], ti), &s, &c);
        base[(int64_t)(2 * j + 1) * N + i] = c;
        base[(int64_t)(2 * j + 2) * N + i] = s;
    }
}

__global__ void peak_stats_kernel(const double* __restrict__ dchi2, const int64_t* __restrict__ idx, int k,
                                  const SeriesInfo* __restrict__ info, double NH, double W, double A1,
                                  double* __restrict__ out)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= k) return;
    const double chi2_base = info->status == 0 ? info->chi2_base : 0.0;
    const int64_t i = idx[j];
    const double z = i >= 0 ? zstat_of(dchi2[i], chi2_base, NH) : 0.0;
    out[2 * j] = z;
    out[2 * j + 1] = i >= 0 ? fap1_of(z, W, A1) : 1.0;
}

// *flag = 1 if any of v[0..n) is not finite (the caller zeroes the flag first)
__global__ void __launch_bounds__(kStatThreads) finite_flag_kernel(const double* __restrict__ v, int64_t n, int* flag)
{
    bool bad = false;
    for (int64_t k = (int64_t)blockIdx.x * kStatThreads + threadIdx.x; k < n; k += (int64_t)gridDim.x * kStatThreads)
        bad |= !isfinite(v[k]);
    if (bad) *flag = 1;
}

unsigned stat_grid(int64_t K)
{
    int64_t b = (K + kStatThreads - 1) / kStatThreads;
    const int64_t cap = 148 * 16;  // a few waves of a grid-stride loop
    return (unsigned)(b < cap ? (b > 0 ? b : 1) : cap);
}

}  // namespace

cudaError_t launch_zstat(const double* dchi2, int64_t K, double chi2_base, double NH, double* z_out, cudaStream_t stream)
{
    zstat_kernel<<<stat_grid(K), kStatThreads, 0, stream>>>(dchi2, K, chi2_base, NH, z_out);
    return cudaGetLastError();
}

cudaError_t launch_fap1(const double* z, int64_t K, double W, double A1, double* fap_out, cudaStream_t stream)
{
    fap1_kernel<<<stat_grid(K), kStatThreads, 0, stream>>>(z, K, W, A1, fap_out);
    return cudaGetLastError();
}

cudaError_t launch_finite_flag(const double* v, int64_t n, int* flag, cudaStream_t stream)
{
    cudaError_t e = cudaMemsetAsync(flag, 0, sizeof(int), stream);
    if (e != cudaSuccess) return e;
    finite_flag_kernel<<<stat_grid(n), kStatThreads, 0, stream>>>(v, n, flag);
    return cudaGetLastError();
}

cudaError_t launch_bandwidth(const double* t, const double* w, int64_t N, double* out4, cudaStream_t stream)
{
    bandwidth_kernel<<<1, kStatThreads, 0, stream>>>(t, w, N, out4);
    return cudaGetLastError();
}

cudaError_t launch_sin_base(const double* t, int64_t N, const double* freqs, int m, double* base_out,
                            cudaStream_t stream)
{
    sin_base_kernel<<<(unsigned)((N + kStatThreads - 1) / kStatThreads), kStatThreads, 0, stream>>>(t, N, freqs, m,
                                                                                                  base_out);
    return cudaGetLastError();
}

cudaError_t launch_peak_stats(const double* dchi2, const int64_t* idx, int k, const SeriesInfo* info, double NH,
                              double W, double A1, double* out2k, cudaStream_t stream)
{
    peak_stats_kernel<<<(k + 127) / 128, 128, 0, stream>>>(dchi2, idx, k, info, NH, W, A1, out2k);
    return cudaGetLastError();
}

}  // namespace fredec
