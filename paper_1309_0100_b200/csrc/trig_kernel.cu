// trig_kernel.cu -- see trig_kernel.cuh.  Bound: FP64 ALU (one exact sincos, ~45 FP64 instructions,
// plus 14 multiply-adds per (frequency, observation) pair); the lists are short (pool sizes <= N/10
// and their pairwise sums and differences), so this is a latency-sized kernel.
#include "trig_kernel.cuh"

namespace fredec {

namespace {

constexpr int kTrigThreads = 256;

__global__ void __launch_bounds__(kTrigThreads) trig_averages_kernel(const double* __restrict__ t,
                                                                    const double* __restrict__ x,
                                                                    const double* __restrict__ w, int64_t N,
                                                                    const double* __restrict__ freqs,
                                                                    double* __restrict__ out)
{
    __shared__ double red[kTrigThreads / 32][kTrigCols];
    const double f = freqs[blockIdx.x];
    double a[kTrigCols];
#pragma unroll
    for (int q = 0; q < kTrigCols; ++q) a[q] = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += kTrigThreads) {
        const double ti = t[i], wi = w[i], xi = x[i];
        double s, c;
        sincospi(2.0 * frac_prod(f, ti), &s, &c);
        const double wc = wi * c, ws = wi * s, wt = wi * ti;
        const double wtc = wt * c, wts = wt * s;
        a[0] += wc;
        a[1] += ws;
        a[2] += wtc;
        a[3] += wts;
        a[4] = fma(xi, wc, a[4]);
        a[5] = fma(xi, ws, a[5]);
        a[6] = fma(xi, wtc, a[6]);
        a[7] = fma(xi, wts, a[7]);
        a[8] = fma(ti, wtc, a[8]);
        a[9] = fma(ti, wts, a[9]);
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < kTrigCols; ++q) {
        double v = a[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[wid][q] = v;
    }
    __syncthreads();
    if (threadIdx.x < kTrigCols) {
        double v = 0.0;
#pragma unroll
        for (int k = 0; k < kTrigThreads / 32; ++k) v += red[k][threadIdx.x];  // fixed order
        out[(int64_t)blockIdx.x * kTrigCols + threadIdx.x] = v;
    }
}

}  // namespace

cudaError_t launch_trig_averages(const double* t, const double* x, const double* w, int64_t N, const double* freqs,
                                 int64_t M, double* out, cudaStream_t stream)
{
    trig_averages_kernel<<<(unsigned)M, kTrigThreads, 0, stream>>>(t, x, w, N, freqs, out);
    return cudaGetLastError();
}

}  // namespace fredec
