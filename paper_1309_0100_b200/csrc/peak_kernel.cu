// peak_kernel.cu -- FP64 FMA peak microbenchmark (roofline denominator; not part of the method).
// Each thread runs 8 independent register-resident DFMA chains; nothing touches memory until
// the final (never-taken in practice) store that keeps the compiler honest.
#include "peak_kernel.cuh"

namespace fredec {

namespace {

constexpr int kChains = 8;

__global__ void __launch_bounds__(256) dfma_kernel(int64_t iters, double a, double b, double* sink)
{
    double v[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) v[c] = (double)(threadIdx.x + c) * 1e-3;
    for (int64_t it = 0; it < iters; it += 8) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) v[c] = fma(v[c], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += v[c];
    if (s == 123.456) sink[0] = s;  // practically never true; defeats dead-code elimination
}

}  // namespace

cudaError_t launch_dfma(int64_t iters, int blocks, double* sink, cudaStream_t stream)
{
    dfma_kernel<<<blocks, 256, 0, stream>>>(iters, 0.999999, 1e-7, sink);
    return cudaGetLastError();
}

double dfma_flops(int64_t iters, int blocks)
{
    const int64_t it8 = (iters + 7) / 8 * 8;
    return 2.0 * (double)it8 * kChains * 256.0 * (double)blocks;
}

}  // namespace fredec
