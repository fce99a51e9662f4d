// common.cuh -- shared device-side definitions of the B200 periodogram scan.
// (Product code.  Shares nothing with oracle/.)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace fredec {

// Per-series scalars produced by the prep kernel.
struct SeriesInfo {
    double W;          // <1> = sum w
    double chi2_base;  // min chi2 of the base model alone
    double t_mid;      // time origin used for centring
    int status;        // FREDEC_OK / FREDEC_EDATA / FREDEC_ESINGULAR
    int pad;
};

// Relative pivot thresholds (S6): a trial column is dropped when its Schur pivot
// is <= kTauTrial x its un-projected diagonal; the base is singular when a Gram-Schmidt
// residual norm^2 is <= kTauBase x the function's own norm^2.
constexpr double kTauTrial = 1e-10;
constexpr double kTauBase = 1e-12;

// frac(a*b) in turns, |result| <= 1/2 (+ rounding), exact up to the final addition:
// a*b = hi + lo exactly (FMA), hi - rint(hi) is exact.
__device__ __forceinline__ double frac_prod(double a, double b)
{
    double hi = a * b;
    double lo = fma(a, b, -hi);
    return (hi - rint(hi)) + lo;
}

// ---------------------------------------------------------------------------------------
// mbarrier + bulk-copy (TMA, 1-D) helpers: inline PTX for sm_100a.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, 0x989680;\n\t"
        "@p bra WAIT_DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "WAIT_DONE:\n\t"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// global -> shared bulk copy; bytes % 16 == 0, both addresses 16-byte aligned.
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

}  // namespace fredec
