// peak_kernel.cu -- FP64 roofline probes (measurement tooling behind include/fredec_bench.h; not
// part of the method).  Register-resident loops on all SMs:
//   DFMA only          the FP64 FMA peak of the chip (roofline denominator)
//   DMMA only          the same FP64 units driven by mma.sync.m8n8k4.f64 (the scan kernel's path)
//   DMMA + DFMA mixes  what one scalar FP64 instruction costs next to a saturated DMMA stream, from
//                      the same warp (singly or in bursts) or from a third warp of the sub-partition
// Nothing touches memory until a final, practically never taken store.
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

#define PROBE_DMMA(c, a, b)                                                                      \
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" \
                 : "+d"((c)[0]), "+d"((c)[1])                                                    \
                 : "d"(a), "d"(b))
#define PROBE_DFMA(d, a, b) asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(d) : "d"(a), "d"(b))
#define PROBE_IMAD(d, a, b) asm volatile("mad.lo.s32 %0, %1, %2, %0;" : "+r"(d) : "r"(a), "r"(b))

constexpr int kProbeMmaWarps = 8;    // two per SM sub-partition, as in the scan kernel
constexpr int kProbeTiles = 32;      // accumulator tiles per warp (128 registers)
constexpr int kProbeStep = 256;      // DMMAs per warp between two visits of the third warp (mode "third warp")

// Every MMA warp runs `iters` x 64 DMMAs over 32 independent accumulator tiles.  After every EVERY
// DMMAs it issues BURST scalar instructions: FP64 FMAs on independent registers (KIND 0), on one
// dependent chain (KIND 1), or 32-bit integer multiply-adds (KIND 2).  With EXTRA > 0 the CTA has four
// more warps (one per sub-partition) that issue EXTRA independent DFMAs per kProbeStep DMMAs of the
// MMA warps, paced by a named barrier with the two MMA warps of their sub-partition.
template <int EVERY, int BURST, int KIND, int EXTRA, bool PACED>
__global__ void __launch_bounds__(384, 1) dmma_probe_kernel(int64_t iters, double a0, double b0, double* sink)
{
    const int w = threadIdx.x >> 5;
    double f[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) f[i] = a0 + i;
    int ii[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) ii[i] = threadIdx.x + i;
    const double a = a0 + threadIdx.x, b = b0 * threadIdx.x;
    double s = 0.0;
    if (w < kProbeMmaWarps) {
        double acc[kProbeTiles][2];
#pragma unroll
        for (int i = 0; i < kProbeTiles; ++i) {
            acc[i][0] = threadIdx.x;
            acc[i][1] = i;
        }
        for (int64_t it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < 64; ++i) {
                PROBE_DMMA(acc[i % kProbeTiles], a, b);
                if (EVERY > 0 && (i % EVERY) == EVERY - 1) {
#pragma unroll
                    for (int j = 0; j < BURST; ++j) {
                        if (KIND == 0) PROBE_DFMA(f[j % 8], a, b);
                        if (KIND == 1) PROBE_DFMA(f[0], a, b);
                        if (KIND == 2) PROBE_IMAD(ii[j % 8], ii[(j + 1) % 8], ii[(j + 2) % 8]);
                    }
                }
            }
            if (PACED && (it % (kProbeStep / 64)) == kProbeStep / 64 - 1)
                asm volatile("bar.sync %0, 96;" ::"r"(1 + (w & 3)) : "memory");
        }
#pragma unroll
        for (int i = 0; i < kProbeTiles; ++i) s += acc[i][0] + acc[i][1];
    } else if (PACED) {
        for (int64_t it = 0; it < iters / (kProbeStep / 64); ++it) {
#pragma unroll
            for (int j = 0; j < EXTRA; ++j) PROBE_DFMA(f[j % 8], a, b);
            asm volatile("bar.sync %0, 96;" ::"r"(1 + (w & 3)) : "memory");
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) s += f[i] + (double)ii[i];
    if (s == 1.2345) sink[0] = s;
}

struct Probe {
    const char* name;
    void (*kernel)(int64_t, double, double, double*);
    int threads;
    int scalar_per_64;  // scalar instructions per 64 DMMAs of an MMA warp (same-warp modes)
};

#define PROBE(name, every, burst, kind, extra, paced, threads, per64) \
    Probe{name, dmma_probe_kernel<every, burst, kind, extra, paced>, threads, per64}

const Probe kProbes[] = {
    PROBE("dmma only, 8 warps", 0, 0, 0, 0, false, 256, 0),
    PROBE("dmma + 1 independent dfma per 4 dmma, same warp", 4, 1, 0, 0, false, 256, 16),
    PROBE("dmma + 2 independent dfma per 8 dmma, same warp", 8, 2, 0, 0, false, 256, 16),
    PROBE("dmma + 4 independent dfma per 16 dmma, same warp", 16, 4, 0, 0, false, 256, 16),
    PROBE("dmma + 8 independent dfma per 32 dmma, same warp", 32, 8, 0, 0, false, 256, 16),
    PROBE("dmma + 16 independent dfma per 64 dmma, same warp", 64, 16, 0, 0, false, 256, 16),
    PROBE("dmma + 1 dependent dfma per 4 dmma, same warp", 4, 1, 1, 0, false, 256, 16),
    PROBE("dmma + 8 dependent dfma per 32 dmma, same warp", 32, 8, 1, 0, false, 256, 16),
    PROBE("dmma + 1 dfma per 8 dmma, same warp", 8, 1, 0, 0, false, 256, 8),
    PROBE("dmma + 1 dfma per 16 dmma, same warp", 16, 1, 0, 0, false, 256, 4),
    PROBE("dmma + 1 imad per 1 dmma, same warp", 1, 1, 2, 0, false, 256, 64),
    PROBE("dmma + third warp paced by a barrier every 256 dmma, 0 dfma", 0, 0, 0, 0, true, 384, 0),
    PROBE("dmma + third warp: 32 dfma per 256 dmma", 0, 0, 0, 32, true, 384, 0),
    PROBE("dmma + third warp: 64 dfma per 256 dmma", 0, 0, 0, 64, true, 384, 0),
    PROBE("dmma + third warp: 128 dfma per 256 dmma", 0, 0, 0, 128, true, 384, 0),
};
constexpr int kNumProbes = (int)(sizeof(kProbes) / sizeof(kProbes[0]));

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

int dmma_probe_count() { return kNumProbes; }

const char* dmma_probe_name(int mode) { return mode >= 0 && mode < kNumProbes ? kProbes[mode].name : nullptr; }

cudaError_t launch_dmma_probe(int mode, int64_t iters, int blocks, double* sink, cudaStream_t stream)
{
    if (mode < 0 || mode >= kNumProbes) return cudaErrorInvalidValue;
    kProbes[mode].kernel<<<blocks, kProbes[mode].threads, 0, stream>>>(iters, 1.0, 0.5, sink);
    return cudaGetLastError();
}

double dmma_probe_flops(int64_t iters, int blocks)
{
    return (double)blocks * kProbeMmaWarps * (double)iters * 64.0 * 512.0;  // 8x8x4 FMAs = 512 flops
}

}  // namespace fredec
