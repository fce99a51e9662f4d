/*
 * fredec_bench.h -- measurement tooling, exported by libfredec_bench.so (built beside the product library
 * libfredec_b200.so, which exports fredec.h and nothing else; only bench.py loads it).  Nothing here is part
 * of the method (arXiv:1309.0100); these calls exist so that bench.py
 * can state the FP64 roofline denominator of the box it runs on (MEASURED_PEAKS.json has no FP64
 * figure) and what a scalar FP64 instruction costs next to the scan kernel's FP64 MMA stream.
 * Status codes as in fredec.h; the probes run on the default stream and return when they have completed.
 */
#ifndef FREDEC_BENCH_H
#define FREDEC_BENCH_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/*
 * fredec_bench_fp64 -- runs one register-resident FP64 probe on all SMs and times it with CUDA events
 * on the default stream (one warm-up launch first).
 *   mode 0     DFMA only, 2048 threads per SM, 8 independent chains per thread: the FP64 FMA peak.
 *              iters = FMAs per chain (>= 1024); tflops_out counts 2 flops per FMA.
 *   mode >= 1  a DMMA (mma.sync.m8n8k4.f64) loop, one CTA of 8 MMA warps per SM, optionally mixed with
 *              scalar instructions; fredec_bench_fp64_name(mode) describes it.  iters = blocks of 64
 *              DMMAs per warp (>= 64, a multiple of 4); tflops_out counts the DMMA flops only (512 per
 *              warp instruction), so the drop against the DMMA-only mode is the cost of the mix.
 * Returns FREDEC_OK, FREDEC_EINVAL (unknown mode, iters out of range, NULL tflops_out) or FREDEC_ECUDA.
 */
int fredec_bench_fp64(int32_t mode, int64_t iters, double* tflops_out, double* ms_out);

/* Description of a probe mode; NULL for mode < 0 or past the last one. */
const char* fredec_bench_fp64_name(int32_t mode);

#ifdef __cplusplus
}
#endif
#endif /* FREDEC_BENCH_H */
