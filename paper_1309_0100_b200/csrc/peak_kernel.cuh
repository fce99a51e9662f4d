// peak_kernel.cuh -- FP64 roofline probes (include/fredec_bench.h); measurement tooling, not the method.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace fredec {
cudaError_t launch_dfma(int64_t iters, int blocks, double* sink, cudaStream_t stream);
double dfma_flops(int64_t iters, int blocks);  // flops one launch executes (FMA = 2)

int dmma_probe_count();
const char* dmma_probe_name(int mode);  // nullptr outside [0, dmma_probe_count())
// `iters` blocks of 64 DMMAs per MMA warp, `blocks` CTAs of 8 MMA warps (+ 4 more in the third-warp modes)
cudaError_t launch_dmma_probe(int mode, int64_t iters, int blocks, double* sink, cudaStream_t stream);
double dmma_probe_flops(int64_t iters, int blocks);  // DMMA flops of one launch
}  // namespace fredec
