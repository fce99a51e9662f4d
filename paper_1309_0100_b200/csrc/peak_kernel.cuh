// peak_kernel.cuh -- FP64 FMA peak microbenchmark interface.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace fredec {
cudaError_t launch_dfma(int64_t iters, int blocks, double* sink, cudaStream_t stream);
double dfma_flops(int64_t iters, int blocks);  // flops one launch executes (FMA = 2)
}  // namespace fredec
