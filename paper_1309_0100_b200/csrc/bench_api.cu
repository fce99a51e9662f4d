// bench_api.cu -- libfredec_bench.so: the FP64 roofline probes of include/fredec_bench.h.  Measurement
// tooling, built apart from the product library (libfredec_b200.so exports include/fredec.h and nothing
// else) and loaded by bench.py only.  Shares no state with the product: its own events, its own 64-byte sink.
#include <cstdint>
#include <cuda_runtime.h>
#include "fredec.h"  // status codes
#include "fredec_bench.h"
#include "peak_kernel.cuh"

namespace {

struct BenchState {
    bool ready = false;
    int sm_count = 0;
    double* sink = nullptr;
    cudaEvent_t ev[2] = {};
};
BenchState b;

#define BCK(expr)                         \
    do {                                  \
        if ((expr) != cudaSuccess) {      \
            (void)cudaGetLastError();     \
            return FREDEC_ECUDA;          \
        }                                 \
    } while (0)

int ensure_ready()
{
    if (b.ready) return FREDEC_OK;
    int n = 0, dev = 0;
    BCK(cudaGetDeviceCount(&n));
    if (n < 1) return FREDEC_ECUDA;
    BCK(cudaGetDevice(&dev));
    BCK(cudaDeviceGetAttribute(&b.sm_count, cudaDevAttrMultiProcessorCount, dev));
    BCK(cudaMalloc(&b.sink, 64));
    BCK(cudaEventCreate(&b.ev[0]));
    BCK(cudaEventCreate(&b.ev[1]));
    b.ready = true;
    return FREDEC_OK;
}

}  // namespace

extern "C" {

int fredec_bench_fp64(int32_t mode, int64_t iters, double* tflops_out, double* ms_out)
{
    using namespace fredec;
    if (!tflops_out || mode < 0 || mode > dmma_probe_count()) return FREDEC_EINVAL;
    if (mode == 0 ? iters < 1024 : (iters < 64 || iters % 4 != 0)) return FREDEC_EINVAL;
    const int rc = ensure_ready();
    if (rc) return rc;
    cudaStream_t st = nullptr;  // the default stream
    double flops;
    if (mode == 0) {
        const int blocks = b.sm_count * 8;  // 2048 threads per SM
        BCK(launch_dfma(1024, blocks, b.sink, st));  // warm-up
        BCK(cudaEventRecord(b.ev[0], st));
        BCK(launch_dfma(iters, blocks, b.sink, st));
        flops = dfma_flops(iters, blocks);
    } else {
        BCK(launch_dmma_probe(mode - 1, 64, b.sm_count, b.sink, st));
        BCK(cudaEventRecord(b.ev[0], st));
        BCK(launch_dmma_probe(mode - 1, iters, b.sm_count, b.sink, st));
        flops = dmma_probe_flops(iters, b.sm_count);
    }
    BCK(cudaEventRecord(b.ev[1], st));
    BCK(cudaStreamSynchronize(st));
    float ms = 0.f;
    BCK(cudaEventElapsedTime(&ms, b.ev[0], b.ev[1]));
    *tflops_out = ms > 0.f ? flops / ((double)ms * 1e-3) * 1e-12 : 0.0;
    if (ms_out) *ms_out = (double)ms;
    return FREDEC_OK;
}

const char* fredec_bench_fp64_name(int32_t mode)
{
    if (mode == 0) return "dfma only, 2048 threads per SM";
    return fredec::dmma_probe_name(mode - 1);
}

}  // extern "C"
