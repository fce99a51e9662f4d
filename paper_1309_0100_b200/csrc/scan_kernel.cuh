// scan_kernel.cuh -- launch interface of the frequency-scan kernel.
#pragma once
#include "common.cuh"

namespace fredec {

struct ScanParams {
    const double* rec;       // [B][n_pass][N][rec_stride(NB)] packed observation records
    const SeriesInfo* info;  // [B]
    double* z;               // [B][K] out
    double* ws;              // [B][7][Kpad] partial sums between passes (nullptr if n_pass == 1)
    int64_t N, K, Kpad;
    double f0, df;
    int n_pass, pass;
    int FW;  // frequency-warps per CTA: the CTA owns FW*32 runs of R consecutive frequencies
    int S;   // observation split: S warps share a run, each over 1/S of every tile
    int TI;  // observations per shared-memory tile (multiple of S)
};

// Supported (R, NB) instantiations; returns false if (R, NB) is not built.
bool scan_config_supported(int R, int NB);
int scan_max_warps();  // FW * S may not exceed this
size_t scan_smem_bytes(int R, int NB, const ScanParams& p);
cudaError_t launch_scan(int R, int NB, const ScanParams& p, int64_t B, cudaStream_t stream);

}  // namespace fredec
