// prep_kernel.cuh -- launch interface of the orthogonalisation / packing kernel.
#pragma once
#include "common.cuh"
#include "scan_mma_kernel.cuh"

namespace fredec {

struct PrepParams {
    const double* t;     // [B][N]
    const double* x;     // [B][N]
    const double* w;     // [B][N]
    const double* base;  // [B][d][N] or nullptr when d == 0
    double* psi;         // workspace [B][d][N]
    double* xt;          // workspace [B][N]
    SeriesInfo* info;    // out [B]
    int64_t N;
    int d;
};

// a3 (layouts: scan_mma_kernel.cuh): table + seed records from the prep kernel's psi, x~
struct TableParams {
    const double* t;         // [B][N]
    const double* w;         // [B][N]
    const double* psi;       // [B][d][N] orthonormal base (prep kernel)
    const double* xt;        // [B][N] residual x~ (prep kernel)
    const SeriesInfo* info;  // [B]
    double* tab;             // out [B][n_pass][G4][NF][NT][32]
    SeedRec* srec;           // out [B][G4 * 4]
    int64_t N, G4;
    int d, NB, n_pass, H;
    double df;
};

cudaError_t launch_table(const TableParams& p, int64_t B, cudaStream_t stream);

cudaError_t launch_prep(const PrepParams& p, int64_t B, cudaStream_t stream);

// Incremental a2 for one series: appends cos / sin(2 pi f t) to the orthonormal base psi [d0][N] (rows d0 and
// d0 + 1 must be allocated) and updates x~ and chi2_base; see prep_kernel.cu.
struct PrepAppendParams {
    const double* t;     // [N]
    const double* w;     // [N]
    const double* freq;  // device pointer to the new frequency
    double* psi;         // [d0 + 2][N]
    double* xt;          // [N]
    SeriesInfo* info;
    int64_t N;
    int d0;
};
cudaError_t launch_prep_append(const PrepAppendParams& p, cudaStream_t stream);

}  // namespace fredec
