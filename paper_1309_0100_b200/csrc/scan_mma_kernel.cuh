// scan_mma_kernel.cuh -- launch interface of the frequency-scan kernel (steps a4-a10).
#pragma once
#include "common.cuh"

namespace fredec {

// Layout constants shared by the table kernel (writer) and the scan kernel (reader).
//
// The grid is cut into RUNS of R = 2H consecutive frequencies, symmetric about the run's
// centre frequency f_c (half a grid step between two grid points); eight runs make a UNIT
// (one 8-row MMA tile).  For an observation i the phase at grid point f_c +- (h - 1/2) df is
// phi_i +- alpha_hi with phi_i = 2 pi f_c t'_i (depends on the run: a "seed") and
// alpha_hi = 2 pi (h - 1/2) df t'_i (the same for every run: a per-observation TABLE).
//
// Table, per group of 4 observations: [family][column tile pair][32 lanes in B-fragment order][2 tiles],
// families: 0 = y (w x~), 1..NB = p_j (w psi_j), NB+1 = w/2.  Column n = 2 hh + type of tile
// nt belongs to h = 4 nt + hh + 1; type 0 = cos, 1 = sin of alpha_h (of 2 alpha_h in the
// w family); the entry is multiplier x trig value.  Fragment order: element (k = observation
// within the group, n = column) belongs to lane n * 4 + k, the lane that owns it in mma.m8n8k4's
// B operand; the lane's entries of tiles 2p and 2p+1 are adjacent (one LDS.128).  H % 8 == 0.
__host__ __device__ constexpr int mma_nt(int H) { return H / 4; }
__host__ __device__ constexpr int mma_nf(int NB) { return NB + 2; }
__host__ __device__ constexpr int mma_group_doubles(int H, int NB) { return mma_nf(NB) * mma_nt(H) * 32; }

// Per-observation seed record: t', (cos, sin) of the rotation by one unit (8 runs = 8R grid
// steps), 2 cos of it (coefficient of the two-term recurrence along the units), and (cos, sin)
// of the rotation by four runs (4R grid steps).
struct __align__(16) SeedRec {
    double t, cu, su, tcu, c4, s4;
};

struct MmaScanParams {
    const double* tab;       // [B][n_pass][G4][NF][NT][32]
    const SeedRec* srec;     // [B][G4 * 4]
    const SeriesInfo* info;  // [B]
    double* z;               // [B][K] out
    double* ws;              // [B][7][Kpad] partial sums between passes (nullptr if n_pass == 1)
    double* red;             // [grid][MMA warps][mma_red_doubles] scratch of the observation-split reduction
    double* part;            // shared mode: [2 grid][MMA warps][mma_part_doubles] partial sums of the segments
    int64_t N, K, Kpad;
    int64_t G4;  // groups of 4 observations per series = ceil(N / 4)
    int64_t U;   // units per series = ceil(K / (8 R))
    int64_t T;   // total units = B * U
    double f0, df;
    int n_pass, pass;
    int TI;    // observations per shared-memory slot (multiple of 4)
    int NS;    // slots of the (table tile, seeds) ring in shared memory
    int grid;  // CTAs (persistent; each owns a contiguous range of units)
    // shared mode (one series, one pass; see Cursor in scan_mma_kernel.cu): F full rounds per CTA, then
    // Rt left-over rounds cut across the observations and finished by the tail-solve kernel
    int shared, F, Rt;
    // Fused peak extraction (a11 in the epilogue; z == nullptr, one pass): every MMA warp keeps a sorted
    // top-k list per (series, CTA) pair -- list group = series + CTA, a bijection for contiguous ranges;
    // the left-over rounds of the shared mode use the groups tail_group0 + round -- and every unit writes
    // an edge record (its first and last grid point cannot be tested inside the unit).
    // topk_fused_merge_kernel (topk_kernel.cu) merges the lists and settles the unit boundaries.
    int fused_k;         // 0: off (z is written); else k <= kFusedMaxK
    int tail_group0;
    double* list_z;      // [groups][MMA warps][fused_k]
    int64_t* list_i;     // same shape; < 0: empty entry (filled with 0xFF bytes before the launch)
    double* edges;       // [B][U][4]: z_first, first_ok, z_last, last_ok (flags 1.0 / 0.0)
    // [groups]: bit pattern of the largest k-th entry among the group's full lists (0: none yet; z >= 0, so
    // the patterns order like the values).  A value below it cannot be among the series' k highest peaks.
    unsigned long long* group_thr;
};
constexpr int kFusedMaxK = 32;  // one list entry per lane

struct MmaScanConfig {
    int H, NOCT, NW;  // half run length, units per MMA warp and round, MMA warps per CTA
};

// The (H, NOCT) the library is built with for NB base functions per pass (NB <= kMmaMaxNB).
constexpr int kMmaMaxNB = 9;
MmaScanConfig mma_scan_config(int NB);
size_t mma_scan_slot_bytes(int NB, int TI);
size_t mma_red_doubles(int NB);  // per MMA warp: the accumulators of one unit
size_t mma_part_doubles(int NB); // per MMA warp: all its accumulators  // one ring slot; the kernel needs NS of them
constexpr int kMmaMaxSlots = 8;
cudaError_t launch_mma_scan(int NB, const MmaScanParams& p, cudaStream_t stream);

}  // namespace fredec
