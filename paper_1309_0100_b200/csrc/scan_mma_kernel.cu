// scan_mma_kernel.cu -- steps a4-a10: the periodogram scan kernel for sm_100a.
//
// For every grid frequency f_k the kernel forms the weighted trigonometric sums of
// PAPER.md:165-171 (eqs. 15, 16) against the orthonormalised base (prep kernel):
//
//   YC = <x~ cos>, YS = <x~ sin>, CC = <cos^2>, CS = <cos sin>, (SS = <1> - CC)
//   A_j = <psi_j cos>, B_j = <psi_j sin>,  j < NB
//
// and solves the 2x2 Schur complement (the last two steps of the Cholesky forward
// substitution of PAPER.md:175/183) in the epilogue: z = a_d^2 + a_{d+1}^2.
//
// How the sums are formed.  The grid is cut into runs of R = 2H consecutive frequencies,
// symmetric about the run centre f_c.  With phi_i = 2 pi f_c t'_i and
// alpha_hi = 2 pi (h - 1/2) df t'_i  (h = 1..H), the two grid points at distance h - 1/2 from
// the centre have
//
//   sum_i m_i cos(phi_i +- alpha_hi) = sum_i (cos phi_i)(m_i cos alpha_hi) -+ sum_i (sin phi_i)(m_i sin alpha_hi)
//   sum_i m_i sin(phi_i +- alpha_hi) = sum_i (sin phi_i)(m_i cos alpha_hi) +- sum_i (cos phi_i)(m_i sin alpha_hi)
//
// for any per-observation multiplier m (y, p_j; w/2 with doubled angles for CC, CS).  The
// right-hand sides are a dense contraction over the observations: a matrix of SEEDS
// (rows = runs x {cos phi, sin phi}, columns = observations) times the per-observation TABLE
// (rows = observations, columns = families x h x {cos, sin}) that the table kernel writes once
// per scan.  It runs on the FP64 MMA path (mma.sync.m8n8k4.f64 = DMMA.8x8x4, the same FP64
// units as DFMA at full rate and without the register-bandwidth limit of three-operand DFMAs),
// one FMA per (frequency, observation, sum), and there is no per-pair recurrence or sincos:
// the only other per-pair work is the seed, one complex rotation per (run, observation).
//
// Work decomposition.  8 runs = one UNIT (an 8-row MMA tile, 8R frequencies).  The CTA is
// persistent and owns a contiguous range of units, processed in ROUNDS of up to
// kNW * NOCT units of one series; within a round warp w owns up to NOCT units, whose
// 2 * NF * NT accumulator tiles per unit stay in registers while the round streams over all
// observations tile by tile:
//
//   stage   table tile + seed records, global -> shared by 1-D TMA (cp.async.bulk + mbarrier),
//           three stages
//   phase A seeds e^{i phi} for every (run of the round, observation of the NEXT tile) into
//           shared memory in A-fragment order: one exact evaluation (range-reduced phase,
//           sincospi) at the round's first unit, then one FP64 rotation per further unit
//   phase B per 4 observations: A fragments (seeds; double-angle seeds by 4 flops), B fragments
//           (table), 2 * NF * NT MMAs per unit
//   a9/a10  after the last tile the thread that holds all sums of a frequency solves and stores z.
//
// Every accumulation order is fixed, so results are bitwise reproducible run to run.
#include "scan_mma_kernel.cuh"

namespace fredec {

namespace {

constexpr int kNW = 8;      // warps per CTA (two per SM sub-partition)
constexpr int kStages = 3;  // shared-memory stages of (table tile, seed records)

#define FREDEC_DMMA(c, a, b)                                                                  \
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"       \
        : "+d"((c)[0]), "+d"((c)[1])                                                          \
        : "d"(a), "d"(b))

// Position of a CTA in its sequence of (round, tile) steps.  Three cursors walk the same
// sequence: the loader two steps ahead, the seeder one step ahead, the MMA loop.
struct Cursor {
    int64_t g, g_end;  // next unit after this round / end of the CTA's range (global numbering)
    int64_t b, u;      // series and first unit (within the series) of the current round
    int n;             // units in the current round
    int tile;          // tile within the round
    int step;          // steps taken so far: selects the stage and the seed buffer
    bool valid;

    __device__ __forceinline__ void set_round(int64_t U, int cap)
    {
        b = g / U;
        u = g - b * U;
        int64_t m = U - u;
        if (g_end - g < m) m = g_end - g;
        n = m < cap ? (int)m : cap;
    }
    __device__ __forceinline__ void init(int64_t g0, int64_t g1, int64_t U, int cap)
    {
        g = g0;
        g_end = g1;
        tile = 0;
        step = 0;
        valid = g < g_end;
        b = u = 0;
        n = 0;
        if (valid) set_round(U, cap);
    }
    __device__ __forceinline__ void advance(int ntiles, int64_t U, int cap)
    {
        ++step;
        if (++tile == ntiles) {
            tile = 0;
            g += n;
            valid = g < g_end;
            if (valid) set_round(U, cap);
        }
    }
};

// units of the round owned by warp w: cnt units starting at slot off
__device__ __forceinline__ void warp_share(int n, int w, int& off, int& cnt)
{
    const int q = n / kNW, r = n - q * kNW;
    cnt = q + (w < r ? 1 : 0);
    off = w * q + (w < r ? w : r);
}

template <int H, int NOCT, int NB>
struct Tiles {
    static constexpr int NT = H / 4, NF = NB + 2;
    double v[NOCT][2][NF][NT][2];
    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int o = 0; o < NOCT; ++o)
#pragma unroll
            for (int x = 0; x < 2; ++x)
#pragma unroll
                for (int f = 0; f < NF; ++f)
#pragma unroll
                    for (int t = 0; t < NT; ++t) v[o][x][f][t][0] = v[o][x][f][t][1] = 0.0;
    }
};

// phase B for one tile: CNT = units this warp owns in the round
template <int CNT, int H, int NOCT, int NB>
__device__ __forceinline__ void mma_tile(Tiles<H, NOCT, NB>& acc, const double* tabs, const double2* sb, int ngrp,
                                         int cap)
{
    constexpr int NT = H / 4, NF = NB + 2, GROUP = NF * NT * 32;
#pragma unroll 1
    for (int ks = 0; ks < ngrp; ++ks) {
        double2 a[CNT];
        double c2[CNT], s2[CNT];
#pragma unroll
        for (int o = 0; o < CNT; ++o) {
            a[o] = sb[((size_t)ks * cap + o) * 32];
            c2[o] = fma(a[o].x, a[o].x, -(a[o].y * a[o].y));  // cos 2 phi
            s2[o] = (a[o].x + a[o].x) * a[o].y;              // sin 2 phi
        }
        const double* tk = tabs + (size_t)ks * GROUP;
#pragma unroll
        for (int f = 0; f < NF; ++f) {
#pragma unroll
            for (int t = 0; t < NT; ++t) {
                const double bf = tk[(f * NT + t) * 32];
#pragma unroll
                for (int o = 0; o < CNT; ++o) {
                    if (f < NF - 1) {
                        FREDEC_DMMA(acc.v[o][0][f][t], a[o].x, bf);
                        FREDEC_DMMA(acc.v[o][1][f][t], a[o].y, bf);
                    } else {
                        FREDEC_DMMA(acc.v[o][0][f][t], c2[o], bf);
                        FREDEC_DMMA(acc.v[o][1][f][t], s2[o], bf);
                    }
                }
            }
        }
    }
}

// a9 for one frequency: 2x2 Schur solve with the singular rule S6
__device__ __forceinline__ double solve_z(double YC, double YS, double CC, double CS, double Saa, double Sab,
                                          double Sbb, double W)
{
    const double SS = W - CC;  // <sin^2> = <1> - <cos^2>
    const double Scc = CC - Saa, Scs = CS - Sab, Sss = SS - Sbb;
    double z = 0.0, ys = YS, piv2 = Sss;
    if (Scc > kTauTrial * CC) {  // S6: otherwise the cos column is in the span of the base
        const double q = Scs / Scc;
        z = YC * YC / Scc;
        ys = fma(-q, YC, YS);
        piv2 = fma(-q, Scs, Sss);
    }
    if (piv2 > kTauTrial * SS) z = fma(ys, ys / piv2, z);
    return z;
}

template <int H, int NOCT, int NB>
__global__ void __launch_bounds__(kNW * 32, 1) scan_mma_kernel(MmaScanParams p)
{
    constexpr int R = 2 * H, NT = H / 4, NF = NB + 2, GROUP = NF * NT * 32, CAP = kNW * NOCT;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar[kStages];

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int KS = p.TI / 4;  // groups of 4 observations per tile
    const size_t tab_bytes = (size_t)KS * GROUP * 8;
    const size_t stage_bytes = tab_bytes + (size_t)p.TI * sizeof(SeedRec);
    double2* const seeds = reinterpret_cast<double2*>(smem_raw + kStages * stage_bytes);  // [2][KS][CAP][32]
    const size_t seed_buf = (size_t)KS * CAP * 32;
    const int ntiles = (int)((p.G4 + KS - 1) / KS);
    const int64_t U = p.U;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(&bar[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    const int64_t g0 = (int64_t)blockIdx.x * p.T / p.grid, g1 = (int64_t)(blockIdx.x + 1) * p.T / p.grid;
    Cursor ld, sd, cm;
    ld.init(g0, g1, U, CAP);
    sd = ld;
    cm = ld;
    if (!cm.valid) return;

    auto issue = [&](const Cursor& c) {  // one thread: stage the tile of step c
        const int64_t grp0 = (int64_t)c.tile * KS;
        const int ngrp = (int)min((int64_t)KS, p.G4 - grp0);
        const uint32_t b_tab = (uint32_t)ngrp * GROUP * 8u, b_rec = (uint32_t)ngrp * 4u * (uint32_t)sizeof(SeedRec);
        const int st = c.step % kStages;
        unsigned char* dst = smem_raw + st * stage_bytes;
        mbar_expect_tx(&bar[st], b_tab + b_rec);
        bulk_g2s(dst, p.tab + ((c.b * p.n_pass + p.pass) * p.G4 + grp0) * GROUP, b_tab, &bar[st]);
        bulk_g2s(dst + tab_bytes, p.srec + (c.b * p.G4 + grp0) * 4, b_rec, &bar[st]);
    };
    auto wait_stage = [&](const Cursor& c) {
        mbar_wait(&bar[c.step % kStages], (uint32_t)((c.step / kStages) & 1));
    };
    // phase A: seeds of step c into seed buffer c.step & 1
    auto seed_tile = [&](const Cursor& c) {
        wait_stage(c);
        const SeedRec* recs =
            reinterpret_cast<const SeedRec*>(smem_raw + (c.step % kStages) * stage_bytes + tab_bytes);
        const int ngrp = (int)min((int64_t)KS, p.G4 - (int64_t)c.tile * KS);
        double2* sb = seeds + (c.step & 1) * seed_buf + lane;
        const int m = lane >> 2, k = lane & 3;
        // centre of run m of the round's first unit: f_c = f0 + (run R + H - 1/2) df   (S1)
        const double kc = (double)((c.u * 8 + m) * R + H) - 0.5;
        const double fc = fma(kc, p.df, p.f0);
        for (int ks = wid; ks < ngrp; ks += kNW) {
            const SeedRec r = recs[ks * 4 + k];
            double cs, sn;
            sincospi(2.0 * frac_prod(fc, r.t), &sn, &cs);
            double2* dst = sb + (size_t)ks * CAP * 32;
            for (int slot = 0; slot < c.n; ++slot) {
                dst[slot * 32] = make_double2(cs, sn);
                const double nc = fma(cs, r.cu, -(sn * r.su));
                const double ns = fma(sn, r.cu, cs * r.su);
                cs = nc;
                sn = ns;
            }
        }
    };

    Tiles<H, NOCT, NB> acc;
    acc.clear();

    // phase B (+ epilogue after the last tile) of step c
    auto mma_step = [&](const Cursor& c) {
        int off, cnt;
        warp_share(c.n, wid, off, cnt);
        if (cnt == 0) return;
        wait_stage(c);
        const double* tabs = reinterpret_cast<const double*>(smem_raw + (c.step % kStages) * stage_bytes) + lane;
        const double2* sb = seeds + (c.step & 1) * seed_buf + (size_t)off * 32 + lane;
        const int ngrp = (int)min((int64_t)KS, p.G4 - (int64_t)c.tile * KS);
        if (NOCT == 1 || cnt == 1) {
            mma_tile<1>(acc, tabs, sb, ngrp, CAP);
        } else if (NOCT == 2 || cnt == 2) {
            mma_tile<(NOCT >= 2 ? 2 : 1)>(acc, tabs, sb, ngrp, CAP);
        } else if (NOCT == 3 || cnt == 3) {
            mma_tile<(NOCT >= 3 ? 3 : 1)>(acc, tabs, sb, ngrp, CAP);
        } else {
            mma_tile<NOCT>(acc, tabs, sb, ngrp, CAP);
        }
        if (c.tile + 1 < ntiles) return;

        // ---- a9/a10: this thread holds every sum of 2 * NT frequencies per unit ----------
        const SeriesInfo info = p.info[c.b];
        const int m = lane >> 2, q = lane & 3;
        const bool last_pass = p.pass + 1 == p.n_pass;
#pragma unroll
        for (int o = 0; o < NOCT; ++o) {
            if (o < cnt) {
                const int64_t k0 = ((c.u + off + o) * 8 + m) * R;  // first grid point of the run
#pragma unroll
                for (int t = 0; t < NT; ++t) {
                    const int h = 4 * t + q + 1;
#pragma unroll
                    for (int sg = 0; sg < 2; ++sg) {  // sg = 0: f_c + (h - 1/2) df, 1: f_c - (h - 1/2) df
                        const double sgn = sg == 0 ? 1.0 : -1.0;
                        const int64_t k = sg == 0 ? k0 + H - 1 + h : k0 + H - h;
                        double sums[NF][2];  // (cos sum, sin sum) per family
#pragma unroll
                        for (int f = 0; f < NF; ++f) {
                            sums[f][0] = fma(-sgn, acc.v[o][1][f][t][1], acc.v[o][0][f][t][0]);
                            sums[f][1] = fma(sgn, acc.v[o][0][f][t][1], acc.v[o][1][f][t][0]);
                        }
                        double YC = sums[0][0], YS = sums[0][1];
                        double CC = fma(0.5, info.W, sums[NF - 1][0]), CS = sums[NF - 1][1];
                        double Saa = 0.0, Sab = 0.0, Sbb = 0.0;
#pragma unroll
                        for (int j = 0; j < NB; ++j) {
                            Saa = fma(sums[1 + j][0], sums[1 + j][0], Saa);
                            Sab = fma(sums[1 + j][0], sums[1 + j][1], Sab);
                            Sbb = fma(sums[1 + j][1], sums[1 + j][1], Sbb);
                        }
                        if (k < p.K && info.status == 0) {
                            if (p.n_pass > 1) {  // multi-pass: carry the seven partial sums through global memory
                                double* wsp = p.ws + (c.b * 7) * p.Kpad + k;
                                if (p.pass > 0) {
                                    YC = wsp[0 * p.Kpad];
                                    YS = wsp[1 * p.Kpad];
                                    CC = wsp[2 * p.Kpad];
                                    CS = wsp[3 * p.Kpad];
                                    Saa += wsp[4 * p.Kpad];
                                    Sab += wsp[5 * p.Kpad];
                                    Sbb += wsp[6 * p.Kpad];
                                }
                                if (!last_pass) {
                                    if (p.pass == 0) {
                                        wsp[0 * p.Kpad] = YC;
                                        wsp[1 * p.Kpad] = YS;
                                        wsp[2 * p.Kpad] = CC;
                                        wsp[3 * p.Kpad] = CS;
                                    }
                                    wsp[4 * p.Kpad] = Saa;
                                    wsp[5 * p.Kpad] = Sab;
                                    wsp[6 * p.Kpad] = Sbb;
                                }
                            }
                            if (last_pass) p.z[c.b * p.K + k] = solve_z(YC, YS, CC, CS, Saa, Sab, Sbb, info.W);
                        }
                    }
                }
            }
        }
        acc.clear();
    };

    // ---- prologue: stage steps 0 and 1, seeds of step 0 ---------------------------------
    if (tid == 0) {
        issue(ld);
        ld.advance(ntiles, U, CAP);
        if (ld.valid) issue(ld);
        ld.advance(ntiles, U, CAP);
    } else {
        ld.advance(ntiles, U, CAP);
        ld.advance(ntiles, U, CAP);
    }
    seed_tile(sd);
    sd.advance(ntiles, U, CAP);
    __syncthreads();

    // ---- main loop over steps -----------------------------------------------------------
    while (cm.valid) {
        // stage step+2: its stage was last read in step-1, which every warp has left
        if (tid == 0 && ld.valid) issue(ld);
        ld.advance(ntiles, U, CAP);
        // two warps share a sub-partition's FP64 pipe: one seeds while the other multiplies
        if (wid < kNW / 2) {
            if (sd.valid) seed_tile(sd);
            mma_step(cm);
        } else {
            mma_step(cm);
            if (sd.valid) seed_tile(sd);
        }
        sd.advance(ntiles, U, CAP);
        cm.advance(ntiles, U, CAP);
        __syncthreads();
    }
}

template <int H, int NOCT, int NB>
cudaError_t launch_one(const MmaScanParams& p, cudaStream_t stream)
{
    const size_t smem = mma_scan_smem_bytes(NB, p.TI);
    static size_t attr_smem = 0;
    if (smem > attr_smem) {
        cudaError_t e = cudaFuncSetAttribute(scan_mma_kernel<H, NOCT, NB>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_smem = smem;
    }
    scan_mma_kernel<H, NOCT, NB><<<p.grid, kNW * 32, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace

// (H, NOCT) per NB: NOCT * (2 + NB) * H accumulator doubles per thread
#define FREDEC_MMA_CONFIGS(X) \
    X(8, 2, 0) X(8, 2, 1) X(8, 2, 2) X(8, 2, 3) X(8, 1, 4) X(8, 1, 5) X(8, 1, 6) X(8, 1, 7) X(8, 1, 8) X(8, 1, 9)

MmaScanConfig mma_scan_config(int NB)
{
#define X(h, noct, nb) \
    if (NB == nb) return MmaScanConfig{h, noct, kNW};
    FREDEC_MMA_CONFIGS(X)
#undef X
    return MmaScanConfig{0, 0, 0};
}

size_t mma_scan_smem_bytes(int NB, int TI)
{
    const MmaScanConfig c = mma_scan_config(NB);
    const size_t stage = (size_t)(TI / 4) * mma_group_doubles(c.H, NB) * 8 + (size_t)TI * sizeof(SeedRec);
    const size_t seeds = 2 * (size_t)(TI / 4) * (c.NW * c.NOCT) * 32 * 16;
    return kStages * stage + seeds;
}

cudaError_t launch_mma_scan(int NB, const MmaScanParams& p, cudaStream_t stream)
{
#define X(h, noct, nb) \
    if (NB == nb) return launch_one<h, noct, nb>(p, stream);
    FREDEC_MMA_CONFIGS(X)
#undef X
    return cudaErrorInvalidValue;
}

}  // namespace fredec
