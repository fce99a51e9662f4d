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
// kMmaWarps * NOCT units of one series; within a round MMA warp w owns up to NOCT units, whose
// 2 * NF * NT accumulator tiles per unit stay in registers while the round streams over all
// observations, one STEP = one tile of TI observations at a time.
//
// The CTA is warp-specialised (three warpgroups; registers moved between them with
// setmaxnreg) around a ring of NS shared-memory slots, slot = (table tile, seeds) of one step:
//
//   seed warps (4, one per SM sub-partition)  wait until the MMA warps have left the slot
//           (mbarrier "done"); one lane stages the table tile global -> shared by 1-D TMA
//           (cp.async.bulk, mbarrier "tab"); then a5: seeds e^{i phi} for every (run of the
//           round, observation of the tile) in A-fragment order -- one exact evaluation
//           (range-reduced phase, sincospi) at the round's first unit, rotations by 4 units and
//           by 1 unit for the others (four independent chains) -- and arrive on mbarrier "seed".
//   MMA warps (8, two per sub-partition)  wait for "tab" and "seed"; per 4 observations:
//           A fragments (seeds; double-angle seeds by 4 flops), B fragments (table),
//           2 * NF * NT MMAs per unit; arrive on "done".  After the last tile of a round the
//           thread that holds all sums of a frequency solves (a9) and stores z (a10).
//
// The seed warps run up to NS steps ahead of the MMA warps, so the latency of the seed chains
// (which share the FP64 pipe with the MMAs) is off the MMA warps' critical path.
// Every accumulation order is fixed, so results are bitwise reproducible run to run.
#include "scan_mma_kernel.cuh"

namespace fredec {

namespace {

constexpr int kNW = 8;         // MMA warps per CTA (two per SM sub-partition)
constexpr int kSeedWarps = 4;  // seed warps per CTA (one per SM sub-partition)
constexpr int kThreads = (kNW + kSeedWarps) * 32;
// registers per thread after setmaxnreg: 128 * (2 * kRegsMma + kRegsSeed) <= 65536
constexpr int kRegsMma = 224, kRegsSeed = 56;

constexpr int kSeedGroups = 2;  // groups of 4 observations per seed warp and step at most (TI <= 32)

// non-blocking: has the phase of the given parity completed?
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

#define FREDEC_DMMA(c, a, b)                                                                  \
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"       \
        : "+d"((c)[0]), "+d"((c)[1])                                                          \
        : "d"(a), "d"(b))

// Position of a CTA in its sequence of (round, tile) steps.  The seed warps and the MMA warps
// walk the same sequence, each with its own cursor.
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

// a9/a10 for the units of one warp after the last tile of a round: this thread holds every sum
// of 2 * NT frequencies per unit.
template <int H, int NOCT, int NB>
__device__ __forceinline__ void solve_and_store(const Tiles<H, NOCT, NB>& acc, const MmaScanParams& p, int64_t b,
                                                int64_t unit0, int cnt, int lane)
{
    constexpr int R = 2 * H, NT = H / 4, NF = NB + 2;
    const SeriesInfo info = p.info[b];
    const int m = lane >> 2, q = lane & 3;
    const bool last_pass = p.pass + 1 == p.n_pass;
#pragma unroll
    for (int o = 0; o < NOCT; ++o) {
        if (o < cnt) {
            const int64_t k0 = ((unit0 + o) * 8 + m) * R;  // first grid point of the run
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
                            double* wsp = p.ws + (b * 7) * p.Kpad + k;
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
                        if (last_pass) p.z[b * p.K + k] = solve_z(YC, YS, CC, CS, Saa, Sab, Sbb, info.W);
                    }
                }
            }
        }
    }
}

// complex rotation (c, s) <- (c, s) * (rc, rs)
__device__ __forceinline__ void rotate(double& c, double& s, double rc, double rs)
{
    const double nc = fma(c, rc, -(s * rs));
    const double ns = fma(s, rc, c * rs);
    c = nc;
    s = ns;
}

template <int H, int NOCT, int NB>
__global__ void __launch_bounds__(kThreads, 1) scan_mma_kernel(MmaScanParams p)
{
    constexpr int R = 2 * H, NT = H / 4, NF = NB + 2, GROUP = NF * NT * 32, CAP = kNW * NOCT;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar_tab[kMmaMaxSlots], bar_seed[kMmaMaxSlots], bar_done[kMmaMaxSlots];

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int KS = p.TI / 4;  // groups of 4 observations per slot
    const int NS = p.NS;
    const size_t tab_bytes = (size_t)KS * GROUP * 8;
    const size_t slot_bytes = tab_bytes + (size_t)KS * CAP * 32 * sizeof(double2);
    const int ntiles = (int)((p.G4 + KS - 1) / KS);
    const int64_t U = p.U;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) {
            mbar_init(&bar_tab[s], 1);
            mbar_init(&bar_seed[s], kSeedWarps);
            mbar_init(&bar_done[s], kNW);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int64_t g0 = (int64_t)blockIdx.x * p.T / p.grid, g1 = (int64_t)(blockIdx.x + 1) * p.T / p.grid;
    Cursor c;
    c.init(g0, g1, U, CAP);

    if (wid >= kNW) {
        // ================= seed warps: table staging (a4) + seeds (a5) =====================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsSeed));
        const int pw = wid - kNW;
        const int m = lane >> 2, k = lane & 3;
        const SeedRec* srec = p.srec + k;
        int slot = 0;
        uint32_t par = 0;  // parity of the slot's current use
        bool first_lap = true;
        while (c.valid) {
            const int ngrp = (int)min((int64_t)KS, p.G4 - (int64_t)c.tile * KS);
            // this warp's records (groups pw, pw + 4) -- in flight while waiting for the slot
            const SeedRec* rp = srec + (c.b * p.G4 + (int64_t)c.tile * KS + pw) * 4;
            double rt[kSeedGroups], rcu[kSeedGroups], rsu[kSeedGroups], rc4[kSeedGroups], rs4[kSeedGroups];
#pragma unroll
            for (int j = 0; j < kSeedGroups; ++j) {
                if (pw + kSeedWarps * j < ngrp) {
                    const SeedRec* r = rp + kSeedWarps * j * 4;
                    rt[j] = r->t; rcu[j] = r->cu; rsu[j] = r->su; rc4[j] = r->c4; rs4[j] = r->s4;
                }
            }
            if (!first_lap) mbar_wait(&bar_done[slot], par ^ 1u);
            unsigned char* base = smem_raw + slot * slot_bytes;
            if (pw == 0 && lane == 0) {
                const uint32_t bytes = (uint32_t)ngrp * GROUP * 8u;
                mbar_expect_tx(&bar_tab[slot], bytes);
                bulk_g2s(base, p.tab + ((c.b * p.n_pass + p.pass) * p.G4 + (int64_t)c.tile * KS) * GROUP, bytes,
                         &bar_tab[slot]);
            }
            // centre of run m of the round's first unit: f_c = f0 + (run R + H - 1/2) df   (S1)
            const double kc = (double)((c.u * 8 + m) * R + H) - 0.5;
            const double fc = fma(kc, p.df, p.f0);
            double2* sb = reinterpret_cast<double2*>(base + tab_bytes) + lane;
#pragma unroll
            for (int j = 0; j < kSeedGroups; ++j) {
                const int ks = pw + kSeedWarps * j;
                if (ks < ngrp) {
                    double cs[CAP / 4], sn[CAP / 4];
                    sincospi(2.0 * frac_prod(fc, rt[j]), &sn[0], &cs[0]);
#pragma unroll
                    for (int q = 1; q < CAP / 4; ++q) {  // units 4, 8, 12: rotations by four units
                        cs[q] = cs[q - 1];
                        sn[q] = sn[q - 1];
                        rotate(cs[q], sn[q], rc4[j], rs4[j]);
                    }
                    double2* dst = sb + (size_t)ks * CAP * 32;
#pragma unroll
                    for (int i = 0; i < 4; ++i) {  // units 4q + i: CAP/4 independent chains
#pragma unroll
                        for (int q = 0; q < CAP / 4; ++q) {
                            dst[(4 * q + i) * 32] = make_double2(cs[q], sn[q]);
                            if (i < 3) rotate(cs[q], sn[q], rcu[j], rsu[j]);
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_seed[slot]);
            c.advance(ntiles, U, CAP);
            if (++slot == NS) {
                slot = 0;
                par ^= 1u;
                first_lap = false;
            }
        }
    } else {
        // ================= MMA warps: a6 (as a contraction), a9, a10 ========================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsMma));
        Tiles<H, NOCT, NB> acc;
        acc.clear();
        int slot = 0;
        uint32_t par = 0;
        bool ready = false;  // the slot's barriers were seen complete one step ahead
        while (c.valid) {
            int off, cnt;
            warp_share(c.n, wid, off, cnt);
            if (!ready) {
                mbar_wait(&bar_tab[slot], par);
                mbar_wait(&bar_seed[slot], par);
            }
            // look at the next slot's barriers now; the answer is needed after this step's MMAs
            int nslot = slot + 1;
            uint32_t npar = par;
            if (nslot == NS) {
                nslot = 0;
                npar ^= 1u;
            }
            ready = mbar_test(&bar_tab[nslot], npar) & mbar_test(&bar_seed[nslot], npar);
            if (cnt > 0) {
                const unsigned char* base = smem_raw + slot * slot_bytes;
                const double* tabs = reinterpret_cast<const double*>(base) + lane;
                const double2* sb = reinterpret_cast<const double2*>(base + tab_bytes) + (size_t)off * 32 + lane;
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
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_done[slot]);
            if (c.tile + 1 == ntiles && cnt > 0) {
                solve_and_store<H, NOCT, NB>(acc, p, c.b, c.u + off, cnt, lane);
                acc.clear();
            }
            c.advance(ntiles, U, CAP);
            slot = nslot;
            par = npar;
        }
    }
}

template <int H, int NOCT, int NB>
cudaError_t launch_one(const MmaScanParams& p, cudaStream_t stream)
{
    const size_t smem = (size_t)p.NS * mma_scan_slot_bytes(NB, p.TI);
    static size_t attr_smem = 0;
    if (smem > attr_smem) {
        cudaError_t e = cudaFuncSetAttribute(scan_mma_kernel<H, NOCT, NB>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_smem = smem;
    }
    if (p.NS < 2 || p.NS > kMmaMaxSlots || p.TI < 4 || p.TI % 4 || p.TI > 16 * kSeedGroups) return cudaErrorInvalidValue;
    scan_mma_kernel<H, NOCT, NB><<<p.grid, kThreads, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace

// (H, NOCT) per NB: NOCT * (2 + NB) * H accumulator doubles per thread
#define FREDEC_MMA_CONFIGS(X) \
    X(16, 2, 0) X(16, 1, 1) X(16, 1, 2) X(8, 2, 3) X(8, 1, 4) X(8, 1, 5) X(8, 1, 6) X(8, 1, 7) X(8, 1, 8) X(8, 1, 9)

MmaScanConfig mma_scan_config(int NB)
{
#define X(h, noct, nb) \
    if (NB == nb) return MmaScanConfig{h, noct, kNW};
    FREDEC_MMA_CONFIGS(X)
#undef X
    return MmaScanConfig{0, 0, 0};
}

size_t mma_scan_slot_bytes(int NB, int TI)
{
    const MmaScanConfig c = mma_scan_config(NB);
    return (size_t)(TI / 4) * (mma_group_doubles(c.H, NB) * 8 + (size_t)(c.NW * c.NOCT) * 32 * 16);
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
