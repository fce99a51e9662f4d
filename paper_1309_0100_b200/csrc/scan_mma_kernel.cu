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
// setmaxnreg) around a ring of NS shared-memory slots, slot = (table tile, seeds) of one step
// (laid out as the NS table tiles followed by the NS seed blocks):
//
//   seed warps (4, one per SM sub-partition; the FIRST warpgroup: the scheduler favours them)
//           wait until the MMA warps have left the slot
//           (mbarrier "done"); one lane stages the table tile global -> shared by 1-D TMA
//           (cp.async.bulk, mbarrier "tab"); then a5: seeds e^{i phi} for every (run of the
//           round, observation of the tile) in A-fragment order -- per lane one exact evaluation
//           (range-reduced phase, table + short polynomial) at the round's first unit for one run,
//           a rotation by four runs for a second run, and for both one rotation to the second
//           unit, then the two-term recurrence e_{u+1} = 2 cos(theta) e_u - e_{u-1} along the
//           units -- and arrive on mbarrier "seed".
//   MMA warps (8, two per sub-partition)  wait for "tab" and "seed"; per 4 observations:
//           A fragments (seeds; double-angle seeds by 2 FP64 instructions), B fragments (table),
//           2 * NF * NT MMAs per unit; arrive on "done".  After the last tile of a round the
//           thread that holds all sums of a frequency solves (a9) and stores z (a10) -- or, in
//           the FUSED instantiation (no periodogram wanted), tests its values for peaks and
//           keeps the warp's top-k list (a11, fused_emit).
//
// Rounds hold a power of two of units.  A round of fewer units than MMA warps (the tail of a
// CTA's range, or a short grid) splits the observations between the warps that share a unit
// (a8); their partial sums are added in fixed order through a per-CTA scratch in global memory.
// For one long series (at least one full round per CTA) the left-over rounds are instead cut
// across the observations BETWEEN CTAs ("shared" mode of the Cursor): every CTA ends with a piece
// of a left-over round, writes its partial sums to a workspace, and tail_solve_kernel adds the
// pieces in fixed order and solves -- also row a8, at the scale of the chip.
//
// The seed warps run up to NS steps ahead of the MMA warps, so the latency of the seed chains
// (which share the FP64 pipe with the MMAs) is off the MMA warps' critical path.
// Every accumulation order is fixed, so results are bitwise reproducible run to run.
#include "scan_mma_kernel.cuh"
#include "topk_list.cuh"

namespace fredec {

namespace {

constexpr int kNW = 8;         // MMA warps per CTA (two per SM sub-partition)
constexpr int kSeedWarps = 4;  // seed warps per CTA (one per SM sub-partition)
constexpr int kThreads = (kNW + kSeedWarps) * 32;
// Registers per thread after setmaxnreg.  The CTA is launched with kLaunchRegs registers for each of its
// 384 threads, and that pool is all setmaxnreg can redistribute (an increase beyond it waits for ever):
// 8 mma + 4 seed <= 12 kLaunchRegs.  The accumulators of an MMA thread are 2 * NOCT * (NB + 2) * H
// registers; up to 176 of them leave 72 registers to the seed warps, 192 (the largest tiles: the fewest
// seeds per MMA) leave 40.
constexpr int kLaunchRegs = 168;  // 65536 / 384 rounded down to the allocation unit of 8
template <int H, int NOCT, int NB>
struct ScanRegs {
    static constexpr int kAcc = 2 * NOCT * (NB + 2) * H;
#ifdef FREDEC_EXP_REGS_224_56  // measurement build: 8 registers moved from every MMA thread to the seed warps
    static constexpr int kMma = kAcc > 176 ? 224 : 216;
    static constexpr int kSeed = kAcc > 176 ? 56 : 72;
#else
    static constexpr int kMma = kAcc > 176 ? 232 : 216;
    static constexpr int kSeed = kAcc > 176 ? 40 : 72;
#endif
    static_assert(kAcc <= 192, "accumulators do not fit the MMA warps' registers");
    static_assert(kNW * kMma + kSeedWarps * kSeed <= (kNW + kSeedWarps) * kLaunchRegs, "register pool exceeded");
};

constexpr int kSeedGroups = 2;  // groups of 4 observations per seed warp and step at most (TI <= 32): one per half warp

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
// walk the same sequence, each with its own cursor.  Two ways of cutting the work:
//   ranges  (several series, or several passes): the CTA owns a contiguous range of units and
//           cuts it into rounds of a power of two of units; every round covers all tiles.
//   shared  (one series, one pass): every CTA first runs F full rounds of `cap` units of its own;
//           the rounds that are left over (fewer than one per CTA) are cut ACROSS THE OBSERVATIONS:
//           the CTA takes a contiguous piece of the sequence (left-over round, tile), i.e. at most
//           two SEGMENTS (round, tile range), whose partial sums go to a workspace (seg >= 0) and
//           are added and solved by tail_solve_kernel.  All CTAs then finish together, and no round
//           streams the table for a fraction of the work.
struct Cursor {
    int64_t g, g_end;  // ranges: first unit of this round / end of the CTA's range (global numbering)
    int64_t b, u;      // series and first unit (within the series) of the current round
    int n;             // units in the current round
    int tile;          // current tile
    int tile_end;      // end of the round's tile range
    int seg;           // >= 0: a segment of a left-over round (partial sums), -1: a whole round
    bool valid;
    // shared mode
    bool shared;
    int it, F, ntiles_, cap_;
    int64_t s0, s1, tail_u0;

    __device__ __forceinline__ void set_round(int64_t U, int cap)
    {
        if (shared) {
            n = cap_;
            b = 0;
            if (it < F) {
                u = ((int64_t)blockIdx.x * F + it) * cap_;
                tile = 0;
                tile_end = ntiles_;
                seg = -1;
                valid = true;
            } else {
                const int j = it - F;
                const int64_t r = s0 / ntiles_ + j;
                const int64_t lo = max(s0, r * ntiles_), hi = min(s1, (r + 1) * ntiles_);
                valid = j < 2 && lo < hi;
                u = tail_u0 + r * cap_;
                tile = (int)(lo - r * ntiles_);
                tile_end = (int)(hi - r * ntiles_);
                seg = 2 * (int)blockIdx.x + j;
            }
            return;
        }
        b = g / U;
        u = g - b * U;
        int64_t m = U - u;
        if (g_end - g < m) m = g_end - g;
        n = m < cap ? (int)m : cap;
        n = 1 << (31 - __clz(n));  // a power of two: rounds smaller than kNW split the observations
    }
    __device__ __forceinline__ void init(const MmaScanParams& p, int ntiles, int cap)
    {
        shared = p.shared != 0;
        tile = 0;
        tile_end = ntiles;
        seg = -1;
        b = u = 0;
        n = 0;
        g = g_end = 0;
        it = 0;
        F = p.F;
        ntiles_ = ntiles;
        cap_ = cap;
        s0 = s1 = tail_u0 = 0;
        if (shared) {
            const int64_t S = (int64_t)p.Rt * ntiles;
            s0 = (int64_t)blockIdx.x * S / p.grid;
            s1 = (int64_t)(blockIdx.x + 1) * S / p.grid;
            tail_u0 = (int64_t)p.grid * F * cap;
            set_round(p.U, cap);
            return;
        }
        g = (int64_t)blockIdx.x * p.T / p.grid;
        g_end = (int64_t)(blockIdx.x + 1) * p.T / p.grid;
        valid = g < g_end;
        if (valid) set_round(p.U, cap);
    }
    __device__ __forceinline__ void next_round(int64_t U, int cap)
    {
        if (shared) {
            ++it;
            set_round(U, cap);
            return;
        }
        g += n;
        valid = g < g_end;
        if (valid) set_round(U, cap);
    }
    __device__ __forceinline__ void advance(int ntiles, int64_t U, int cap)
    {
        if (++tile == tile_end) {
            tile = 0;
            tile_end = ntiles;
            next_round(U, cap);
        }
    }
};

// Role of MMA warp w in a round of n units (n a power of two <= kNW * NOCT):
//   n >= kNW  the warp owns cnt = n / kNW units starting at slot off, all observations (S = 1)
//   n <  kNW  S = kNW / n warps share the unit in slot off; the warp takes the groups of 4
//             observations with (group within the ring slot) % S == sp  (a8: observation split;
//             the partial sums are added in fixed order before the solve)
struct WarpRole {
    int off, cnt, S, sp;
};
__device__ __forceinline__ WarpRole warp_role(int n, int w)
{
    WarpRole r;
    if (n >= kNW) {
        r.cnt = n / kNW;
        r.off = w * r.cnt;
        r.S = 1;
        r.sp = 0;
    } else {
        r.cnt = 1;
        r.S = kNW / n;
        r.off = w / r.S;
        r.sp = w % r.S;
    }
    return r;
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

// Ring position of a warp: the slot it is at, the parity of the slot's current use, and whether
// the slot's "tab" and "seed" barriers were already seen complete (looked at one slot ahead).
struct RingPos {
    int slot;
    uint32_t par;
    bool ready;
};

// 2 x for a finite |x| < 2^1023 by an exponent increment on the integer pipe.  x = +-0 gives +-2^-1022
// (an absolute error of 2e-308) and a subnormal x a value below 2^-1021: both far below one rounding
// error of the sums they enter.
__device__ __forceinline__ double twice(double x)
{
    return __hiloint2double(__double2hiint(x) + 0x00100000, __double2loint(x));
}

// a6 for one group of 4 observations: A fragments (seeds), B fragments (table), 2 * NF * NT MMAs per unit.
// BASE_ONLY (passes after the first of a scan with more than 9 base functions): the y and w/2 families of
// such a pass have all-zero tables (their sums were formed by the first pass and are carried in the
// workspace), so their MMAs are left out.
template <int CNT, int H, int NOCT, int NB, bool BASE_ONLY>
__device__ __forceinline__ void mma_group(Tiles<H, NOCT, NB>& acc, const double2* tk, const double2* sk)
{
    constexpr int NT = H / 4, NF = NB + 2;
    double2 a[CNT];
    double c2[CNT], s2[CNT];
#pragma unroll
    for (int o = 0; o < CNT; ++o) {
        a[o] = sk[o * 32];
        // double-angle seeds with two FP64 instructions (every scalar FP64 instruction of an MMA warp
        // takes pipe cycles from the MMAs): 2 cos phi comes from the integer unit
        const double tc = twice(a[o].x);
        c2[o] = fma(tc, a[o].x, -1.0);  // cos 2 phi = 2 cos^2 phi - 1
        s2[o] = tc * a[o].y;            // sin 2 phi = 2 cos phi sin phi
    }
#pragma unroll
    for (int f = BASE_ONLY ? 1 : 0; f < (BASE_ONLY ? NF - 1 : NF); ++f) {
#pragma unroll
        for (int tp = 0; tp < NT / 2; ++tp) {
            const double2 b2 = tk[(f * (NT / 2) + tp) * 32];
#pragma unroll
            for (int h2 = 0; h2 < 2; ++h2) {
                const int t = 2 * tp + h2;
                const double bf = h2 == 0 ? b2.x : b2.y;
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

// ---- a6 with an explicit instruction order, for the configurations whose accumulators take 192 registers.
// With 40 registers left, the compiler's own schedule of mma_group (table loads hoisted far ahead)
// runs out of registers and pays for it in register moves, each of which costs the MMA stream an issue
// cycle.  Here the order is fixed with volatile asm: the 16-byte table loads run kDepth - 1 loads (8 or
// 12 MMAs) ahead of their MMAs and continue into the next group; the w family comes last in a group, its
// double-angle seeds are formed as one pair of adjacent FP64 instructions (a pair costs the MMA stream
// about as much as one single instruction) and the next group's seeds are loaded once the current ones
// are dead.
#define FREDEC_DMMA_V(c, a, b)                                                                       \
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"     \
                 : "+d"((c)[0]), "+d"((c)[1])                                                        \
                 : "d"(a), "d"(b))

__device__ __forceinline__ double2 lds128(uint32_t addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

// State of the load pipeline of one warp inside a ring slot.
template <int D>
struct LoadPipe {
    double2 a;     // seeds of the current group
    double2 b[D];  // table loads in flight
};

// One group of 4 observations of one unit (NOCT = 1).  tk / sk: shared-memory addresses of this lane's
// table fragments / seeds of the group; tk_next / sk_next: those of the group that follows (== tk / sk
// after the last one: the values are then loaded again and not used).
template <int H, int NB, int D>
__device__ __forceinline__ void mma_group_pipelined(Tiles<H, 1, NB>& acc, LoadPipe<D>& lp, uint32_t tk, uint32_t sk,
                                                    uint32_t tk_next, uint32_t sk_next)
{
    constexpr int NT = H / 4, NF = NB + 2, NP = NF * NT / 2, PW = (NF - 1) * (NT / 2);  // PW: first load of the w family
    static_assert(NP % D == 0 && PW >= 2, "load ring must divide the loads of a group");
    double c2 = 0.0, s2 = 0.0;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        const int q = p + D - 1;  // the load issued now
        lp.b[q % D] = q < NP ? lds128(tk + q * 512) : lds128(tk_next + (q - NP) * 512);
        if (p == PW - 1) {
            const double tc = twice(lp.a.x);
            asm volatile("fma.rn.f64 %0, %2, %3, 0dBFF0000000000000;\n\tmul.rn.f64 %1, %2, %4;"
                         : "=&d"(c2), "=&d"(s2)
                         : "d"(tc), "d"(lp.a.x), "d"(lp.a.y));  // cos 2 phi = 2 cos^2 phi - 1, sin 2 phi = 2 cos phi sin phi
        }
        const int f = p / (NT / 2), t0 = 2 * (p % (NT / 2));
        const double2 bb = lp.b[p % D];
        if (f < NF - 1) {
            FREDEC_DMMA_V(acc.v[0][0][f][t0], lp.a.x, bb.x);
            FREDEC_DMMA_V(acc.v[0][1][f][t0], lp.a.y, bb.x);
            FREDEC_DMMA_V(acc.v[0][0][f][t0 + 1], lp.a.x, bb.y);
            FREDEC_DMMA_V(acc.v[0][1][f][t0 + 1], lp.a.y, bb.y);
        } else {
            if (p == PW) lp.a = lds128(sk_next);  // the current seeds are dead from here on
            FREDEC_DMMA_V(acc.v[0][0][f][t0], c2, bb.x);
            FREDEC_DMMA_V(acc.v[0][1][f][t0], s2, bb.x);
            FREDEC_DMMA_V(acc.v[0][0][f][t0 + 1], c2, bb.y);
            FREDEC_DMMA_V(acc.v[0][1][f][t0 + 1], s2, bb.y);
        }
    }
}

// The loads of a group's successor are issued whether or not there is one (no selects in the loop): past
// the last group of a slot they read the next table tile / seed block of the ring or the kPipePad bytes
// the launch adds behind it, and the values are not used.
constexpr int kPipePad = 8192;

template <int H, int NB>
__device__ __forceinline__ void round_mma_pipelined(Tiles<H, 1, NB>& acc, RingPos& rp, const unsigned char* smem,
                                                    size_t slot_bytes, size_t tab_bytes, int NS, int KS, int64_t G4,
                                                    int tile0, int tile1, WarpRole role, int lane, uint64_t* bar_tab,
                                                    uint64_t* bar_seed, uint64_t* bar_done)
{
    constexpr int NT = H / 4, NF = NB + 2, CAP = kNW, D = 3;
    constexpr uint32_t GROUP_B = NF * NT * 32 * 8, SEED_B = CAP * 32 * 16;  // bytes per group: table, seeds
    static_assert(SEED_B + 16 <= kPipePad && (D - 1) * 512 <= kPipePad, "padding behind the ring too small");
    const int64_t g_end = min((int64_t)tile1 * KS, G4);
    const uint32_t seed_slot = (uint32_t)(slot_bytes - tab_bytes);
    const uint32_t tab_ring = smem_u32(smem), seed_ring = tab_ring + NS * (uint32_t)tab_bytes;
#pragma unroll 1
    for (int64_t g = (int64_t)tile0 * KS; g < g_end; g += KS) {
        const int ngrp = (int)min((int64_t)KS, g_end - g);
        if (!rp.ready) {
            mbar_wait(&bar_tab[rp.slot], rp.par);
            mbar_wait(&bar_seed[rp.slot], rp.par);
        }
        int nslot = rp.slot + 1;
        uint32_t npar = rp.par;
        if (nslot == NS) {
            nslot = 0;
            npar ^= 1u;
        }
        uint32_t tk = tab_ring + rp.slot * (uint32_t)tab_bytes + lane * 16;
        uint32_t sk = seed_ring + rp.slot * seed_slot + (role.off * 32 + lane) * 16;
        rp.ready = false;
        LoadPipe<D> lp;
        if (role.S == 1) {
            // every group of the slot, two per iteration; the next slot's barriers are looked at two or
            // three groups before the end, so that the MMA stream continues across slots.  (The load
            // pipeline restarts in every slot: carrying it across the slot boundary was measured and is
            // slower -- profiles/r2_experiments.md.)
            lp.a = lds128(sk);
#pragma unroll
            for (int q = 0; q < D - 1; ++q) lp.b[q] = lds128(tk + q * 512);
            int left = ngrp;
#pragma unroll 1
            for (; left >= 2; left -= 2) {
                if (left <= 3) rp.ready = mbar_test(&bar_tab[nslot], npar) & mbar_test(&bar_seed[nslot], npar);
                mma_group_pipelined<H, NB, D>(acc, lp, tk, sk, tk + GROUP_B, sk + SEED_B);
                mma_group_pipelined<H, NB, D>(acc, lp, tk + GROUP_B, sk + SEED_B, tk + 2 * GROUP_B, sk + 2 * SEED_B);
                tk += 2 * GROUP_B;
                sk += 2 * SEED_B;
            }
            if (left == 1) {
                if (ngrp == 1) rp.ready = mbar_test(&bar_tab[nslot], npar) & mbar_test(&bar_seed[nslot], npar);
                mma_group_pipelined<H, NB, D>(acc, lp, tk, sk, tk + GROUP_B, sk + SEED_B);
            }
        } else if (role.sp < ngrp) {
            // a8: the S warps of a unit take the slot's groups in turn
            const uint32_t tstep = GROUP_B * role.S, sstep = SEED_B * role.S;
            tk += role.sp * GROUP_B;
            sk += role.sp * SEED_B;
            lp.a = lds128(sk);
#pragma unroll
            for (int q = 0; q < D - 1; ++q) lp.b[q] = lds128(tk + q * 512);
#pragma unroll 1
            for (int ks = role.sp; ks < ngrp; ks += role.S) {
                const bool last = ks + role.S >= ngrp;
                mma_group_pipelined<H, NB, D>(acc, lp, tk, sk, last ? tk : tk + tstep, last ? sk : sk + sstep);
                tk += tstep;
                sk += sstep;
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&bar_done[rp.slot]);
        rp.slot = nslot;
        rp.par = npar;
    }
}

// a6 for one round: all tiles of the series, CNT = units this warp owns in the round.  The ring slot
// changes every KS groups; the next slot's barriers are looked at before the slot's last groups so
// that the MMA stream continues across slots.
template <int CNT, bool BASE_ONLY, int H, int NOCT, int NB>
__device__ __forceinline__ void round_mma(Tiles<H, NOCT, NB>& acc, RingPos& rp, const unsigned char* smem,
                                          size_t slot_bytes, size_t tab_bytes, int NS, int KS, int64_t G4,
                                          int tile0, int tile1, WarpRole role, int lane, uint64_t* bar_tab,
                                          uint64_t* bar_seed, uint64_t* bar_done)
{
    constexpr int NT = H / 4, NF = NB + 2, GROUP2 = NF * NT * 16, CAP = kNW * NOCT;  // GROUP2: double2 per group
    const int64_t g_end = min((int64_t)tile1 * KS, G4);
#pragma unroll 1
    for (int64_t g = (int64_t)tile0 * KS; g < g_end; g += KS) {
        const int ngrp = (int)min((int64_t)KS, g_end - g);
        if (!rp.ready) {
            mbar_wait(&bar_tab[rp.slot], rp.par);
            mbar_wait(&bar_seed[rp.slot], rp.par);
        }
        // ring layout: the NS table tiles, then the NS seed blocks
        const double2* tk = reinterpret_cast<const double2*>(smem + rp.slot * tab_bytes) + lane;  // this lane's table fragments
        const double2* sk = reinterpret_cast<const double2*>(smem + NS * tab_bytes + rp.slot * (slot_bytes - tab_bytes)) +
                            (size_t)role.off * 32 + lane;
        int nslot = rp.slot + 1;
        uint32_t npar = rp.par;
        if (nslot == NS) {
            nslot = 0;
            npar ^= 1u;
        }
        if (role.S == 1) {
            // all but the last two groups, the look at the next slot, the last two groups
            const int head = ngrp > 2 ? (ngrp - 2) & ~1 : 0;
#pragma unroll 1
            for (int ks = 0; ks < head; ks += 2) {
                mma_group<CNT, H, NOCT, NB, BASE_ONLY>(acc, tk, sk);
                mma_group<CNT, H, NOCT, NB, BASE_ONLY>(acc, tk + GROUP2, sk + CAP * 32);
                tk += 2 * GROUP2;
                sk += 2 * CAP * 32;
            }
            rp.ready = mbar_test(&bar_tab[nslot], npar) & mbar_test(&bar_seed[nslot], npar);
#pragma unroll 1
            for (int ks = head; ks < ngrp; ++ks) {
                mma_group<CNT, H, NOCT, NB, BASE_ONLY>(acc, tk, sk);
                tk += GROUP2;
                sk += CAP * 32;
            }
        } else {
            // a8: the S warps of a unit take the slot's groups in turn
            rp.ready = false;
#pragma unroll 1
            for (int ks = role.sp; ks < ngrp; ks += role.S)
                mma_group<CNT, H, NOCT, NB, BASE_ONLY>(acc, tk + (size_t)ks * GROUP2, sk + (size_t)ks * CAP * 32);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&bar_done[rp.slot]);
        rp.slot = nslot;
        rp.par = npar;
    }
}

// a9 for one frequency: 2x2 Schur solve with the singular rule S6
__device__ __forceinline__ double solve_z(double YC, double YS, double CC, double CS, double Saa, double Sab,
                                          double Sbb, double W)
{
#ifdef FREDEC_EXP_NO_SOLVE  // measurement build (wrong results): what the Schur solves cost
    return YC + YS + CC + CS + Saa + Sab + Sbb + W;
#endif
    const double SS = W - CC;  // <sin^2> = <1> - <cos^2>
    const double Scc = CC - Saa, Scs = CS - Sab, Sss = SS - Sbb;
    // two reciprocals instead of three divisions: the epilogue's FP64 instructions run while no MMA does
    double z = 0.0, ys = YS, piv2 = Sss;
    if (Scc > kTauTrial * CC) {  // S6: otherwise the cos column is in the span of the base
        const double r = 1.0 / Scc;
        const double q = Scs * r;
        z = YC * YC * r;
        ys = fma(-q, YC, YS);
        piv2 = fma(-q, Scs, Sss);
    }
    if (piv2 > kTauTrial * SS) z = fma(ys * ys, 1.0 / piv2, z);
    return z;
}

// a11 fused into the epilogue: the peaks among the 8R grid points of one unit, held as zu[t] (run position
// H + 4t + q) and zl[t] (position H - 1 - 4t - q) by thread (run m = lane / 4, q = lane % 4), go to the warp's
// sorted top-k list of its (series, CTA) pair in global memory; the unit's first and last point, whose outer
// neighbours belong to other units, go to the unit's edge record instead.  A unit with no value at or above
// the list's k-th entry costs two shuffles, one vote and two small loads.
template <int H>
__device__ __forceinline__ void fused_emit(double (&zu)[H / 4], double (&zl)[H / 4], const MmaScanParams& p, int64_t b,
                                           int64_t unit, int lane, int64_t group, int w, unsigned long long thr_bits)
{
    constexpr int R = 2 * H, NT = H / 4;
    constexpr unsigned kFull = 0xffffffffu;
    const int m = lane >> 2, q = lane & 3, quad = lane & ~3;
    const int64_t k0 = (unit * 8 + m) * R;
    // points past the end of the grid count as -infinity (S7): only the last unit of a series has any
    if ((unit + 1) * 8 * R > p.K) {
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            if (k0 + H + 4 * t + q >= p.K) zu[t] = -INFINITY;
            if (k0 + H - 1 - 4 * t - q >= p.K) zl[t] = -INFINITY;
        }
    }
    // edge record: the half of the peak test that the unit can decide (NaN counts as -infinity)
    const double z_first = sanitize(zl[NT - 1]), z_last = sanitize(zu[NT - 1]);
    const double right_of_first = __shfl_sync(kFull, z_first, 2);  // run 0, position 1
    const double left_of_last = __shfl_sync(kFull, z_last, 30);    // run 7, position R - 2
    double2* er = reinterpret_cast<double2*>(p.edges + (b * p.U + unit) * 4);
    if (lane == 3) __stcg(er, make_double2(z_first, z_first >= right_of_first ? 1.0 : 0.0));
    if (lane == 31) __stcg(er + 1, make_double2(z_last, z_last > left_of_last ? 1.0 : 0.0));
    // nothing at or above the group's threshold (the largest k-th entry of its full lists): no candidate.
    // One comparison per value and one vote (a NaN compares false) -- the common case must stay cheap: its
    // FP64 instructions compete with the MMAs of the sub-partition's other warp.
    const double group_thr = thr_bits ? __longlong_as_double((long long)thr_bits) : -INFINITY;
    bool reach = false;
#pragma unroll
    for (int t = 0; t < NT; ++t) reach |= (zu[t] >= group_thr) | (zl[t] >= group_thr);
    if (!__any_sync(kFull, reach)) return;
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        zu[t] = sanitize(zu[t]);
        zl[t] = sanitize(zl[t]);
    }
    // the warp's list
    const int k = p.fused_k;
    double* lz = p.list_z + ((size_t)group * kNW + w) * k;
    int64_t* li = p.list_i + ((size_t)group * kNW + w) * k;
    WarpList<1> L;
    L.init(k, lane);
    if (lane < k) {
        const int64_t id = __ldcg(li + lane);
        if (id >= 0 && id != kEmptyIdx) {
            L.z[0] = __ldcg(lz + lane);
            L.id[0] = id;
        }
    }
    L.thr_z = __shfl_sync(kFull, L.z[0], k - 1);
    L.thr_i = shfl_i64(L.id[0], k - 1);
    const double next_run_first = __shfl_down_sync(kFull, zl[NT - 1], 4);  // position 0 of run m + 1 (lane q = 3)
    const double prev_run_last = __shfl_up_sync(kFull, zu[NT - 1], 4);     // position R - 1 of run m - 1
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        // a step none of whose 64 points reaches the list's k-th entry (which rises as the unit is read) needs
        // no neighbours: almost every step of a unit that got this far
        if (!__any_sync(kFull, zu[t] >= L.thr_z || zl[t] >= L.thr_z)) continue;
        {  // upper half, position H + 4t + q: left is lane q - 1 | step t - 1 of q = 3 | own zl[0]
            const double a = __shfl_up_sync(kFull, zu[t], 1), c = __shfl_down_sync(kFull, zu[t], 1);
            const double a3 = __shfl_sync(kFull, zu[t > 0 ? t - 1 : 0], quad | 3);
            const double c0 = __shfl_sync(kFull, zu[t < NT - 1 ? t + 1 : t], quad);
            const double left = q > 0 ? a : (t > 0 ? a3 : zl[0]);
            const double right = q < 3 ? c : (t < NT - 1 ? c0 : next_run_first);
            const bool inner = !(t == NT - 1 && lane == 31);  // the unit's last point: edge record
            L.offer(zu[t], k0 + H + 4 * t + q, inner && zu[t] > left && zu[t] >= right);
        }
        {  // lower half, position H - 1 - 4t - q: right is lane q - 1 | step t - 1 of q = 3 | own zu[0]
            const double c = __shfl_up_sync(kFull, zl[t], 1), a = __shfl_down_sync(kFull, zl[t], 1);
            const double c3 = __shfl_sync(kFull, zl[t > 0 ? t - 1 : 0], quad | 3);
            const double a0 = __shfl_sync(kFull, zl[t < NT - 1 ? t + 1 : t], quad);
            const double right = q > 0 ? c : (t > 0 ? c3 : zu[0]);
            const double left = q < 3 ? a : (t < NT - 1 ? a0 : prev_run_last);
            const bool inner = !(t == NT - 1 && lane == 3);  // the unit's first point: edge record
            L.offer(zl[t], k0 + H - 1 - 4 * t - q, inner && zl[t] > left && zl[t] >= right);
        }
    }
    if (lane < k) {
        __stcg(lz + lane, L.z[0]);
        __stcg(li + lane, L.id[0]);
    }
    // a full list raises the group's threshold to its k-th entry (z >= 0: the bit patterns order like the values)
    if (lane == 0 && L.thr_i != kEmptyIdx && L.thr_z > group_thr)
        atomicMax(p.group_thr + group, (unsigned long long)__double_as_longlong(L.thr_z));
}

// a9/a10 for the units of one warp after the last tile of a round: this thread holds every sum
// of 2 * NT frequencies per unit.
// FUSED: nothing is stored; the values of a unit go to fused_emit (a11) with the warp's list (group, w).
template <int H, int NOCT, int NB, bool FUSED>
__device__ __forceinline__ void solve_and_store(const Tiles<H, NOCT, NB>& acc, const MmaScanParams& p, int64_t b,
                                                int64_t unit0, int cnt, int lane, int64_t group = 0, int w = 0)
{
    constexpr int R = 2 * H, NT = H / 4, NF = NB + 2;
    const SeriesInfo info = p.info[b];
    const int m = lane >> 2, q = lane & 3;
    const bool last_pass = p.pass + 1 == p.n_pass;
    if (FUSED && info.status != 0) return;  // no periodogram for this series: no lists, no edge records
    unsigned long long thr_bits = 0;
    if constexpr (FUSED) {
        // fetched HERE, before the solves, and used after them: volatile, so that the compiler does not sink
        // the load to its use and leave the epilogue waiting for a round trip to the L2
        asm volatile("ld.global.cg.u64 %0, [%1];" : "=l"(thr_bits) : "l"(p.group_thr + group) : "memory");
    }
#pragma unroll
    for (int o = 0; o < NOCT; ++o) {
        if (o < cnt) {
            const int64_t k0 = ((unit0 + o) * 8 + m) * R;  // first grid point of the run
            double zz[2][NT];  // FUSED: z at positions H + 4t + q (sg = 0) and H - 1 - 4t - q (sg = 1)
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
                    if constexpr (FUSED) {
                        zz[sg][t] = solve_z(YC, YS, CC, CS, Saa, Sab, Sbb, info.W);
                    } else if (k < p.K && info.status == 0) {
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
            if constexpr (FUSED) {
                // (a left-over round of the shared mode can reach past the last unit)
                if (unit0 + o < p.U) fused_emit<H>(zz[0], zz[1], p, b, unit0 + o, lane, group, w, thr_bits);
            }
        }
    }
}

// (cos, sin)(2 pi x) for |x| <= 1/2 (+ rounding): x = j/64 + r with |r| <= 1/128, the j part
// from a 64-entry table in shared memory, the r part by Taylor polynomials in y = 2 pi r
// (|y| <= 0.0491: truncation errors y^10/10! < 3e-20 and y^9/9! < 5e-18), combined by one
// complex rotation.  About 20 FP64 instructions instead of ~45 for sincospi.
__device__ __forceinline__ void sincos_turns(double x, const double2* trig64, double& c, double& s)
{
    const double jd = rint(x * 64.0);
    const double r = fma(jd, -0.015625, x);  // exact
    const double2 tj = trig64[(int)jd & 63];
    const double y = r * 6.283185307179586477;
    const double y2 = y * y;
    double pc = fma(y2, 1.0 / 40320.0, -1.0 / 720.0);
    pc = fma(pc, y2, 1.0 / 24.0);
    pc = fma(pc, y2, -0.5);
    pc = fma(pc, y2, 1.0);  // cos y
    double ps = fma(y2, -1.0 / 5040.0, 1.0 / 120.0);
    ps = fma(ps, y2, -1.0 / 6.0);
    ps = fma(ps * y2, y, y);  // sin y
    c = fma(tj.x, pc, -(tj.y * ps));
    s = fma(tj.y, pc, tj.x * ps);
}

// complex rotation (c, s) <- (c, s) * (rc, rs)
__device__ __forceinline__ void rotate(double& c, double& s, double rc, double rs)
{
    const double nc = fma(c, rc, -(s * rs));
    const double ns = fma(s, rc, c * rs);
    c = nc;
    s = ns;
}

template <int H, int NOCT, int NB, bool FUSED>
__global__ void __launch_bounds__(kThreads, 1) scan_mma_kernel(MmaScanParams p)
{
    constexpr int R = 2 * H, NT = H / 4, NF = NB + 2, GROUP = NF * NT * 32, CAP = kNW * NOCT;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar_tab[kMmaMaxSlots], bar_seed[kMmaMaxSlots], bar_done[kMmaMaxSlots];
    __shared__ double2 trig64[64];  // (cos, sin)(2 pi j / 64)

    // Warps 0-3 (the first warpgroup) are the seed warps, warps 4-11 the MMA warps `wid` = 0-7: the warp
    // scheduler favours the oldest (lowest-numbered) of the warps that compete for the FP64 pipe, and the
    // seed warps' few instructions must not queue behind the two MMA warps of their sub-partition.
#ifdef FREDEC_EXP_SEED_LAST  // measurement build: the seed warps are the last warpgroup
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const bool seed_warp = wid >= kNW;
    const int pw = wid - kNW;
#else
    const int tid = threadIdx.x, lane = tid & 31, wid = (tid >> 5) - kSeedWarps;
    const bool seed_warp = wid < 0;
    const int pw = wid + kSeedWarps;
#endif
    const int KS = p.TI / 4;  // groups of 4 observations per slot
    const int NS = p.NS;
    const size_t tab_bytes = (size_t)KS * GROUP * 8;
    const size_t slot_bytes = tab_bytes + (size_t)KS * CAP * 32 * sizeof(double2);
    const int ntiles = (int)((p.G4 + KS - 1) / KS);
    const int64_t U = p.U;

    if (tid >= 64 && tid < 128) {
        double sj, cj;
        sincospi((double)(tid - 64) * 0.03125, &sj, &cj);
        trig64[tid - 64] = make_double2(cj, sj);
    }
    if (tid == 0) {
        for (int s = 0; s < NS; ++s) {
            mbar_init(&bar_tab[s], 1);
            mbar_init(&bar_seed[s], kSeedWarps);
            mbar_init(&bar_done[s], kNW);
        }
        mbar_fence_init();
    }
    __syncthreads();

    Cursor c;
    c.init(p, ntiles, CAP);
    // the tail-solve kernel (launched with programmatic stream serialisation) may be scheduled as soon as SMs
    // become free; it waits for this grid's completion before it reads anything
    asm volatile("griddepcontrol.launch_dependents;");

    if (seed_warp) {
        // ================= seed warps: table staging (a4) + seeds (a5) =====================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(ScanRegs<H, NOCT, NB>::kSeed));
        // lane = (j, mp, k): group pw + 4 j of the slot, observation k of it, runs mp and mp + 4 of each
        // unit.  One exact evaluation per lane and step serves two runs (the second by a rotation).
        const int k = lane & 3, mp = (lane >> 2) & 3, ks = pw + kSeedWarps * (lane >> 4);
        const SeedRec* srec = p.srec + k;
        int slot = 0;
        uint32_t par = 0;  // parity of the slot's current use
        bool first_lap = true;
        // the lane's record is fetched one step ahead
        SeedRec nxt = {0.0, 1.0, 0.0, 2.0, 1.0, 0.0};
        auto fetch = [&](const Cursor& cc) {
            const int ng = (int)min((int64_t)KS, p.G4 - (int64_t)cc.tile * KS);
            if (ks < ng) nxt = srec[(cc.b * p.G4 + (int64_t)cc.tile * KS + ks) * 4];
        };
        if (c.valid) fetch(c);
        while (c.valid) {
            const int ngrp = (int)min((int64_t)KS, p.G4 - (int64_t)c.tile * KS);
            const SeedRec r = nxt;
            const int nunits = c.n;
            const int64_t u0 = c.u;
            const double* tab_src = p.tab + ((c.b * p.n_pass + p.pass) * p.G4 + (int64_t)c.tile * KS) * GROUP;
            c.advance(ntiles, U, CAP);
            if (c.valid) fetch(c);
            if (!first_lap) mbar_wait(&bar_done[slot], par ^ 1u);
            // ring layout: the NS table tiles, then the NS seed blocks (consecutive slots adjacent)
            unsigned char* tab_dst = smem_raw + slot * tab_bytes;
            unsigned char* seed_dst = smem_raw + NS * tab_bytes + slot * (slot_bytes - tab_bytes);
            if (pw == 0 && lane == 0) {
                const uint32_t bytes = (uint32_t)ngrp * GROUP * 8u;
                mbar_expect_tx(&bar_tab[slot], bytes);
                bulk_g2s(tab_dst, tab_src, bytes, &bar_tab[slot]);
            }
#ifdef FREDEC_EXP_STUB_SEEDS  // measurement build (wrong results): the seed warps stage the table and arrive
            if (false) {
#else
            if (ks < ngrp) {
#endif
                // centre of run mp of the round's first unit: f_c = f0 + (run R + H - 1/2) df   (S1)
                const double kc = (double)((u0 * 8 + mp) * R + H) - 0.5;
                const double fc = fma(kc, p.df, p.f0);
                // unit 0 of run mp exactly; run mp + 4 by one rotation; per run: unit 1 by one rotation,
                // then the two-term recurrence e_{u+1} = 2 cos(theta) e_u - e_{u-1} (theta = one unit step)
                double ca0, sa0;
                sincos_turns(frac_prod(fc, r.t), trig64, ca0, sa0);
                double cb0 = ca0, sb0 = sa0;
                rotate(cb0, sb0, r.c4, r.s4);
                double ca1 = ca0, sa1 = sa0, cb1 = cb0, sb1 = sb0;
                rotate(ca1, sa1, r.cu, r.su);
                rotate(cb1, sb1, r.cu, r.su);
                double2* da = reinterpret_cast<double2*>(seed_dst) + (size_t)ks * CAP * 32 + mp * 4 + k;
                double2* db = da + 16;  // run mp + 4
                da[0] = make_double2(ca0, sa0);
                db[0] = make_double2(cb0, sb0);
                da[32] = make_double2(ca1, sa1);
                db[32] = make_double2(cb1, sb1);
#pragma unroll
                for (int u = 2; u < CAP; ++u) {
                    if (u >= nunits) break;  // rounds of fewer units need fewer seeds
                    const double ca2 = fma(r.tcu, ca1, -ca0), sa2 = fma(r.tcu, sa1, -sa0);
                    const double cb2 = fma(r.tcu, cb1, -cb0), sb2 = fma(r.tcu, sb1, -sb0);
                    da[u * 32] = make_double2(ca2, sa2);
                    db[u * 32] = make_double2(cb2, sb2);
                    ca0 = ca1; sa0 = sa1; ca1 = ca2; sa1 = sa2;
                    cb0 = cb1; sb0 = sb1; cb1 = cb2; sb1 = sb2;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_seed[slot]);
            if (++slot == NS) {
                slot = 0;
                par ^= 1u;
                first_lap = false;
            }
        }
    } else {
        // ================= MMA warps: a6 (as a contraction), a9, a10 ========================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(ScanRegs<H, NOCT, NB>::kMma));
        Tiles<H, NOCT, NB> acc;
        acc.clear();
        RingPos rp = {0, 0u, false};
        while (c.valid) {  // one round per iteration
            const WarpRole role = warp_role(c.n, wid);
#define FREDEC_ROUND(CNT) \
    round_mma<CNT, false>(acc, rp, smem_raw, slot_bytes, tab_bytes, NS, KS, p.G4, c.tile, c.tile_end, role, lane, bar_tab, \
                   bar_seed, bar_done)
            if (NB == 8 && p.pass > 0) {
                // a later pass of a multi-pass scan: base families only (NB == 8 is the pass size)
                round_mma<1, true>(acc, rp, smem_raw, slot_bytes, tab_bytes, NS, KS, p.G4, c.tile, c.tile_end, role, lane,
                                   bar_tab, bar_seed, bar_done);
            } else if constexpr (ScanRegs<H, NOCT, NB>::kAcc > 176) {
                round_mma_pipelined<H, NB>(acc, rp, smem_raw, slot_bytes, tab_bytes, NS, KS, p.G4, c.tile, c.tile_end,
                                           role, lane, bar_tab, bar_seed, bar_done);
            } else if (NOCT == 1 || role.cnt == 1) {
                FREDEC_ROUND(1);
            } else if (NOCT == 2 || role.cnt == 2) {
                FREDEC_ROUND((NOCT >= 2 ? 2 : 1));
            } else {
                FREDEC_ROUND(NOCT);
            }
#undef FREDEC_ROUND
            bool solve = true;
            if (role.S > 1) {
                // a8: the S warps of the unit add their partial sums in fixed order (sp = 1, 2, ...
                // onto sp = 0) through the CTA's scratch in global memory; warp sp = 0 solves
                constexpr int ACC1 = 2 * NF * NT * 2;
                double* mine = p.red + ((size_t)blockIdx.x * kNW + wid) * (ACC1 * 32) + lane;
                if (role.sp > 0) {
#pragma unroll
                    for (int x = 0; x < 2; ++x)
#pragma unroll
                        for (int f = 0; f < NF; ++f)
#pragma unroll
                            for (int t = 0; t < NT; ++t) {
                                __stcg(mine + (((x * NF + f) * NT + t) * 2 + 0) * 32, acc.v[0][x][f][t][0]);
                                __stcg(mine + (((x * NF + f) * NT + t) * 2 + 1) * 32, acc.v[0][x][f][t][1]);
                            }
                    solve = false;
                }
                // Named barrier of the S warps that share the unit.  The id depends on S as well as on
                // the unit (S = 2: ids 1-4, S = 4: ids 5-6, S = 8: id 7), so an id always has the same
                // participants and thread count, whatever the sequence of round sizes.
                const int bar_id = (role.S == 2 ? 1 : role.S == 4 ? 5 : 7) + role.off;
                asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "r"(role.S * 32) : "memory");
                if (role.sp == 0) {
                    for (int sp = 1; sp < role.S; ++sp) {
                        const double* other = mine + (size_t)sp * (ACC1 * 32);
#pragma unroll
                        for (int x = 0; x < 2; ++x)
#pragma unroll
                            for (int f = 0; f < NF; ++f)
#pragma unroll
                                for (int t = 0; t < NT; ++t) {
                                    acc.v[0][x][f][t][0] += __ldcg(other + (((x * NF + f) * NT + t) * 2 + 0) * 32);
                                    acc.v[0][x][f][t][1] += __ldcg(other + (((x * NF + f) * NT + t) * 2 + 1) * 32);
                                }
                    }
                }
                // the writers may not start the next split round's stores into `mine` before warp
                // sp = 0 has read this round's (the seed warps run ahead, so nothing else holds them)
                asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "r"(role.S * 32) : "memory");
            }
            if (c.seg >= 0) {
                // a segment of a left-over round: the sums over its tiles go to the workspace
                constexpr int ACCW = NOCT * 2 * NF * NT * 2;
                double* dst = p.part + ((size_t)c.seg * kNW + wid) * (ACCW * 32) + lane;
#pragma unroll
                for (int o = 0; o < NOCT; ++o)
#pragma unroll
                    for (int x = 0; x < 2; ++x)
#pragma unroll
                        for (int f = 0; f < NF; ++f)
#pragma unroll
                            for (int t = 0; t < NT; ++t) {
                                __stcg(dst + ((((o * 2 + x) * NF + f) * NT + t) * 2 + 0) * 32, acc.v[o][x][f][t][0]);
                                __stcg(dst + ((((o * 2 + x) * NF + f) * NT + t) * 2 + 1) * 32, acc.v[o][x][f][t][1]);
                            }
            } else if (solve) {
                solve_and_store<H, NOCT, NB, FUSED>(acc, p, c.b, c.u + role.off, role.cnt, lane, c.b + blockIdx.x, wid);
            }
            acc.clear();
            c.next_round(U, CAP);
        }
    }
}

// Shared mode: adds the partial sums of the segments of left-over round blockIdx.x in the order of
// the CTAs that produced them (fixed: bitwise reproducible), then a9/a10 as in the scan kernel.
template <int H, int NOCT, int NB, bool FUSED>
__global__ void __launch_bounds__(kNW * 32) tail_solve_kernel(MmaScanParams p)
{
    constexpr int NT = H / 4, NF = NB + 2, CAP = kNW * NOCT, ACCW = NOCT * 2 * NF * NT * 2;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int KS = p.TI / 4;
    const int ntiles = (int)((p.G4 + KS - 1) / KS);
    const int64_t r = blockIdx.x, S = (int64_t)p.Rt * ntiles;
    Tiles<H, NOCT, NB> acc;
    acc.clear();
    // launched with programmatic stream serialisation: everything above overlaps the scan kernel's end; the
    // partial sums are read only after the scan kernel has completed and flushed
    asm volatile("griddepcontrol.wait;" ::: "memory");
    // only the CTAs whose piece [cta S / grid, (cta + 1) S / grid) can meet the round's steps [r, r + 1) ntiles
    const int c_lo = (int)max((int64_t)0, r * ntiles * p.grid / S - 1);
    const int c_hi = (int)min((int64_t)p.grid - 1, ((r + 1) * ntiles * p.grid + S - 1) / S);
    for (int cta = c_lo; cta <= c_hi; ++cta) {
        const int64_t s0 = (int64_t)cta * S / p.grid, s1 = (int64_t)(cta + 1) * S / p.grid;
        const int64_t j = r - s0 / ntiles;
        if (j < 0 || j > 1) continue;
        if (max(s0, r * ntiles) >= min(s1, (r + 1) * ntiles)) continue;
        const double* src = p.part + ((size_t)(2 * cta + (int)j) * kNW + wid) * (ACCW * 32) + lane;
#pragma unroll
        for (int o = 0; o < NOCT; ++o)
#pragma unroll
            for (int x = 0; x < 2; ++x)
#pragma unroll
                for (int f = 0; f < NF; ++f)
#pragma unroll
                    for (int t = 0; t < NT; ++t) {
                        acc.v[o][x][f][t][0] += __ldcg(src + ((((o * 2 + x) * NF + f) * NT + t) * 2 + 0) * 32);
                        acc.v[o][x][f][t][1] += __ldcg(src + ((((o * 2 + x) * NF + f) * NT + t) * 2 + 1) * 32);
                    }
    }
    const int64_t u = (int64_t)p.grid * p.F * CAP + r * CAP + wid * NOCT;
    solve_and_store<H, NOCT, NB, FUSED>(acc, p, 0, u, NOCT, lane, p.tail_group0 + r, wid);
}

template <int H, int NOCT, int NB, bool FUSED>
cudaError_t launch_one(const MmaScanParams& p, cudaStream_t stream)
{
    const size_t smem = (size_t)p.NS * mma_scan_slot_bytes(NB, p.TI) + kPipePad;
    static size_t attr_smem = 0;
    if (smem > attr_smem) {
        cudaError_t e = cudaFuncSetAttribute(scan_mma_kernel<H, NOCT, NB, FUSED>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_smem = smem;
    }
    if (p.NS < 2 || p.NS > kMmaMaxSlots || p.TI < 4 || p.TI % 4 || p.TI > 16 * kSeedGroups) return cudaErrorInvalidValue;
    if (FUSED && (p.n_pass != 1 || p.fused_k < 1 || p.fused_k > kFusedMaxK)) return cudaErrorInvalidValue;
    scan_mma_kernel<H, NOCT, NB, FUSED><<<p.grid, kThreads, smem, stream>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess || !p.shared || p.Rt == 0) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)p.Rt, 1, 1);
    cfg.blockDim = dim3(kNW * 32, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, tail_solve_kernel<H, NOCT, NB, FUSED>, p);
}

}  // namespace

// (H, NOCT) per NB: NOCT * (2 + NB) * H accumulator doubles per thread.  The seeds (the only FP64 scalar
// work per pair) are one complex number per (run of 2H frequencies, observation): the longest run the
// registers allow, 96 accumulator doubles, for d <= 2 and d = 4.
#define FREDEC_MMA_CONFIGS(X) \
    X(48, 1, 0) X(32, 1, 1) X(24, 1, 2) X(16, 1, 3) X(16, 1, 4) X(8, 1, 5) X(8, 1, 6) X(8, 1, 7) X(8, 1, 8) X(8, 1, 9)

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

size_t mma_red_doubles(int NB)
{
    const MmaScanConfig c = mma_scan_config(NB);
    return (size_t)2 * mma_nf(NB) * mma_nt(c.H) * 2 * 32;
}

size_t mma_part_doubles(int NB)
{
    const MmaScanConfig c = mma_scan_config(NB);
    return (size_t)c.NOCT * 2 * mma_nf(NB) * mma_nt(c.H) * 2 * 32;
}

cudaError_t launch_mma_scan(int NB, const MmaScanParams& p, cudaStream_t stream)
{
#define X(h, noct, nb) \
    if (NB == nb) return p.fused_k > 0 ? launch_one<h, noct, nb, true>(p, stream) : launch_one<h, noct, nb, false>(p, stream);
    FREDEC_MMA_CONFIGS(X)
#undef X
    return cudaErrorInvalidValue;
}

}  // namespace fredec
