// scan_kernel.cu -- steps a4-a10: the periodogram scan kernel for sm_100a.
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
// Work decomposition.  A thread owns a RUN of R consecutive grid frequencies and keeps their
// R*(4+2NB) sums in registers; a CTA owns J = 32*FW consecutive runs.  Observation records
// are staged tile by tile into shared memory with 1-D TMA bulk copies (cp.async.bulk +
// mbarrier, double buffered) and read as warp-broadcast LDS.128.  Per tile:
//
//   phase A (seeds)  e^{i phi} at the FIRST frequency of every run, for every observation of
//                    the tile, into shared memory.  Along the run axis consecutive seeds
//                    differ by the per-observation rotation e^{i 2 pi R df t'}: every
//                    kSeedChain-th seed is evaluated from the exactly range-reduced phase
//                    (frac(f t') by an FMA split, then sincospi), the ones in between by the
//                    FP64 rotation recurrence.  Cost: ~5 FP64 instructions per seed.
//   phase B (sums)   each thread walks the tile's observations; for each it loads its seed,
//                    makes the second starting value with one rotation by e^{i 2 pi df t'}
//                    and then advances along the frequency axis with the two-term form of
//                    the rotation recurrence, c_{r+1} = 2 cos(d) c_r - c_{r-1} (same for s),
//                    2 FMA per step, re-seeded every R steps.  No per-pair sincos.
//
// Partial sums of warps that split the observations of a tile are combined in a fixed order
// through shared memory (bitwise reproducible run to run).
#include "scan_kernel.cuh"

namespace fredec {

namespace {

// Tunables (overridable with -D for experiments under _work/).
#ifndef FREDEC_SCAN_MAXT
#define FREDEC_SCAN_MAXT 128   // threads per CTA the kernel is compiled for
#endif
// CTAs per SM the register allocation targets: 3 (<= 168 registers) when the R*(4+2NB) FP64
// accumulators leave room, else 2 (<= 255 registers); spilling in the hot loop is ruinous.
#ifdef FREDEC_SCAN_MINB
__host__ __device__ constexpr int scan_min_blocks(int, int) { return FREDEC_SCAN_MINB; }
#else
__host__ __device__ constexpr int scan_min_blocks(int R, int NB) { return 2 * R * (4 + 2 * NB) + 64 <= 168 ? 3 : 2; }
#endif
#ifndef FREDEC_SCAN_PREFETCH
#define FREDEC_SCAN_PREFETCH 1 // load observation i+1's record and seed before computing i
#endif
constexpr int kMaxScanThreads = FREDEC_SCAN_MAXT;

template <int R, int NB>
struct Acc {
    double YC[R], YS[R], CC[R], CS[R];
    double A[R][NB > 0 ? NB : 1], B[R][NB > 0 ? NB : 1];

    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            YC[r] = YS[r] = CC[r] = CS[r] = 0.0;
#pragma unroll
            for (int j = 0; j < NB; ++j) A[r][j] = B[r][j] = 0.0;
        }
    }
    // visit every accumulator with a compile-time index (used by the split reduction)
    template <class F>
    __device__ __forceinline__ void for_each(F&& f)
    {
        int a = 0;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            f(YC[r], a++);
            f(YS[r], a++);
            f(CC[r], a++);
            f(CS[r], a++);
#pragma unroll
            for (int j = 0; j < NB; ++j) {
                f(A[r][j], a++);
                f(B[r][j], a++);
            }
        }
    }
};

// registers holding one observation's record and this thread's seed for it
template <int NB>
struct ObsRegs {
    static constexpr int NP = (NB + 1) / 2;
    double2 h0, h1, h3, sd;
    double2 pq[NP > 0 ? NP : 1];
    __device__ __forceinline__ void load(const double* tb, const double2* myseed, int i, int RS)
    {
        const double2* r2 = reinterpret_cast<const double2*>(tb + (size_t)i * RS);
        h0 = r2[0];  // t', 2 cos d
        h1 = r2[1];  // cos d, sin d
        h3 = r2[3];  // w, y
#pragma unroll
        for (int m = 0; m < NP; ++m) pq[m] = r2[kHdr / 2 + m];
        sd = myseed[i];
    }
    __device__ __forceinline__ double p(int j) const { return (j & 1) ? pq[j >> 1].y : pq[j >> 1].x; }
};


// ---------------------------------------------------------------------------------------
// Hand-ordered FP64 instruction stream of phase B.
//
// On sm_100 a DFMA that reads three distinct registers from the register file occupies the
// FP64 pipe for 3 cycles instead of 2 (measured: 24.5 vs 33.8 TFLOP/s chip-wide).  An operand
// that the PREVIOUS instruction of the warp read in the same operand slot comes from the
// operand-reuse cache instead.  The accumulation is therefore issued multiplier-major:
// runs of R consecutive FMAs share their first operand (y, p_j or w), so all but the first
// read only two registers.  `asm volatile` pins that order (ptxas otherwise re-interleaves
// the stream and loses about half of the reuse).  The recurrence of the NEXT observation
// is slotted in between the runs, one step per boundary, which hides its dependent latency.
// ---------------------------------------------------------------------------------------
#define FREDEC_DFMA_ACC(accv, m, v) asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(accv) : "d"(m), "d"(v))
#define FREDEC_DMUL(dst, a, b) asm volatile("mul.rn.f64 %0, %1, %2;" : "=d"(dst) : "d"(a), "d"(b))
#define FREDEC_DFMA(dst, a, b, c) asm volatile("fma.rn.f64 %0, %1, %2, %3;" : "=d"(dst) : "d"(a), "d"(b), "d"(c))
#define FREDEC_DFMS(dst, a, b, c) \
    asm volatile("{\n\t.reg .f64 t;\n\tneg.f64 t, %3;\n\tfma.rn.f64 %0, %1, %2, t;\n\t}" : "=d"(dst) : "d"(a), "d"(b), "d"(c))

// (cos, sin) of one observation at the R frequencies of the thread's run
template <int R>
struct Trig {
    double c[R], s[R];
    double t1, t2;  // partial products of the first rotation
    // a7, step q of the run: q = 0 seed + partial products, q = 1 rotation by d,
    // q >= 2 two-term recurrence c_q = 2 cos(d) c_{q-1} - c_{q-2}
    template <int NB>
    __device__ __forceinline__ void step(int q, const ObsRegs<NB>& o)
    {
        if (q == 0) {
            c[0] = o.sd.x;
            s[0] = o.sd.y;
            FREDEC_DMUL(t1, s[0], o.h1.y);
            FREDEC_DMUL(t2, c[0], o.h1.y);
        } else if (q == 1) {
            FREDEC_DFMS(c[1], c[0], o.h1.x, t1);
            FREDEC_DFMA(s[1], s[0], o.h1.x, t2);
        } else {
            FREDEC_DFMS(c[q], o.h0.y, c[q - 1], c[q - 2]);
            FREDEC_DFMS(s[q], o.h0.y, s[q - 1], s[q - 2]);
        }
    }
    template <int NB>
    __device__ __forceinline__ void build(const ObsRegs<NB>& o)
    {
#pragma unroll
        for (int q = 0; q < R; ++q) step(q, o);
    }
};

// a6 for observation `oc`, whose trig values are in `t`; as each (c_r, s_r) is used for the
// last time it is replaced IN PLACE by the value of the next observation `on` (a7), so only
// one run of trig values is live and the recurrence's latency hides behind the tail's FMAs.
template <int R, int NB>
__device__ __forceinline__ void accumulate_and_build(Acc<R, NB>& acc, const ObsRegs<NB>& oc, Trig<R>& t,
                                                     const ObsRegs<NB>& on)
{
    const double y = oc.h3.y, w = oc.h3.x;
#pragma unroll
    for (int r = 0; r < R; ++r) FREDEC_DFMA_ACC(acc.YC[r], y, t.c[r]);
#pragma unroll
    for (int r = 0; r < R; ++r) FREDEC_DFMA_ACC(acc.YS[r], y, t.s[r]);
#pragma unroll
    for (int j = 0; j < NB; ++j) {
        const double pj = oc.p(j);
#pragma unroll
        for (int r = 0; r < R; ++r) FREDEC_DFMA_ACC(acc.A[r][j], pj, t.c[r]);
#pragma unroll
        for (int r = 0; r < R; ++r) FREDEC_DFMA_ACC(acc.B[r][j], pj, t.s[r]);
    }
    double u[R];
    FREDEC_DMUL(u[0], w, t.c[0]);
    if (R > 1) FREDEC_DMUL(u[1], w, t.c[1]);
#pragma unroll
    for (int r = 0; r < R; ++r) {
        FREDEC_DFMA_ACC(acc.CC[r], u[r], t.c[r]);
        FREDEC_DFMA_ACC(acc.CS[r], u[r], t.s[r]);
        if (r + 2 < R) FREDEC_DMUL(u[r + 2], w, t.c[r + 2]);
        t.template step<NB>(r, on);  // (c_r, s_r) of this observation are dead: next one's go there
    }
}

// one thread's share of phase A: two independent chains of kSeedChain seeds
constexpr int kSeedChain = 16;

template <int R, int NB>
__global__ void __launch_bounds__(kMaxScanThreads, scan_min_blocks(R, NB)) scan_kernel(ScanParams p)
{
    constexpr int RS = rec_stride(NB);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar[2];

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int FW = p.FW, S = p.S, TI = p.TI;
    const int J = FW * 32, T = J * S;
    const int SROW = TI + 1;  // seed row stride in double2 (odd: conflict-free both ways)
    double* const tile_buf = reinterpret_cast<double*>(smem_raw);                      // [2][TI][RS]
    double2* const seeds = reinterpret_cast<double2*>(tile_buf + (size_t)2 * TI * RS);  // [J][SROW]

    const int fw = wid % FW, sp = wid / FW;
    const int jrun = fw * 32 + lane;  // this thread's run within the CTA
    const int64_t b = blockIdx.y;
    const SeriesInfo info = p.info[b];
    if (info.status != 0) return;  // uniform over the CTA; the host reports the error

    const int64_t N = p.N, K = p.K;
    const int64_t run0 = (int64_t)blockIdx.x * J;  // first run of the CTA
    const int64_t k0 = (run0 + jrun) * R;
    const bool active = k0 < K;
    const double* rec = p.rec + ((b * p.n_pass + p.pass) * N) * RS;

    const int ntiles = (int)((N + TI - 1) / TI);
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int tile) {
        const int64_t first = (int64_t)tile * TI;
        const int rows = (int)min((int64_t)TI, N - first);
        const uint32_t bytes = (uint32_t)rows * RS * 8u;
        uint64_t* mb = &bar[tile & 1];
        mbar_expect_tx(mb, bytes);
        bulk_g2s(tile_buf + (size_t)(tile & 1) * TI * RS, rec + first * RS, bytes, mb);
    };
    if (tid == 0) issue(0);

    Acc<R, NB> acc;
    acc.clear();

    const int rows_per_split = TI / S;
    const int nseg = J / kSeedChain;  // chains per observation
    for (int tile = 0; tile < ntiles; ++tile) {
        if (tid == 0 && tile + 1 < ntiles) issue(tile + 1);  // stage (tile+1)&1 was released by the
                                                             // __syncthreads that ended tile-1
        mbar_wait(&bar[tile & 1], (uint32_t)((tile >> 1) & 1));
        const int rows = (int)min((int64_t)TI, N - (int64_t)tile * TI);
        const double* tb = tile_buf + (size_t)(tile & 1) * TI * RS;

        // ---- phase A: seeds[j][i] = (cos, sin)(2 pi f_{(run0+j)R} t'_i) -----------------------
        // chain c = (segment g, observation i), i fastest => conflict-free STS.128
        const int nchains = nseg * rows;
        for (int c0 = tid; c0 < nchains; c0 += 2 * T) {
            const int c1 = c0 + T;
            const bool two = c1 < nchains;
            const int ia = c0 % rows, ga = c0 / rows;
            const int ib = two ? c1 % rows : ia, gb = two ? c1 / rows : ga;
            const double2* ra = reinterpret_cast<const double2*>(tb + (size_t)ia * RS);
            const double2* rb = reinterpret_cast<const double2*>(tb + (size_t)ib * RS);
            const double ta = ra[0].x, tbb = rb[0].x;
            const double2 Ga = ra[2], Gb = rb[2];  // (cos, sin) of one run step
            // exact seeds at the head of each chain (S1: f = fl(f0 + k df))
            const double fa = fma((double)((run0 + (int64_t)ga * kSeedChain) * R), p.df, p.f0);
            const double fb = fma((double)((run0 + (int64_t)gb * kSeedChain) * R), p.df, p.f0);
            double ca, sa, cb, sb;
            sincospi(2.0 * frac_prod(fa, ta), &sa, &ca);
            sincospi(2.0 * frac_prod(fb, tbb), &sb, &cb);
            double2* da = seeds + (size_t)(ga * kSeedChain) * SROW + ia;
            double2* db = seeds + (size_t)(gb * kSeedChain) * SROW + ib;
#pragma unroll
            for (int q = 0; q < kSeedChain; ++q) {
                da[(size_t)q * SROW] = make_double2(ca, sa);
                if (two) db[(size_t)q * SROW] = make_double2(cb, sb);
                if (q + 1 < kSeedChain) {
                    const double na = fma(ca, Ga.x, -(sa * Ga.y));
                    const double ma = fma(sa, Ga.x, ca * Ga.y);
                    const double nb = fma(cb, Gb.x, -(sb * Gb.y));
                    const double mb = fma(sb, Gb.x, cb * Gb.y);
                    ca = na; sa = ma; cb = nb; sb = mb;
                }
            }
        }
        __syncthreads();

        // ---- phase B: accumulate this warp's share of the tile --------------------------------
        const int i_begin = sp * rows_per_split;
        const int i_end = min(rows, i_begin + rows_per_split);
        if (active && i_begin < i_end) {
            const double2* myseed = seeds + (size_t)jrun * SROW;
            // Software pipeline over observations (unrolled by two so that the record registers
            // alternate): while observation i is accumulated, the record of i+1 is in flight and
            // its (cos, sin) run replaces i's in place.
            ObsRegs<NB> oa, ob;
            Trig<R> trig;
            oa.load(tb, myseed, i_begin, RS);
            trig.build(oa);
            for (int i = i_begin; i < i_end; i += 2) {
                ob.load(tb, myseed, min(i + 1, i_end - 1), RS);
                accumulate_and_build<R, NB>(acc, oa, trig, ob);
                if (i + 1 < i_end) {
                    oa.load(tb, myseed, min(i + 2, i_end - 1), RS);
                    accumulate_and_build<R, NB>(acc, ob, trig, oa);
                }
            }
        }
        __syncthreads();
    }

    // ---- a8: combine the observation split in a fixed order ------------------------------
    if (S > 1) {
        double* red = tile_buf;  // every bulk copy has completed and been consumed
        const int col = jrun;
        for (int q = 1; q < S; ++q) {
            if (sp == q) acc.for_each([&](double& v, int a) { red[a * J + col] = v; });
            __syncthreads();
            if (sp == 0) acc.for_each([&](double& v, int a) { v += red[a * J + col]; });
            __syncthreads();
        }
    }
    if (sp != 0 || !active) return;

    // ---- a9: per-frequency solve ------------------------------------------------------------
    double* zp = p.z + b * K + k0;
    double zr[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        double Saa = 0.0, Sab = 0.0, Sbb = 0.0;
#pragma unroll
        for (int j = 0; j < NB; ++j) {
            Saa = fma(acc.A[r][j], acc.A[r][j], Saa);
            Sab = fma(acc.A[r][j], acc.B[r][j], Sab);
            Sbb = fma(acc.B[r][j], acc.B[r][j], Sbb);
        }
        double YC = acc.YC[r], YS = acc.YS[r], CC = acc.CC[r], CS = acc.CS[r];
        if (p.n_pass > 1) {  // multi-pass: carry the seven partial sums through global memory
            double* wsp = p.ws + (b * 7) * p.Kpad + k0 + r;
            if (p.pass > 0) {
                YC += wsp[0 * p.Kpad];
                YS += wsp[1 * p.Kpad];
                CC += wsp[2 * p.Kpad];
                CS += wsp[3 * p.Kpad];
                Saa += wsp[4 * p.Kpad];
                Sab += wsp[5 * p.Kpad];
                Sbb += wsp[6 * p.Kpad];
            }
            if (p.pass + 1 < p.n_pass) {
                wsp[0 * p.Kpad] = YC;
                wsp[1 * p.Kpad] = YS;
                wsp[2 * p.Kpad] = CC;
                wsp[3 * p.Kpad] = CS;
                wsp[4 * p.Kpad] = Saa;
                wsp[5 * p.Kpad] = Sab;
                wsp[6 * p.Kpad] = Sbb;
            }
        }
        const double SS = info.W - CC;  // <sin^2> = <1> - <cos^2>
        const double Scc = CC - Saa, Scs = CS - Sab, Sss = SS - Sbb;
        double z = 0.0, ys = YS, piv2 = Sss;
        if (Scc > kTauTrial * CC) {  // S6: otherwise the cos column is in the span of the base
            const double q = Scs / Scc;
            z = YC * YC / Scc;
            ys = fma(-q, YC, YS);
            piv2 = fma(-q, Scs, Sss);
        }
        if (piv2 > kTauTrial * SS) z = fma(ys, ys / piv2, z);
        zr[r] = z;
    }
    if (p.pass + 1 < p.n_pass) return;

    // ---- a10: store -----------------------------------------------------------------------
    if (k0 + R <= K && (reinterpret_cast<uintptr_t>(zp) & 15) == 0 && R % 2 == 0) {
#pragma unroll
        for (int r = 0; r < R; r += 2) reinterpret_cast<double2*>(zp)[r / 2] = make_double2(zr[r], zr[r + 1]);
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (k0 + r < K) zp[r] = zr[r];
    }
}

template <int R, int NB>
cudaError_t launch_one(const ScanParams& p, int64_t B, cudaStream_t stream)
{
    const size_t smem = scan_smem_bytes(R, NB, p);
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(scan_kernel<R, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             200 * 1024);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const int64_t runs = (p.K + R - 1) / R;
    const int64_t per_cta = (int64_t)p.FW * 32;
    dim3 grid((unsigned)((runs + per_cta - 1) / per_cta), (unsigned)B);
    scan_kernel<R, NB><<<grid, p.FW * p.S * 32, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace

size_t scan_smem_bytes(int R, int NB, const ScanParams& p)
{
    const size_t tiles = 2 * (size_t)p.TI * rec_stride(NB) * 8;
    const size_t seeds = (size_t)p.FW * 32 * (p.TI + 1) * 16;
    const size_t red = p.S > 1 ? (size_t)R * (4 + 2 * NB) * p.FW * 32 * 8 : 0;
    return (tiles > red ? tiles : red) + seeds;
}

#ifdef FREDEC_SCAN_ONLY_R  // experiments: build a single instantiation
#define FREDEC_SCAN_CONFIGS(X) X(FREDEC_SCAN_ONLY_R, FREDEC_SCAN_ONLY_NB)
#else
#define FREDEC_SCAN_CONFIGS(X) \
    X(8, 0) X(8, 1) X(8, 2) X(8, 3) X(4, 4) X(4, 5) X(4, 6) X(4, 7) X(4, 8) X(4, 9)
#endif

int scan_max_warps() { return kMaxScanThreads / 32; }

bool scan_config_supported(int R, int NB)
{
#define X(r, nb) \
    if (R == r && NB == nb) return true;
    FREDEC_SCAN_CONFIGS(X)
#undef X
    return false;
}

cudaError_t launch_scan(int R, int NB, const ScanParams& p, int64_t B, cudaStream_t stream)
{
#define X(r, nb) \
    if (R == r && NB == nb) return launch_one<r, nb>(p, B, stream);
    FREDEC_SCAN_CONFIGS(X)
#undef X
    return cudaErrorInvalidValue;
}

}  // namespace fredec
