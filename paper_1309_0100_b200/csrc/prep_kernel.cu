// prep_kernel.cu -- steps a1-a3 of the scan: validate, centre, orthogonalise the base
// model (prep_kernel, one thread-block cluster per series), per-observation table and seed
// records (table_kernel).  Once per scan.
//
// Generalises the normalisations of PAPER.md:193-197 (eq. 18: <1> = 1, <x> = 0, ...) to an
// arbitrary linear base model: the base functions are replaced by functions psi_j that are
// orthonormal under <.>, and x by its residual after the base fit.  Then the (d+2)x(d+2)
// system of PAPER.md:165-175 (eqs. 15, 16; Cholesky solve) has an identity leading block and
// collapses to the 2x2 Schur complement the scan kernel solves per frequency.
//
// Orthogonalisation = Cholesky QR applied twice.  One pass: the whole weighted Gram matrix of
// (phi_0 .. phi_{d-1}, x) in ONE sweep over the observations (register tiles of 4 x 4 entries per
// warp), Cholesky G = L L^T in shared memory with x carried as the last row (that row
// becomes a = L^{-1} g; one barrier and one reciprocal square root per column), then psi = L^{-1} phi
// and x' = x - sum_j a_j psi_j by one forward substitution per observation.  The first pass leaves an orthogonality error of eps x cond(G); the
// second pass, on the already nearly orthonormal functions, removes it ("twice is enough").  This
// is O(1) sweeps over the data where Gram-Schmidt needs O(d^2) dependent reductions.
//
// A series is shared by the C CTAs of a thread-block cluster (about 1000 observations per CTA, C <= 8;
// C = 1 when there are many series): each CTA owns a contiguous slice of the observations, the partial Gram matrices (and the scalars of a1)
// are added over the cluster through distributed shared memory in rank order, and every CTA then
// factors the same matrix.  All orders are fixed: results are bitwise reproducible.
#include <cstdio>
#include <cooperative_groups.h>

#include "prep_kernel.cuh"

namespace cg = cooperative_groups;

namespace fredec {

namespace {

constexpr int kPrepThreads = 512;  // at most (one long series); 256 when there are many series
constexpr int kPrepWarps = kPrepThreads / 32;
constexpr int kPrepMaxCluster = 8;
constexpr int kGramTile = 4;       // a warp accumulates a 4 x 4 block of Gram entries
constexpr int kGramMinSplit = 64;  // observations per warp at least, when a tile's sweep is split between warps
constexpr int kPrepSliceTarget = 1024;  // observations per CTA aimed at when one series is spread over a cluster

// Shared-memory layout of the prep kernel (doubles), M = d + 1 columns (the base functions and x).
// `stage` holds the CTA's slice of (w, phi_0 .. phi_{d-1}, x), d + 2 rows of `slice` observations, when it
// fits: every pass then runs at shared-memory latency and global memory is read and written once.
struct PrepSmem {
    int M, LD, tiles, splits;
    int64_t slice;  // observations per staged row (0: not staged, the passes run on global memory)
    size_t part, gram, chol, fact, diag0, scal, stage, total;  // offsets in doubles; total in bytes
};
__host__ __device__ inline PrepSmem prep_smem(int d, int splits, int64_t slice)
{
    PrepSmem L;
    L.M = d + 1;
    L.LD = L.M | 1;  // odd leading dimension: rows fall on different banks
    const int tm = (L.M + kGramTile - 1) / kGramTile;
    L.tiles = tm * (tm + 1) / 2;
    L.splits = splits;
    L.slice = slice;
    size_t o = 0;
    L.part = o;  o += (size_t)splits * L.tiles * 16;   // per (split, tile): a 4 x 4 block
    L.gram = o;  o += (size_t)L.M * L.LD;              // this CTA's partial Gram matrix (read by the cluster)
    L.chol = o;  o += (size_t)L.M * L.LD;              // the cluster's Gram matrix, eliminated in place
    L.fact = o;  o += (size_t)L.M * L.LD;              // its Cholesky factor (row d: a = L^{-1} g)
    L.diag0 = o; o += 2 * L.M;                         // original diagonal, then 1 / L[j][j]
    L.scal = o;  o += 16 + 4 * kPrepWarps;
    L.stage = o; o += (size_t)(d + 2) * slice;
    L.total = o * sizeof(double);
    return L;
}

// Fixed-order block reductions, results broadcast to all threads: v[0], v[1] are summed, v[2], v[3]
// minimised.  `red` = 4 * kPrepWarps doubles of smem.  One barrier pair for the four of them.
__device__ void block_reduce4(double v[4], double* red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        v[0] += __shfl_xor_sync(0xffffffffu, v[0], o);
        v[1] += __shfl_xor_sync(0xffffffffu, v[1], o);
        v[2] = fmin(v[2], __shfl_xor_sync(0xffffffffu, v[2], o));
        v[3] = fmin(v[3], __shfl_xor_sync(0xffffffffu, v[3], o));
    }
    __syncthreads();  // protect `red` from the previous call's readers
    if (lane == 0)
        for (int k = 0; k < 4; ++k) red[k * kPrepWarps + wid] = v[k];
    __syncthreads();
    v[0] = v[1] = 0.0;
    v[2] = v[3] = INFINITY;
    for (int q = 0; q < (int)(blockDim.x >> 5); ++q) {  // warp order: the same sum in every thread
        v[0] += red[q];
        v[1] += red[kPrepWarps + q];
        v[2] = fmin(v[2], red[2 * kPrepWarps + q]);
        v[3] = fmin(v[3], red[3 * kPrepWarps + q]);
    }
}

// The CTA's view of its slice: rows (w, columns 0 .. d-1, x) with a common stride, in shared memory
// (staged) or in global memory (then the columns are read from `src`, written to the psi workspace).
struct Rows {
    const double* w;
    double* col;        // column j of observation i: col[j * stride + i]
    double* x;
    int64_t stride, n;  // n observations, i = 0 .. n-1
};

// Partial Gram matrix of the columns (col_0 .. col_{d-1}, x) over the slice:
// gram[a][b] (a >= b within the tiles of the lower block triangle) = sum_i w_i col_a(i) col_b(i).
// Work item = (tile, split); a warp sweeps its share of the slice with the lanes striding over the
// observations and adds the 16 entries over the lanes; the splits are added in fixed order.
__device__ void gram_partial(const PrepSmem& L, double* sm, const Rows& R, int d)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int M = L.M;
    double* part = sm + L.part;
    const int64_t per = (R.n + L.splits - 1) / L.splits;
    for (int item = wid; item < L.tiles * L.splits; item += (blockDim.x >> 5)) {
        const int tile = item % L.tiles, split = item / L.tiles;
        int ta = 0;
        while ((ta + 1) * (ta + 2) / 2 <= tile) ++ta;  // tile = ta (ta + 1) / 2 + tb, tb <= ta
        const int tb = tile - ta * (ta + 1) / 2;
        const double* pa[kGramTile];
        const double* pb[kGramTile];
#pragma unroll
        for (int j = 0; j < kGramTile; ++j) {
            const int ca = ta * kGramTile + j, cb = tb * kGramTile + j;
            // columns past x are padding: they read x and are not stored
            pa[j] = ca < d ? R.col + (int64_t)ca * R.stride : R.x;
            pb[j] = cb < d ? R.col + (int64_t)cb * R.stride : R.x;
        }
        double acc[kGramTile][kGramTile];
#pragma unroll
        for (int j = 0; j < kGramTile; ++j)
#pragma unroll
            for (int k = 0; k < kGramTile; ++k) acc[j][k] = 0.0;
        const int64_t s0 = split * per, s1 = min(R.n, s0 + per);
#pragma unroll 2
        for (int64_t i = s0 + lane; i < s1; i += 32) {
            const double wi = R.w[i];
            double va[kGramTile], vb[kGramTile];
#pragma unroll
            for (int j = 0; j < kGramTile; ++j) {
                va[j] = wi * pa[j][i];
                vb[j] = pb[j][i];
            }
#pragma unroll
            for (int j = 0; j < kGramTile; ++j)
#pragma unroll
                for (int k = 0; k < kGramTile; ++k) acc[j][k] = fma(va[j], vb[k], acc[j][k]);
        }
#pragma unroll
        for (int j = 0; j < kGramTile; ++j)
#pragma unroll
            for (int k = 0; k < kGramTile; ++k) {
                double v = acc[j][k];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                if (lane == 0) part[((size_t)split * L.tiles + tile) * 16 + j * kGramTile + k] = v;
            }
    }
    __syncthreads();
    double* gram = sm + L.gram;
    for (int e = threadIdx.x; e < L.tiles * 16; e += blockDim.x) {
        const int tile = e / 16, j = (e % 16) / kGramTile, k = e % kGramTile;
        int ta = 0;
        while ((ta + 1) * (ta + 2) / 2 <= tile) ++ta;
        const int tb = tile - ta * (ta + 1) / 2;
        const int a = ta * kGramTile + j, b = tb * kGramTile + k;
        if (a < M && b <= a) {
            double v = 0.0;
            for (int sp = 0; sp < L.splits; ++sp) v += part[((size_t)sp * L.tiles + tile) * 16 + j * kGramTile + k];
            gram[a * L.LD + b] = v;
        }
    }
}

__device__ __forceinline__ void cluster_or_cta_sync(cg::cluster_group& cluster, int C)
{
    if (C > 1)
        cluster.sync();
    else
        __syncthreads();
}

// chol = sum over the cluster's CTAs, in rank order, of their partial Gram matrices (lower triangles).
__device__ void gram_cluster_sum(const PrepSmem& L, double* sm, cg::cluster_group& cluster, int C)
{
    cluster_or_cta_sync(cluster, C);  // every CTA's partial matrix is written
    const int M = L.M;
    double* chol = sm + L.chol;
    for (int e = threadIdx.x; e < M * M; e += blockDim.x) {
        const int a = e / M, b = e % M;
        if (b > a) continue;
        double v = 0.0;
        for (int r = 0; r < C; ++r) v += cluster.map_shared_rank(sm + L.gram, r)[a * L.LD + b];
        chol[a * L.LD + b] = v;
        if (a == b) sm[L.diag0 + a] = v;
    }
    cluster_or_cta_sync(cluster, C);  // all remote reads done before anyone overwrites its partial matrix
}

// Cholesky of the leading d x d block of chol (lower triangle) with row d (the column x) carried along as
// a right-hand side.  chol is eliminated in place with UNSCALED columns (so a column is only
// read while its trailing block is updated: one barrier per column); the factor goes to fact:
// fact[i][j] = L[i][j], fact[d][j] = a_j = (L^{-1} g)_j, and dinv[j] = 1 / L[j][j].  Returns false when a
// pivot <= tau x its original diagonal (dependent base functions, S6b).
__device__ bool chol_with_x(const PrepSmem& L, double* sm, int d, double tau, int* flag)
{
    double* S = sm + L.chol;
    double* F = sm + L.fact;
    const double* diag0 = sm + L.diag0;
    double* dinv = sm + L.diag0 + L.M;
    const int LD = L.LD, tid = threadIdx.x;
    if (tid == 0) *flag = 0;
    __syncthreads();
    for (int j = 0; j < d; ++j) {
        const double piv = S[j * LD + j];
        if (!(piv > tau * diag0[j])) {  // uniform across the CTA
            if (tid == 0) *flag = 1;
            break;
        }
        const double inv = rsqrt(piv), ljj = piv * inv, inv2 = inv * inv;  // one reciprocal square root per column
        for (int i = j + tid; i <= d; i += blockDim.x) F[i * LD + j] = i == j ? ljj : S[i * LD + j] * inv;
        if (tid == 0) dinv[j] = inv;
        const int rows = d - j;  // rows j+1 .. d, columns j+1 .. min(row, d-1)
        for (int e = tid; e < rows * rows; e += blockDim.x) {
            const int i = j + 1 + e / rows, k = j + 1 + e % rows;
            if (k <= i && k < d) S[i * LD + k] = fma(-(S[i * LD + j] * inv2), S[k * LD + j], S[i * LD + k]);
        }
        __syncthreads();
    }
    __syncthreads();
    return *flag == 0;
}

// psi_j(i) = (phi_j(i) - sum_{m<j} L[j][m] psi_m(i)) / L[j][j],  x'(i) = x(i) - sum_j a_j psi_j(i), one
// thread per observation of the slice; `src` columns (stride src_stride) are read, R.col / R.x written
// (they may be the same memory: a thread touches its own observation only, and reads back its own writes).
// The inner sums run on two accumulators with 32-bit offsets: the chain per observation is d sums long,
// not d^2 / 2 terms.
__device__ void apply_factor(const PrepSmem& L, double* sm, int d, const double* src, int64_t src_stride,
                             const double* xsrc, const Rows& R)
{
    const double* F = sm + L.fact;
    const double* dinv = sm + L.diag0 + L.M;
    const int LD = L.LD, n = (int)R.n;
    const bool narrow = R.stride * (int64_t)d < (int64_t)1 << 30;  // offsets fit 32 bits (always, when staged)
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        double xv = xsrc[i];
        double* out = R.col + i;
        for (int j = 0; j < d; ++j) {
            const double* row = F + j * LD;
            double s0 = 0.0, s1 = 0.0;
            if (narrow) {
                const int st = (int)R.stride;
                int m = 0;
                for (; m + 1 < j; m += 2) {
                    s0 = fma(row[m], out[m * st], s0);
                    s1 = fma(row[m + 1], out[(m + 1) * st], s1);
                }
                if (m < j) s0 = fma(row[m], out[m * st], s0);
            } else {
                for (int m = 0; m < j; ++m) s0 = fma(row[m], out[(int64_t)m * R.stride], s0);
            }
            const double v = (src[(int64_t)j * src_stride + i] - (s0 + s1)) * dinv[j];
            out[(int64_t)j * R.stride] = v;
            xv = fma(-F[d * LD + j], v, xv);
        }
        R.x[i] = xv;
    }
    __syncthreads();
}

// STAGED: the slice lives in shared memory (the pointers of `Rows` then derive from `sm` alone, so that the
// compiler addresses them as shared memory instead of through generic loads).
template <bool STAGED>
__global__ void __launch_bounds__(kPrepThreads) prep_kernel(PrepParams p, int splits, int64_t slice)
{
    extern __shared__ __align__(16) double sm[];
    __shared__ int flag;
    cg::cluster_group cluster = cg::this_cluster();
    const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
    const int64_t b = blockIdx.y, N = p.N;
    const int d = p.d;
    const PrepSmem L = prep_smem(d, splits, slice);
    const int64_t i0 = N * rank / C, i1 = N * (rank + 1) / C;  // this CTA's observations
    const double* t = p.t + b * N + i0;
    const double* x = p.x + b * N + i0;
    const double* w = p.w + b * N + i0;
    const double* base = p.base ? p.base + b * (int64_t)d * N + i0 : nullptr;
    double* psi = p.psi + b * (int64_t)d * N + i0;  // [d][N]
    double* xt = p.xt + b * N + i0;                 // [N]
    SeriesInfo* info = p.info + b;
    double* scal = sm + L.scal;
    double* red = scal + 16;
    constexpr bool staged = STAGED;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    Rows R;
    R.n = i1 - i0;
    if constexpr (STAGED) {
        R.stride = slice;
        R.w = sm + L.stage;
        R.col = sm + L.stage + slice;
        R.x = sm + L.stage + (d + 1) * slice;
    } else {
        R.stride = N;
        R.w = w;
        R.col = psi;
        R.x = xt;
    }

#ifdef FREDEC_EXP_PREP_TRACE  // measurement build: cycles per phase of CTA 0, printed at the end
    long long tr[16];
    int ntr = 0;
#define FREDEC_TR()             \
    do {                        \
        __syncthreads();        \
        tr[ntr++] = clock64();  \
    } while (0)
#else
#define FREDEC_TR() \
    do {            \
    } while (0)
#endif
    FREDEC_TR();
    // ---- a1: validate, W = <1>, time origin; the slice goes to shared memory when it fits -----------
    double bad = 0.0, wsum = 0.0, tmin = INFINITY, tmax = -INFINITY;
    for (int64_t i = threadIdx.x; i < R.n; i += blockDim.x) {
        const double ti = t[i], xi = x[i], wi = w[i];
        if (!isfinite(ti) || !isfinite(xi) || !isfinite(wi) || wi < 0.0) bad = 1.0;
        wsum += wi;
        tmin = fmin(tmin, ti);
        tmax = fmax(tmax, ti);
        if (staged) {
            sm[L.stage + i] = wi;
            R.x[i] = xi;
        }
    }
    // the base functions: a warp per row, the lanes along it (independent coalesced loads)
    for (int j = wid; j < d; j += (blockDim.x >> 5)) {
        const double* src = base + (int64_t)j * N;
        double* dst = staged ? R.col + (int64_t)j * slice : nullptr;
        for (int64_t i = lane; i < R.n; i += 32) {
            const double v = src[i];
            if (!isfinite(v)) bad = 1.0;
            if (staged) dst[i] = v;
        }
    }
    FREDEC_TR();
    {
        double v4[4] = {bad, wsum, tmin, -tmax};
        block_reduce4(v4, red);
        if (threadIdx.x == 0) {
            scal[0] = v4[0];
            scal[1] = v4[1];
            scal[2] = v4[2];
            scal[3] = -v4[3];
        }
    }
    cluster_or_cta_sync(cluster, C);
    double W = 0.0;
    bad = 0.0;
    tmin = INFINITY;
    tmax = -INFINITY;
    for (int r = 0; r < C; ++r) {  // rank order: every CTA gets the same W
        const double* rs = cluster.map_shared_rank(scal, r);
        bad += rs[0];
        W += rs[1];
        tmin = fmin(tmin, rs[2]);
        tmax = fmax(tmax, rs[3]);
    }
    FREDEC_TR();
    int status = 0;
    if (bad != 0.0 || !(W > 0.0) || !isfinite(W)) status = -2;  // FREDEC_EDATA
    const double t_mid = 0.5 * (tmin + tmax);

    // ---- a2: orthonormal base psi and residual x~ by two passes of Cholesky QR ----------------
    // (with invalid data the passes run on whatever is there and the results are ignored: no CTA may
    // leave the cluster's barriers)
    for (int pass = 0; pass < 2; ++pass) {
        // not staged: the first pass reads the caller's base functions and x, and writes the workspace
        Rows G = R;
        if constexpr (!STAGED) {
            if (pass == 0) {
                G.col = const_cast<double*>(base);
                G.x = const_cast<double*>(x);
            }
        }
        gram_partial(L, sm, G, d);
        FREDEC_TR();
        gram_cluster_sum(L, sm, cluster, C);
        FREDEC_TR();
        // pass 0 decides whether the base functions are dependent (S6b); pass 1 factors a matrix
        // that is the identity up to the first pass's orthogonality error
        const bool ok = chol_with_x(L, sm, d, pass == 0 ? kTauBase : 0.0, &flag);
        if (!ok && status == 0) status = -3;  // FREDEC_ESINGULAR (the same decision in every CTA)
        FREDEC_TR();
        if (ok) apply_factor(L, sm, d, G.col, G.stride, G.x, R);
        FREDEC_TR();
    }
    double chi2 = 0.0;
    for (int64_t i = threadIdx.x; i < R.n; i += blockDim.x) chi2 = fma(R.w[i] * R.x[i], R.x[i], chi2);
    {
        double v4[4] = {chi2, 0.0, 0.0, 0.0};
        block_reduce4(v4, red);
        if (threadIdx.x == 0) scal[4] = v4[0];
    }
    if (staged) {  // results to the workspace: whole rows, coalesced
        for (int j = wid; j < d; j += (blockDim.x >> 5)) {
            const double* src = R.col + (int64_t)j * slice;
            double* dst = psi + (int64_t)j * N;
            for (int64_t i = lane; i < R.n; i += 32) dst[i] = src[i];
        }
        for (int64_t i = threadIdx.x; i < R.n; i += blockDim.x) xt[i] = R.x[i];
    }
    cluster_or_cta_sync(cluster, C);
    if (rank == 0 && threadIdx.x == 0) {
        double total = 0.0;
        for (int r = 0; r < C; ++r) total += cluster.map_shared_rank(scal, r)[4];
        info->W = W;
        info->chi2_base = status == 0 ? total : 0.0;
        info->t_mid = t_mid;
        info->status = status;
        info->pad = 0;
    }
    cluster_or_cta_sync(cluster, C);  // no CTA exits while its shared memory may still be read
#ifdef FREDEC_EXP_PREP_TRACE
    FREDEC_TR();
    if (threadIdx.x == 0 && blockIdx.x == 0 && blockIdx.y == 0) {
        printf("prep trace N=%lld d=%d C=%d (load, reduce, [gram, sum, chol, apply] x 2, rest):", (long long)N, d, C);
        for (int i = 1; i < ntr; ++i) printf(" %lld", tr[i] - tr[i - 1]);
        printf(" total %lld\n", tr[ntr - 1] - tr[0]);
    }
#endif
}

// ---- a2, incremental form (the base model of the next SLICK iteration is the current one plus
// one sinusoid) -------------------------------------------------------------------------------
// psi_0 .. psi_{d0-1} are orthonormal and x~ is the residual of x after them (the previous prep / append).
// The two new base functions cos / sin(2 pi f t) are orthogonalised against them by two rounds of projection
// ("twice is enough"), then against each other and normalised (a 2 x 2 Cholesky step), appended
// as rows d0 and d0 + 1 of psi, and x~ and chi2_base are updated: O(N d) instead of the O(N d^2) of a prep from
// scratch.  One CTA (the driver's series is a single one), fixed-order sums.
constexpr int kAppendThreads = 512;
constexpr int kAppendWarps = kAppendThreads / 32;

// NV fixed-order block sums at once (one barrier pair): `red` = NV * kAppendWarps doubles.
template <int NV>
__device__ void append_block_sum(double (&v)[NV], double* red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int k = 0; k < NV; ++k) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
    __syncthreads();
    if (lane == 0)
#pragma unroll
        for (int k = 0; k < NV; ++k) red[k * kAppendWarps + wid] = v[k];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double r = 0.0;
        for (int q = 0; q < kAppendWarps; ++q) r += red[k * kAppendWarps + q];
        v[k] = r;
    }
}

__global__ void __launch_bounds__(kAppendThreads) prep_append_kernel(PrepAppendParams p)
{
    extern __shared__ __align__(16) double coef[];  // [2][d0]
    __shared__ double red[5 * kAppendWarps];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t N = p.N;
    const int d0 = p.d0;
    double* pa = p.psi + (int64_t)d0 * N;  // the two new rows, worked on in place
    double* pb = pa + N;
    SeriesInfo* info = p.info;
    if (info->status != 0) return;  // uniform: the series already failed
    const double f = *p.freq;
    // the new functions (phase reduced exactly, as the base builder of the from-scratch path does)
    double n0a = 0.0, n0b = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += kAppendThreads) {
        double sv, cv;
        sincospi(2.0 * frac_prod(f, p.t[i]), &sv, &cv);
        pa[i] = cv;
        pb[i] = sv;
        const double wi = p.w[i];
        n0a = fma(wi * cv, cv, n0a);
        n0b = fma(wi * sv, sv, n0b);
    }
    {
        double v[2] = {n0a, n0b};
        append_block_sum(v, red);
        n0a = v[0];
        n0b = v[1];
    }
    for (int round = 0; round < 2; ++round) {
        __syncthreads();
        for (int j = wid; j < d0; j += kAppendWarps) {
            const double* pj = p.psi + (int64_t)j * N;
            double c = 0.0, e = 0.0, c1 = 0.0, e1 = 0.0;
            int64_t i = lane;
            for (; i + 96 < N; i += 128) {  // four independent loads of each array in flight
                const double w0 = p.w[i] * pj[i], w1 = p.w[i + 32] * pj[i + 32];
                const double w2 = p.w[i + 64] * pj[i + 64], w3 = p.w[i + 96] * pj[i + 96];
                c = fma(w0, pa[i], c);
                e = fma(w0, pb[i], e);
                c1 = fma(w1, pa[i + 32], c1);
                e1 = fma(w1, pb[i + 32], e1);
                c = fma(w2, pa[i + 64], c);
                e = fma(w2, pb[i + 64], e);
                c1 = fma(w3, pa[i + 96], c1);
                e1 = fma(w3, pb[i + 96], e1);
            }
            for (; i < N; i += 32) {
                const double wp = p.w[i] * pj[i];
                c = fma(wp, pa[i], c);
                e = fma(wp, pb[i], e);
            }
            c += c1;
            e += e1;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                c += __shfl_xor_sync(0xffffffffu, c, o);
                e += __shfl_xor_sync(0xffffffffu, e, o);
            }
            if (lane == 0) {
                coef[j] = c;
                coef[d0 + j] = e;
            }
        }
        __syncthreads();
        for (int64_t i = threadIdx.x; i < N; i += kAppendThreads) {
            double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
            int j = 0;
            for (; j + 1 < d0; j += 2) {
                const double v0 = p.psi[(int64_t)j * N + i], v1 = p.psi[(int64_t)(j + 1) * N + i];
                a0 = fma(coef[j], v0, a0);
                a1 = fma(coef[j + 1], v1, a1);
                b0 = fma(coef[d0 + j], v0, b0);
                b1 = fma(coef[d0 + j + 1], v1, b1);
            }
            if (j < d0) {
                const double v0 = p.psi[(int64_t)j * N + i];
                a0 = fma(coef[j], v0, a0);
                b0 = fma(coef[d0 + j], v0, b0);
            }
            pa[i] -= a0 + a1;
            pb[i] -= b0 + b1;
        }
    }
    __syncthreads();
    // the 2 x 2 step: Gram of (phi_a, phi_b) with x~ carried as the right-hand side
    double naa = 0.0, nab = 0.0, nbb = 0.0, xa = 0.0, xb = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += kAppendThreads) {
        const double wi = p.w[i], a = pa[i], b = pb[i], xw = wi * p.xt[i];
        naa = fma(wi * a, a, naa);
        nab = fma(wi * a, b, nab);
        nbb = fma(wi * b, b, nbb);
        xa = fma(xw, a, xa);
        xb = fma(xw, b, xb);
    }
    {
        double v[5] = {naa, nab, nbb, xa, xb};
        append_block_sum(v, red);
        naa = v[0]; nab = v[1]; nbb = v[2]; xa = v[3]; xb = v[4];
    }
    int status = 0;
    double ra = 0.0, rb = 0.0, q = 0.0;
    if (naa > kTauBase * n0a) {  // else: the cosine is in the span of the base (S6b)
        ra = rsqrt(naa);
        q = nab * ra;
    } else {
        status = -3;
    }
    const double nbb2 = nbb - q * q;
    if (status == 0 && nbb2 > kTauBase * n0b)
        rb = rsqrt(nbb2);
    else
        status = -3;
    const double aa = xa * ra, ab = (xb - q * aa) * rb;
    double chi2 = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += kAppendThreads) {
        const double va = pa[i] * ra, vb = (pb[i] - q * va) * rb;
        pa[i] = va;
        pb[i] = vb;
        const double xv = p.xt[i] - fma(aa, va, ab * vb);
        p.xt[i] = xv;
        chi2 = fma(p.w[i] * xv, xv, chi2);
    }
    {
        double v[1] = {chi2};
        append_block_sum(v, red);
        chi2 = v[0];
    }
    if (threadIdx.x == 0) {
        info->chi2_base = status == 0 ? chi2 : 0.0;
        info->status = status;
    }
}

// ---- a3: per-observation table and seed records --------------------------
// One thread per (observation, pair of column tiles tp, position hh in a tile): two grid offsets h and h + 4,
// four sincospi of exactly reduced phases, and the entries of every family for them.  The series are
// padded to whole groups of 4 observations with zero multipliers.  Layout: scan_mma_kernel.cuh.
constexpr int kTableObs = 32;  // observations per CTA (threadIdx.x); threadIdx.y = tp * 4 + hh

__global__ void table_kernel(TableParams p)
{
    const int64_t b = blockIdx.z, N = p.N;
    const int pass = blockIdx.y;
    const SeriesInfo info = p.info[b];
    if (info.status != 0) return;
    const int64_t i = (int64_t)blockIdx.x * kTableObs + threadIdx.x;
    if (i >= p.G4 * 4) return;
    const bool real = i < N;
    const int H = p.H, NT = mma_nt(H), NF = mma_nf(p.NB);
    const int tp = threadIdx.y >> 2, hh = threadIdx.y & 3;
    const double tc = real ? p.t[b * N + i] - info.t_mid : 0.0;
    const double wi = real ? p.w[b * N + i] : 0.0;
    if (pass == 0 && threadIdx.y == 0) {
        SeedRec r;
        r.t = tc;
        sincospi(2.0 * frac_prod(p.df * (double)(16 * H), tc), &r.su, &r.cu);  // one unit = 8 runs of 2H steps
        r.tcu = 2.0 * r.cu;
        sincospi(2.0 * frac_prod(p.df * (double)(8 * H), tc), &r.s4, &r.c4);  // four runs
        p.srec[b * p.G4 * 4 + i] = r;
    }
    double* grp = p.tab + ((b * p.n_pass + pass) * p.G4 + i / 4) * mma_group_doubles(H, p.NB);
    const int k = (int)(i & 3);
    const double* psi = p.psi + b * (int64_t)p.d * N;
    // column tiles are stored in pairs (one 16-byte load per lane fetches the fragments of two): the
    // thread writes the entries of tiles 2 tp and 2 tp + 1, i.e. of h and h + 4, as one double2
    double c1[2], s1[2], c2[2], s2[2];
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const int h = 8 * tp + 4 * e + hh + 1;
        // alpha_h = 2 pi (h - 1/2) df t' in turns, range-reduced exactly
        const double x = frac_prod((double)(2 * h - 1) * (0.5 * p.df), tc);
        sincospi(2.0 * x, &s1[e], &c1[e]);
        sincospi(4.0 * x, &s2[e], &c2[e]);
    }
    const int n0 = 2 * hh;
    for (int f = 0; f < NF; ++f) {
        double m;
        const bool dbl = f == NF - 1;  // the w family uses the doubled angles
        if (f == 0) {
            m = (pass == 0 && real) ? wi * p.xt[b * N + i] : 0.0;
        } else if (dbl) {
            m = pass == 0 ? 0.5 * wi : 0.0;
        } else {
            const int j = pass * p.NB + (f - 1);
            m = (j < p.d && real) ? wi * psi[(int64_t)j * N + i] : 0.0;
        }
        double2* tile = reinterpret_cast<double2*>(grp + (f * (NT / 2) + tp) * 64);
        tile[n0 * 4 + k] = make_double2(m * (dbl ? c2[0] : c1[0]), m * (dbl ? c2[1] : c1[1]));
        tile[(n0 + 1) * 4 + k] = make_double2(m * (dbl ? s2[0] : s1[0]), m * (dbl ? s2[1] : s1[1]));
    }
}

}  // namespace

cudaError_t launch_table(const TableParams& p, int64_t B, cudaStream_t stream)
{
    dim3 grid((unsigned)((p.G4 * 4 + kTableObs - 1) / kTableObs), (unsigned)p.n_pass, (unsigned)B);
    dim3 block(kTableObs, (unsigned)(mma_nt(p.H) / 2 * 4));  // at most 32 x 24 threads (H = 48)
    table_kernel<<<grid, block, 0, stream>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_prep_append(const PrepAppendParams& p, cudaStream_t stream)
{
    const size_t smem = (size_t)2 * (p.d0 > 0 ? p.d0 : 1) * sizeof(double);
    prep_append_kernel<<<1, kAppendThreads, smem, stream>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_prep(const PrepParams& p, int64_t B, cudaStream_t stream)
{
    // CTAs per series (a thread-block cluster, at most 8): as few as let the slice of (w, base, x) sit in
    // shared memory beside the matrices, one when there are many series
    constexpr size_t kSmemMax = 220 * 1024;
    const size_t fixed = prep_smem(p.d, kPrepWarps, 0).total;
    int C = 1;
    auto fits = [&](int c) { return fixed + (size_t)(p.d + 2) * ((p.N + c - 1) / c) * 8 <= kSmemMax; };
    if (B <= 64)
        while (C < kPrepMaxCluster && (!fits(C) || (p.N + C - 1) / C > kPrepSliceTarget)) C *= 2;
    const int64_t per_cta = (p.N + C - 1) / C;
    const int64_t slice = fits(C) ? per_cta : 0;
    const int threads = B <= 64 ? kPrepThreads : 256;  // many series: more CTAs per SM instead
    int splits = (threads / 32) / prep_smem(p.d, 1, 0).tiles;
    if (splits > (int)(per_cta / kGramMinSplit)) splits = (int)(per_cta / kGramMinSplit);
    if (splits < 1) splits = 1;
    const PrepSmem L = prep_smem(p.d, splits, slice);
    static size_t attr_smem[2] = {0, 0};
    const int st = slice > 0 ? 1 : 0;
    if (L.total > attr_smem[st]) {
        cudaError_t e = st ? cudaFuncSetAttribute(prep_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total)
                           : cudaFuncSetAttribute(prep_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.total);
        if (e != cudaSuccess) return e;
        attr_smem[st] = L.total;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)C, (unsigned)B, 1);
    cfg.blockDim = dim3(threads, 1, 1);
    cfg.dynamicSmemBytes = L.total;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return st ? cudaLaunchKernelEx(&cfg, prep_kernel<true>, p, splits, slice)
              : cudaLaunchKernelEx(&cfg, prep_kernel<false>, p, splits, slice);
}

}  // namespace fredec
