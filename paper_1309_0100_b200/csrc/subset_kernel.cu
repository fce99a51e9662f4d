// subset_kernel.cu -- see subset_kernel.cuh.
//
// The paper runs "many entirely independent instances of the fitting subroutine" whose arrays
// live in global memory.  Here the full Fisher matrix Q and gradient g of the pool
// are formed ONCE (every subset's Q is a sub-matrix of it: "low-top submatrix"), kept
// in shared memory, and the subsets are walked depth first, one warp per subtree: a subset's Cholesky
// factor is its parent's plus two rows, each found by one forward substitution in the
// warp's shared-memory workspace, and l drops by the squares of the two new entries of a = L^{-1} g.
// The warp stores L^{-1}, so that a new row is two matrix-vector products with independent lanes.
#include "subset_kernel.cuh"

namespace fredec {

namespace {

constexpr int kGramThreads = 256;
constexpr int kSubsetWarps = 8;

__global__ void __launch_bounds__(kGramThreads) gram_kernel(const double* __restrict__ basis,
                                                           const double* __restrict__ x,
                                                           const double* __restrict__ w, int64_t N, int M,
                                                           double* __restrict__ A)
{
    __shared__ double red[kGramThreads / 32];
    const int a = blockIdx.x, b = blockIdx.y;
    if (a > b) return;
    const double* pa = a < M ? basis + (int64_t)a * N : x;
    const double* pb = b < M ? basis + (int64_t)b * N : x;
    double acc = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += kGramThreads) acc = fma(w[i] * pa[i], pb[i], acc);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0;
        for (int k = 0; k < kGramThreads / 32; ++k) v += red[k];  // fixed order
        A[a * (M + 1) + b] = v;
        A[b * (M + 1) + a] = v;
    }
}

// Per-warp state of the depth-first walk over the subsets (all in shared memory).  The warp keeps
// the INVERSE of the Cholesky factor: a new row of L is then a matrix-vector product, y = L^{-1} q,
// every lane summing its own entry with no dependence on the others, where the forward
// substitution would be a chain of i dependent steps.
struct WalkState {
    double* Li;    // [M][M] rows of L^{-1} of the current subset (row-major, odd leading dimension);
                   // an all-zero row marks a dropped function
    double* a;     // [M] a = L^{-1} g
    double2* v;    // [M] the two right-hand sides (cos, sin), then the two new rows of L
    int* ids;      // [M] model-function index of each row
};

// Appends the constant (function 0) as row 0; returns a_0^2.
__device__ __forceinline__ double push_constant(const WalkState& w, const double* __restrict__ A, int M, int lane)
{
    const double q00 = A[0];
    const double inv = q00 > 0.0 ? rsqrt(q00) : 0.0;
    const double a0 = A[M] * inv;  // column M of A holds g = <x phi>
    if (lane == 0) {
        w.Li[0] = inv;
        w.a[0] = a0;
        w.ids[0] = 0;
    }
    __syncwarp();
    return a0 * a0;
}

// Pushes frequency j: its cos and sin rows at positions i and i + 1 (i <= 49); returns the drop of
// l = the squares of the two new entries of a.
__device__ __forceinline__ double push_frequency(const WalkState& w, const double* __restrict__ A, int LDA, int M,
                                                 int i, int j, int lane)
{
    const int c = 2 * j + 1, sn = 2 * j + 2;
    const double* qc = A + c * LDA;
    const double* qs = A + sn * LDA;
    const int k0 = lane, k1 = lane + 32;
    const bool in0 = k0 < i, in1 = k1 < i;
    if (in0) {
        const int id = w.ids[k0];
        w.v[k0] = make_double2(qc[id], qs[id]);
    }
    if (in1) {
        const int id = w.ids[k1];
        w.v[k1] = make_double2(qc[id], qs[id]);
    }
    __syncwarp();
    // rows of L: y = L^{-1} q  (lane k: sum over q <= k)
    double c0 = 0.0, s0 = 0.0, c1 = 0.0, s1 = 0.0;
    if (in0) {
        const double* row = w.Li + k0 * M;
#pragma unroll 4
        for (int q = 0; q <= k0; ++q) {
            const double li = row[q];
            const double2 r = w.v[q];
            c0 = fma(li, r.x, c0);
            s0 = fma(li, r.y, s0);
        }
    }
    if (in1) {
        const double* row = w.Li + k1 * M;
#pragma unroll 4
        for (int q = 0; q <= k1; ++q) {
            const double li = row[q];
            const double2 r = w.v[q];
            c1 = fma(li, r.x, c1);
            s1 = fma(li, r.y, s1);
        }
    }
    double cc = 0.0, ca = 0.0, sc = 0.0, ss = 0.0, sa = 0.0;
    if (in0) {
        const double a0 = w.a[k0];
        cc = c0 * c0; ca = c0 * a0; sc = s0 * c0; ss = s0 * s0; sa = s0 * a0;
    }
    if (in1) {
        const double a1 = w.a[k1];
        cc = fma(c1, c1, cc); ca = fma(c1, a1, ca); sc = fma(s1, c1, sc); ss = fma(s1, s1, ss); sa = fma(s1, a1, sa);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        cc += __shfl_xor_sync(0xffffffffu, cc, o);
        ca += __shfl_xor_sync(0xffffffffu, ca, o);
        sc += __shfl_xor_sync(0xffffffffu, sc, o);
        ss += __shfl_xor_sync(0xffffffffu, ss, o);
        sa += __shfl_xor_sync(0xffffffffu, sa, o);
    }
    // pivots and entries of a; a function that the earlier ones span is dropped (rule S6)
    const double qcc = qc[c], qss = qs[sn];
    const double pc = qcc - cc;
    double invc = 0.0, ac = 0.0;
    if (pc > kTauTrial * qcc) {
        invc = rsqrt(pc);
        ac = (qc[M] - ca) * invc;
    }
    const double ysc = (qs[c] - sc) * invc;  // the sin row's entry in the cos column
    const double ps = qss - fma(ysc, ysc, ss);
    double invs = 0.0, as = 0.0;
    if (ps > kTauTrial * qss) {
        invs = rsqrt(ps);
        as = (qs[M] - fma(ysc, ac, sa)) * invs;
    }
    // the two new rows of L^{-1}: -(1/d) y^T L^{-1} (lane q: sum over k >= q), diagonal 1/d
    __syncwarp();  // every lane has read the right-hand sides
    if (in0) w.v[k0] = make_double2(c0, s0);
    if (in1) w.v[k1] = make_double2(c1, s1);
    __syncwarp();
    if (in0) {
        double uc = 0.0, us = 0.0;
#pragma unroll 4
        for (int k = k0; k < i; ++k) {
            const double li = w.Li[k * M + k0];
            const double2 y = w.v[k];
            uc = fma(y.x, li, uc);
            us = fma(y.y, li, us);
        }
        const double rc = -invc * uc;
        w.Li[i * M + k0] = rc;
        w.Li[(i + 1) * M + k0] = -invs * fma(ysc, rc, us);
    }
    if (in1) {
        double uc = 0.0, us = 0.0;
#pragma unroll 4
        for (int k = k1; k < i; ++k) {
            const double li = w.Li[k * M + k1];
            const double2 y = w.v[k];
            uc = fma(y.x, li, uc);
            us = fma(y.y, li, us);
        }
        const double rc = -invc * uc;
        w.Li[i * M + k1] = rc;
        w.Li[(i + 1) * M + k1] = -invs * fma(ysc, rc, us);
    }
    if (lane == 0) {
        w.Li[i * M + i] = invc;
        w.Li[(i + 1) * M + i] = -invs * ysc * invc;
        w.Li[(i + 1) * M + i + 1] = invs;
        w.a[i] = ac;
        w.a[i + 1] = as;
        w.ids[i] = c;
        w.ids[i + 1] = sn;
    }
    __syncwarp();
    return fma(ac, ac, as * as);
}

// Subsets are walked depth first so that a subset's factor extends its parent's by two rows
// (the smaller Q is a leading block of the larger, and so is its Cholesky factor): one
// warp per task = one choice P of the first s frequencies, then all 2^(n-s) extensions of it.
__global__ void __launch_bounds__(kSubsetWarps * 32) subset_fit_kernel(const double* __restrict__ Aglob, int n, int s,
                                                                      double* __restrict__ l_out)
{
    extern __shared__ double sm[];
    const int M = 2 * n + 1, LDA = M + 1;
    double* A = sm;  // [LDA][LDA] augmented Gram matrix of the whole pool
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int per_warp = (M * M + 3 * M + (M + 1) / 2 + (n + 2) + (n + 1) / 2 + 3) & ~1;  // doubles, even
    double* base = sm + LDA * LDA + (size_t)wid * per_warp;
    WalkState w;
    w.v = reinterpret_cast<double2*>(base);                   // 16-byte aligned: per_warp and LDA^2 are even
    w.Li = base + 2 * M;
    w.a = w.Li + M * M;
    w.ids = reinterpret_cast<int*>(w.a + M);
    double* lstack = w.a + M + (M + 1) / 2;                   // [n + 2] l of the subsets on the walk's path
    int* cur = reinterpret_cast<int*>(lstack + n + 2);        // [n] frequency chosen at each depth
    for (int e = threadIdx.x; e < LDA * LDA; e += blockDim.x) A[e] = Aglob[e];
    __syncthreads();

    const int64_t tasks = (int64_t)1 << s;
    for (int64_t P = (int64_t)blockIdx.x * kSubsetWarps + wid; P < tasks; P += (int64_t)gridDim.x * kSubsetWarps) {
        // the constant, then the chosen ones of the first s frequencies
        double l = A[M * LDA + M] - push_constant(w, A, M, lane);  // D - a_0^2
        int pos = 1;
        for (int j = 0; j < s; ++j)
            if ((P >> j) & 1) {
                l -= push_frequency(w, A, LDA, M, pos, j, lane);
                pos += 2;
            }
        if (lane == 0) l_out[P] = fmax(l, 0.0);
        // depth-first over the extensions by frequencies s .. n-1
        int depth = 0, j = s;
        int64_t mask = P;
        double lcur = l;
        while (true) {
            if (j < n) {
                if (lane == 0) {
                    lstack[depth] = lcur;
                    cur[depth] = j;
                }
                lcur -= push_frequency(w, A, LDA, M, pos, j, lane);
                pos += 2;
                mask |= (int64_t)1 << j;
                if (lane == 0) l_out[mask] = fmax(lcur, 0.0);
                ++depth;
                ++j;
            } else {
                if (depth == 0) break;
                --depth;
                __syncwarp();
                j = cur[depth];
                lcur = lstack[depth];
                mask &= ~((int64_t)1 << j);
                pos -= 2;
                ++j;
            }
        }
        __syncwarp();
    }
}

}  // namespace

cudaError_t launch_gram(const double* basis, const double* x, const double* w, int64_t N, int M, double* A,
                        cudaStream_t stream)
{
    gram_kernel<<<dim3(M + 1, M + 1), kGramThreads, 0, stream>>>(basis, x, w, N, M, A);
    return cudaGetLastError();
}

cudaError_t launch_subset_fits(const double* A, int n, double* l_out, int sm_count, cudaStream_t stream)
{
    const int M = 2 * n + 1, LDA = M + 1;
    const size_t per_warp = ((size_t)M * M + 3 * M + (M + 1) / 2 + (n + 2) + (n + 1) / 2 + 3) & ~(size_t)1;
    const size_t smem = ((size_t)LDA * LDA + kSubsetWarps * per_warp) * 8;
    cudaError_t e = cudaFuncSetAttribute(subset_fit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    // each task walks 2^(n-s) subsets: 64 for large pools; at least 2^11 tasks (when n allows) so
    // that small pools still fill the chip
    int s = n <= 11 ? n : (n - 6 > 11 ? n - 6 : 11);
    const int64_t tasks = (int64_t)1 << s;
    int64_t grid = (tasks + kSubsetWarps - 1) / kSubsetWarps;
    if (grid > (int64_t)sm_count * 8) grid = (int64_t)sm_count * 8;
    subset_fit_kernel<<<(unsigned)grid, kSubsetWarps * 32, smem, stream>>>(A, n, s, l_out);
    return cudaGetLastError();
}

}  // namespace fredec
