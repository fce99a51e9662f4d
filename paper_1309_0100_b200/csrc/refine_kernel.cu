// refine_kernel.cu -- see refine_kernel.cuh.  One CTA per tuple of frequencies, every Gauss-Newton
// iteration on the device: the "many entirely independent instances of the fitting subroutine" of
// PAPER.md:266, with each instance's matrices in shared memory instead of global memory.
//
// Per iteration ONE sweep over the observations forms the Gram matrix of the extended row set
//   E = (1, cos w_k t', sin w_k t', t' cos w_k t', t' sin w_k t', x),  4m + 2 rows for m frequencies,
// which does not depend on the linear coefficients: its leading block is Q and g of eqs. 15-16
// (PAPER.md:165-171), and because d mu / d f_k = 2 pi (b_k t' cos w_k t' - a_k t' sin w_k t') is a
// combination of its rows, Q_f = <J J^T> and g_f = <(x - mu) J> of eq. 17 follow from it
// and the fitted theta by small dense algebra.  (The paper reaches the same sums through the
// product-to-sum identities of systems (19)/(20), one sincos per PAIR of frequencies; summing the
// products directly needs one sincos per frequency and observation, which is cheaper here.)
#include "refine_kernel.cuh"

namespace fredec {

namespace {

constexpr int kRefThreads = 256;
constexpr int kRefObs = 64;         // observations staged per sweep step
constexpr int kRefLDE = kRefObs + 1;  // odd row stride: different rows of one observation fall on different banks
constexpr double kTauRefine = 1e-12;
constexpr double kTwoPi = 6.283185307179586477;

struct RefSmem {
    int R, LDG, LDS;
    size_t E, G, S, diag0, theta, step, y, f, total;  // offsets in doubles; total in bytes
};
__host__ __device__ inline RefSmem ref_smem(int m)
{
    RefSmem L;
    L.R = 4 * m + 2;
    L.LDG = L.R | 1;
    L.LDS = (3 * m + 2) | 1;
    size_t o = 0;
    L.E = o;     o += (size_t)L.R * kRefLDE;
    L.G = o;     o += (size_t)L.R * L.LDG;
    L.S = o;     o += (size_t)(3 * m + 2) * L.LDS;
    L.diag0 = o; o += 3 * m + 2;
    L.theta = o; o += 3 * m + 2;
    L.step = o;  o += 3 * m + 2;
    L.y = o;     o += 3 * m + 2;
    L.f = o;     o += m + 1;
    L.total = o * sizeof(double);
    return L;
}

// In-place Cholesky of the leading n x n block of S (lower triangle, leading dimension LD) with row n
// carried along as a right-hand side: afterwards S[i][j] = L[i][j], S[n][j] = a_j =
// (L^{-1} g)_j and S[n][n] = D - |a|^2.  diag0[j] = the original diagonal.  Returns 0 or -3.
__device__ int chol_with_rhs(double* S, int LD, int n, const double* diag0, int* status_sm)
{
    const int tid = threadIdx.x, nth = blockDim.x;
    __syncthreads();
    if (tid == 0) *status_sm = 0;
    __syncthreads();
    for (int j = 0; j < n; ++j) {
        const double piv = S[j * LD + j];
        if (!(piv > kTauRefine * diag0[j])) {  // uniform across the CTA
            if (tid == 0) *status_sm = -3;
            break;
        }
        const double ljj = sqrt(piv), inv = 1.0 / ljj;
        __syncthreads();
        for (int i = j + tid; i <= n; i += nth) S[i * LD + j] = i == j ? ljj : S[i * LD + j] * inv;
        __syncthreads();
        const int rows = n - j;  // rows j+1 .. n
        for (int e = tid; e < rows * rows; e += nth) {
            const int i = j + 1 + e / rows, k = j + 1 + e % rows;
            if (k <= i) S[i * LD + k] = fma(-S[i * LD + j], S[k * LD + j], S[i * LD + k]);
        }
        __syncthreads();
    }
    __syncthreads();
    return *status_sm;
}

// Back substitution L^T y = a for the unknowns first .. n-1 (theta = L^{-T} a), by warp 0,
// column by column: y_j = v_j / L_jj, then v_i -= L_ji y_j for i < j with the lanes over i.
// out[j] = y_j; `v` is scratch of n doubles.  All threads call; ends with a CTA barrier.
__device__ void back_substitute(const double* S, int LD, int n, int first, double* v, double* out)
{
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        for (int i = lane; i < n; i += 32) v[i] = S[n * LD + i];
        __syncwarp();
        for (int j = n - 1; j >= first; --j) {
            const double y = v[j] / S[j * LD + j];
            __syncwarp();
            if (lane == 0) out[j] = y;
            for (int i = lane; i < j; i += 32) v[i] = fma(-S[j * LD + i], y, v[i]);
            __syncwarp();
        }
    }
    __syncthreads();
}

__device__ __forceinline__ double gsym(const double* G, int LD, int a, int b)
{
    return a >= b ? G[a * LD + b] : G[b * LD + a];
}

__global__ void __launch_bounds__(kRefThreads) refine_batched_kernel(RefineParams p)
{
    extern __shared__ __align__(16) double sm[];
    __shared__ int status_sm;
    __shared__ int sel[32];
    const int tid = threadIdx.x;
    const int64_t tuple = blockIdx.x;
    const int64_t mask = p.masks ? p.masks[tuple] : (((int64_t)1 << p.n_pool) - 1);
    int m = 0;
    for (int j = 0; j < p.n_pool; ++j)
        if ((mask >> j) & 1) {
            if (tid == 0) sel[m] = j;
            ++m;
        }
    const RefSmem L = ref_smem(m);
    double* E = sm + L.E;
    double* G = sm + L.G;
    double* S = sm + L.S;
    double* diag0 = sm + L.diag0;
    double* theta = sm + L.theta;
    double* step = sm + L.step;
    double* scratch = sm + L.y;
    double* f = sm + L.f;
    const int R = L.R, LDG = L.LDG, LDS = L.LDS, lin = 2 * m + 1, full = 3 * m + 1, xr = R - 1;
    const double T_eff = p.bw[0], t0 = p.bw[2];
    const double max_step = 0.5 / T_eff;
    __syncthreads();
    if (tid < m) f[tid] = p.pool[sel[tid]];
    __syncthreads();

    int iters = 0, status = p.bw[3] != 0.0 || !(T_eff > 0.0) ? -2 : 0;
    bool converged = p.max_iter == 0 || m == 0;  // the empty tuple has nothing to iterate
    double l = 0.0;
    while (status == 0) {
        // ---- Gram matrix of the extended rows, one sweep over the observations ----------------
        for (int e = tid; e < R * LDG; e += kRefThreads) G[e] = 0.0;
        for (int64_t c0 = 0; c0 < p.N; c0 += kRefObs) {
            const int nobs = (int)min((int64_t)kRefObs, p.N - c0);
            __syncthreads();  // the previous chunk's rows have been consumed (and G is cleared)
            for (int e = tid; e < (m + 1) * kRefObs; e += kRefThreads) {
                const int k = e / kRefObs, i = e % kRefObs;  // k == m: the constant and x
                double sw = 0.0, tc = 0.0, xi = 0.0;
                if (i < nobs) {
                    sw = sqrt(p.w[c0 + i]);
                    tc = p.t[c0 + i] - t0;
                    xi = p.x[c0 + i];
                }
                if (k == m) {
                    E[i] = sw;
                    E[xr * kRefLDE + i] = sw * xi;
                } else {
                    double s, c;
                    sincospi(2.0 * frac_prod(f[k], tc), &s, &c);
                    c *= sw;
                    s *= sw;
                    E[(1 + 2 * k) * kRefLDE + i] = c;
                    E[(2 + 2 * k) * kRefLDE + i] = s;
                    E[(lin + 2 * k) * kRefLDE + i] = tc * c;
                    E[(lin + 1 + 2 * k) * kRefLDE + i] = tc * s;
                }
            }
            __syncthreads();
            for (int e = tid; e < R * (R + 1) / 2; e += kRefThreads) {
                int a = (int)((sqrt(8.0 * e + 1.0) - 1.0) * 0.5);
                while ((a + 1) * (a + 2) / 2 <= e) ++a;
                while (a * (a + 1) / 2 > e) --a;
                const int b = e - a * (a + 1) / 2;
                const double* ra = E + a * kRefLDE;
                const double* rb = E + b * kRefLDE;
                double acc = 0.0;
#pragma unroll 8
                for (int i = 0; i < kRefObs; ++i) acc = fma(ra[i], rb[i], acc);  // rows are zero beyond nobs
                G[a * LDG + b] += acc;
            }
        }
        __syncthreads();
        // ---- exact linear fit at the current frequencies (eq. 14): Q = L L^T, a = L^{-1} g, theta = L^{-T} a
        for (int e = tid; e < (lin + 1) * (lin + 1); e += kRefThreads) {
            const int i = e / (lin + 1), k = e % (lin + 1);
            if (k > i) continue;
            const int gi = i < lin ? i : xr, gk = k < lin ? k : xr;
            S[i * LDS + k] = G[gi * LDG + gk];
            if (i == k) diag0[i] = G[gi * LDG + gk];
        }
        if (chol_with_rhs(S, LDS, lin, diag0, &status_sm) != 0) {
            status = -3;
            break;
        }
        l = fmax(S[lin * LDS + lin], 0.0);
        if (converged || iters == p.max_iter) break;
        back_substitute(S, LDS, lin, 0, scratch, theta);
        // ---- quadratic model in (theta, f) (eq. 17): Q_f = <J J^T>, g_f = <(x - mu) J>, J = (Phi, d mu / d f)
        for (int e = tid; e < (full + 1) * (full + 1); e += kRefThreads) {
            const int i = e / (full + 1), k = e % (full + 1);
            if (k > i || i == full) continue;  // the right-hand side row is filled below
            double v;
            if (i < lin) {
                v = G[i * LDG + k];
            } else {
                const int ki = i - lin, tci = lin + 2 * ki, tsi = tci + 1;
                const double ai = theta[1 + 2 * ki], bi = theta[2 + 2 * ki];
                if (k < lin) {
                    v = kTwoPi * (bi * G[tci * LDG + k] - ai * G[tsi * LDG + k]);
                } else {
                    const int kk = k - lin, tck = lin + 2 * kk, tsk = tck + 1;
                    const double ak = theta[1 + 2 * kk], bk = theta[2 + 2 * kk];
                    v = kTwoPi * kTwoPi *
                        (bi * bk * gsym(G, LDG, tci, tck) - bi * ak * gsym(G, LDG, tci, tsk) -
                         ai * bk * gsym(G, LDG, tsi, tck) + ai * ak * gsym(G, LDG, tsi, tsk));
                }
            }
            S[i * LDS + k] = v;
            if (i == k) diag0[i] = v;
        }
        for (int a = tid; a < full; a += kRefThreads) {
            // <x J_a> - sum_b theta_b <Phi_b J_a>
            double v;
            if (a < lin) {
                v = G[xr * LDG + a];
                for (int b = 0; b < lin; ++b) v = fma(-theta[b], gsym(G, LDG, a, b), v);
            } else {
                const int ka = a - lin, tca = lin + 2 * ka, tsa = tca + 1;
                const double aa = theta[1 + 2 * ka], ba = theta[2 + 2 * ka];
                double vc = G[xr * LDG + tca], vs = G[xr * LDG + tsa];
                for (int b = 0; b < lin; ++b) {
                    vc = fma(-theta[b], G[tca * LDG + b], vc);
                    vs = fma(-theta[b], G[tsa * LDG + b], vs);
                }
                v = kTwoPi * (ba * vc - aa * vs);
            }
            S[full * LDS + a] = v;
        }
        if (tid == 0) {
            S[full * LDS + full] = 0.0;
            diag0[full] = 1.0;
        }
        if (chol_with_rhs(S, LDS, full, diag0, &status_sm) != 0) {
            status = -3;
            break;
        }
        back_substitute(S, LDS, full, lin, scratch, step);  // only the frequency part of the step is needed
        double worst = 0.0;
        for (int k = 0; k < m; ++k) {
            const double dfk = fmin(fmax(step[lin + k], -max_step), max_step);  // reading R1
            worst = fmax(worst, fabs(dfk));
        }
        __syncthreads();
        if (tid < m) f[tid] += fmin(fmax(step[lin + tid], -max_step), max_step);
        __syncthreads();
        ++iters;
        converged = worst * T_eff <= p.tol;  // reading R2
    }
    __syncthreads();
    if (tid == 0) {
        p.l_out[tuple] = status == 0 ? l : 0.0;
        p.iters_out[tuple] = iters;
        p.status_out[tuple] = status;
    }
    for (int j = tid; j < p.n_pool; j += kRefThreads) p.freqs_out[tuple * p.n_pool + j] = p.pool[j];
    __syncthreads();
    if (tid < m) p.freqs_out[tuple * p.n_pool + sel[tid]] = f[tid];
}

// out[0] = largest number of selected frequencies of any tuple, out[1] = number of masks that are negative
// or select an entry beyond the pool (both start at zero)
__global__ void mask_stats_kernel(const int64_t* __restrict__ masks, int64_t T, int n_pool, int* __restrict__ out)
{
    int m = 0, bad = 0;
    const int64_t limit = (int64_t)1 << n_pool;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < T; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t mk = masks[i];
        if (mk < 0 || mk >= limit) ++bad;
        else m = max(m, __popcll((unsigned long long)mk));
    }
    for (int o = 16; o > 0; o >>= 1) {
        m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
        bad += __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if ((threadIdx.x & 31) == 0) {
        if (m > 0) atomicMax(out, m);
        if (bad > 0) atomicAdd(out + 1, bad);
    }
}

}  // namespace

cudaError_t launch_mask_stats(const int64_t* masks, int64_t T, int n_pool, int* out2, cudaStream_t stream)
{
    cudaError_t e = cudaMemsetAsync(out2, 0, 2 * sizeof(int), stream);
    if (e != cudaSuccess) return e;
    const int64_t blocks = (T + 255) / 256;
    mask_stats_kernel<<<(unsigned)(blocks < 592 ? blocks : 592), 256, 0, stream>>>(masks, T, n_pool, out2);
    return cudaGetLastError();
}

size_t refine_batched_smem(int m_max) { return ref_smem(m_max).total; }

cudaError_t launch_refine_batched(const RefineParams& p, int64_t T, int m_max, cudaStream_t stream)
{
    if (p.n_pool < 1 || p.n_pool > 25 || m_max < 0 || m_max > p.n_pool || T < 1) return cudaErrorInvalidValue;
    const size_t smem = ref_smem(m_max).total;
    static size_t attr_smem = 0;
    if (smem > attr_smem) {
        cudaError_t e = cudaFuncSetAttribute(refine_batched_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_smem = smem;
    }
    refine_batched_kernel<<<(unsigned)T, kRefThreads, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace fredec
