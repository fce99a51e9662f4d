// prep_kernel.cu -- steps a1-a3 of the scan: validate, centre, orthogonalise the base
// model (prep_kernel, one CTA per series), per-observation table and seed records
// (table_kernel).  Once per scan.
//
// Generalises the normalisations of PAPER.md:193-197 (eq. 18: <1> = 1, <x> = 0, ...) to an
// arbitrary linear base model: the base functions are replaced by functions psi_j that are
// orthonormal under <.>, and x by its residual after the base fit.  Then the (d+2)x(d+2)
// system of PAPER.md:165-175 (eqs. 15, 16; Cholesky solve) has an identity leading block and
// collapses to the 2x2 Schur complement the scan kernel solves per frequency.
//
// Orthogonalisation is modified Gram-Schmidt applied twice ("twice is enough"), in the
// weighted inner product <u v> = sum_i w_i u_i v_i, with deterministic (fixed-order)
// block reductions.
#include "prep_kernel.cuh"

namespace fredec {

namespace {

constexpr int kPrepThreadsMax = 1024;  // one long series: as many threads as a CTA can have
constexpr int kPrepThreadsMin = 256;   // many short series: several CTAs per SM

// Fixed-order block sum, result broadcast to all threads.  `red` = 32 doubles of smem.
template <int TH>
__device__ double block_sum(double v, double* red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();  // protect `red` from the previous call's readers
    if (lane == 0) red[wid] = v;
    __syncthreads();
    double r = (lane < (TH >> 5)) ? red[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
    return r;
}

template <int TH>
__device__ double block_min(double v, double* red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    __syncthreads();
    if (lane == 0) red[wid] = v;
    __syncthreads();
    double r = (lane < (TH >> 5)) ? red[lane] : v;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) r = fmin(r, __shfl_xor_sync(0xffffffffu, r, o));
    return r;
}

// <u v> over the series (u may alias v).
template <int TH>
__device__ double wdot(const double* __restrict__ w, const double* u, const double* v, int64_t N, double* red)
{
    double acc = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += TH) acc = fma(w[i] * u[i], v[i], acc);
    return block_sum<TH>(acc, red);
}

template <int TH>
__global__ void __launch_bounds__(TH) prep_kernel(PrepParams p)
{
    __shared__ double red[32];
    const int64_t b = blockIdx.x, N = p.N;
    const int d = p.d;
    const double* t = p.t + b * N;
    const double* x = p.x + b * N;
    const double* w = p.w + b * N;
    const double* base = p.base ? p.base + b * (int64_t)d * N : nullptr;
    double* psi = p.psi + b * (int64_t)d * N;  // [d][N]
    double* xt = p.xt + b * N;                 // [N]
    SeriesInfo* info = p.info + b;

    // ---- a1: validate, W = <1>, time origin --------------------------------------------
    double bad = 0.0, neg = 0.0, wsum = 0.0, tmin = INFINITY, tmax = -INFINITY;
    for (int64_t i = threadIdx.x; i < N; i += TH) {
        double ti = t[i], xi = x[i], wi = w[i];
        if (!isfinite(ti) || !isfinite(xi) || !isfinite(wi)) bad = 1.0;
        if (wi < 0.0) neg = 1.0;
        wsum += wi;
        tmin = fmin(tmin, ti);
        tmax = fmax(tmax, ti);
        for (int j = 0; j < d; ++j)
            if (!isfinite(base[(int64_t)j * N + i])) bad = 1.0;
    }
    bad = block_sum<TH>(bad + neg, red);
    const double W = block_sum<TH>(wsum, red);
    tmin = block_min<TH>(tmin, red);
    tmax = -block_min<TH>(-tmax, red);
    int status = 0;
    if (bad != 0.0 || !(W > 0.0) || !isfinite(W)) status = -2;  // FREDEC_EDATA
    const double t_mid = 0.5 * (tmin + tmax);

    // ---- a2: orthonormal base psi (MGS, two sweeps) and residual x~ -----------------------
    if (status == 0) {
        for (int j = 0; j < d; ++j) {
            double* v = psi + (int64_t)j * N;
            for (int64_t i = threadIdx.x; i < N; i += TH) v[i] = base[(int64_t)j * N + i];
            __syncthreads();
            const double n0 = wdot<TH>(w, v, v, N, red);
            for (int sweep = 0; sweep < 2; ++sweep)
                for (int k = 0; k < j; ++k) {
                    const double* q = psi + (int64_t)k * N;
                    const double r = wdot<TH>(w, q, v, N, red);
                    for (int64_t i = threadIdx.x; i < N; i += TH) v[i] = fma(-r, q[i], v[i]);
                    __syncthreads();
                }
            const double n1 = wdot<TH>(w, v, v, N, red);
            if (!(n1 > kTauBase * n0)) {
                status = -3;  // FREDEC_ESINGULAR (uniform across the block)
                break;
            }
            const double inv = 1.0 / sqrt(n1);
            for (int64_t i = threadIdx.x; i < N; i += TH) v[i] *= inv;
            __syncthreads();
        }
    }
    double chi2 = 0.0;
    if (status == 0) {
        for (int64_t i = threadIdx.x; i < N; i += TH) xt[i] = x[i];
        __syncthreads();
        for (int sweep = 0; sweep < 2; ++sweep)
            for (int k = 0; k < d; ++k) {
                const double* q = psi + (int64_t)k * N;
                const double r = wdot<TH>(w, q, xt, N, red);
                for (int64_t i = threadIdx.x; i < N; i += TH) xt[i] = fma(-r, q[i], xt[i]);
                __syncthreads();
            }
        chi2 = wdot<TH>(w, xt, xt, N, red);
    }
    if (threadIdx.x == 0) {
        info->W = W;
        info->chi2_base = chi2;
        info->t_mid = t_mid;
        info->status = status;
        info->pad = 0;
    }
}

// ---- a3: per-observation table and seed records --------------------------
// One thread per observation (padded to whole groups of 4 with zero multipliers).  Layout:
// scan_mma_kernel.cuh.
constexpr int kTableThreads = 128;

__global__ void __launch_bounds__(kTableThreads) table_kernel(TableParams p)
{
    const int64_t b = blockIdx.z, N = p.N;
    const int pass = blockIdx.y;
    const SeriesInfo info = p.info[b];
    if (info.status != 0) return;
    const int64_t i = (int64_t)blockIdx.x * kTableThreads + threadIdx.x;
    if (i >= p.G4 * 4) return;
    const bool real = i < N;
    const int H = p.H, NT = mma_nt(H), NF = mma_nf(p.NB);
    const double tc = real ? p.t[b * N + i] - info.t_mid : 0.0;
    const double wi = real ? p.w[b * N + i] : 0.0;
    if (pass == 0) {
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
    for (int tp = 0; tp < NT / 2; ++tp) {
        for (int hh = 0; hh < 4; ++hh) {
            double c1[2], s1[2], c2[2], s2[2];
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
    }
}

}  // namespace

cudaError_t launch_table(const TableParams& p, int64_t B, cudaStream_t stream)
{
    dim3 grid((unsigned)((p.G4 * 4 + kTableThreads - 1) / kTableThreads), (unsigned)p.n_pass, (unsigned)B);
    table_kernel<<<grid, kTableThreads, 0, stream>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_prep(const PrepParams& p, int64_t B, cudaStream_t stream)
{
    if (B >= 64 || p.N <= 2048)
        prep_kernel<kPrepThreadsMin><<<(unsigned)B, kPrepThreadsMin, 0, stream>>>(p);
    else
        prep_kernel<kPrepThreadsMax><<<(unsigned)B, kPrepThreadsMax, 0, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace fredec
