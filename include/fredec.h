/*
 * fredec.h -- C-ABI of libfredec_b200.so: the single-frequency (residual) periodogram
 * scan of FREDEC (Baluev 2013, arXiv:1309.0100) on one NVIDIA B200 (sm_100a).
 *
 * Citations "PAPER.md:NNN" are line numbers of the paper text this build was written
 * from; "DESIGN.md Sx/Gx" are this build's readings of points the paper leaves open.
 *
 * Notation (section 2): a time series of N times t_i, measurements x_i and
 * weights w_i; <phi> = sum_i w_i phi(t_i) (eq. 3); chi2 = <(x - mu)^2>
 * (eq. 4).  The base model is mu_base(t) = sum_{j<d} theta_j phi_j(t), given by
 * the VALUES of its d functions on the times (a constant, eq. 1; a polynomial,
 * PAPER.md:51; constant + accepted sinusoids, eq. 2).  The trial model adds
 * a cos(2 pi f t) + b sin(2 pi f t) with f fixed and all d+2 linear coefficients fitted
 * exactly (eq. 5; eq. 10 with n = 1).
 *
 * Conventions for every entry point
 *   - All floating-point arrays are IEEE double, all indices int64_t, row-major, dense.
 *   - Every data pointer may be a HOST pointer or a CUDA DEVICE pointer (of the current
 *     device); the library classifies each one with cudaPointerGetAttributes.  Host
 *     buffers are staged through library-owned device memory; device buffers are used in
 *     place (this is the measured path).  Inputs are never modified.
 *   - The caller owns every buffer it passes; the library keeps no pointer after return.
 *     Internal workspace is library-owned, grows lazily and is freed by fredec_shutdown().
 *   - Work is enqueued on the stream set by fredec_set_stream() (default: the legacy
 *     default stream).  By default every compute entry point returns AFTER its work has
 *     completed on that stream, so that the returned status is final and outputs are ready.
 *     fredec_set_async(1) selects the asynchronous form for the scan / top-k calls whose
 *     pointers are all device pointers: they return once their work is enqueued, outputs are
 *     ready after the caller's own synchronisation of the stream, and fredec_last_status()
 *     delivers what the synchronous call would have returned.
 *   - Return value: FREDEC_OK (0) or a count >= 0 on success, a negative FREDEC_E* code
 *     on failure.  Nothing throws, aborts or prints.  On failure outputs are unspecified.
 *   - There is NO CPU fallback: without a usable CUDA device compute calls return
 *     FREDEC_ECUDA.
 *   - Not thread-safe: one caller at a time per process (one process per GPU).
 */
#ifndef FREDEC_H
#define FREDEC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FREDEC_OK 0
#define FREDEC_EINVAL (-1)    /* NULL required pointer, N < d+3, d < 0 or d > FREDEC_D_MAX, B < 1, K < 1,
                                 k < 1, k > K or k > FREDEC_TOPK_MAX, df <= 0, f0 < 0, non-finite f0/df */
#define FREDEC_EDATA (-2)     /* non-finite t/x/w/base value, w_i < 0, sum w = 0 */
#define FREDEC_ESINGULAR (-3) /* base functions linearly dependent (S6b) */
#define FREDEC_ECUDA (-4)     /* CUDA runtime error; see fredec_last_cuda_error() */
#define FREDEC_ELIMIT (-5)    /* a size exceeds the fixed capacity of an entry point that owns no growable
                                 memory (fredec_topk_noalloc: k > FREDEC_TOPK_NOALLOC_K_MAX) */

#define FREDEC_D_MAX 64       /* the paper's pools reach n = 25 sinusoids => d = 51 */
#define FREDEC_TOPK_MAX 1024
#define FREDEC_TOPK_NOALLOC_K_MAX 128 /* longest peak list of fredec_topk_noalloc (its scratch array is fixed) */

/*
 * fredec_scan -- periodogram scan (section 4.2 "single-frequency residual
 * periodograms"; eq. 10; sums of PAPER.md:165-171 eqs. 15-16; solve of
 * PAPER.md:175).  For k = 0..K-1, with f_k = f0 + k*df (cycles per unit of t):
 *
 *   z_out[k] = min_theta chi2(base)  -  min_{theta,a,b} chi2(base + a cos 2 pi f_k t + b sin 2 pi f_k t)
 *
 * i.e. the chi-square reduction, in the units of sum w x^2; 0 <= z_out[k] <= chi2_base.
 * The paper's statistic is the monotone transform z = (N_H/2) ln(chi2_base/(chi2_base - z_out))
 * (eq. 8, reading G1), so peak positions are identical.
 *
 *   t, x, w      [N]     times, measurements, weights (w_i >= 0); any order of t
 *   N                    number of observations, N >= d + 3 (N_H = N - 3n - 1 > 0)
 *   base_funcs   [d][N]  values phi_j(t_i) of the base-model functions; NULL allowed iff d == 0
 *   d                    0 <= d <= FREDEC_D_MAX
 *   f0, df, K            frequency grid, f0 >= 0, df > 0, K >= 1 ("dense enough ... grid")
 *   z_out        [K]     output
 *
 * A trial frequency whose cos/sin column lies in the span of the base (f = 0 with a constant
 * in the base; f equal to a base frequency) contributes nothing: that column is dropped and
 * z stays finite (reading S6).  Never writes NaN or inf.
 */
int fredec_scan(const double* t, const double* x, const double* w, int64_t N,
                const double* base_funcs, int32_t d,
                double f0, double df, int64_t K, double* z_out);

/*
 * fredec_scan_batched -- B independent series of equal length on a shared grid.
 *   t, x, w [B][N];  base_funcs [B][d][N];  z_out [B][K].
 */
int fredec_scan_batched(const double* t, const double* x, const double* w, int64_t B, int64_t N,
                        const double* base_funcs, int32_t d,
                        double f0, double df, int64_t K, double* z_out);

/*
 * fredec_chi2_base -- chi2_base = min_theta <(x - sum_j theta_j phi_j)^2>, the l_m of
 * PAPER.md:81 (eq. 7) for the base model alone; upper bound of z_out and the quantity the
 * paper's statistic normalises by.  Arguments as fredec_scan; chi2_base_out is one double
 * ([B] doubles for the batched form).
 */
int fredec_chi2_base(const double* t, const double* x, const double* w, int64_t N,
                     const double* base_funcs, int32_t d, double* chi2_base_out);
int fredec_chi2_base_batched(const double* t, const double* x, const double* w, int64_t B, int64_t N,
                             const double* base_funcs, int32_t d, double* chi2_base_out);

/*
 * fredec_topk -- peak extraction on a periodogram ("the largest peak
 * remaining" and the "other periodogram peaks").  Reading S7: index i is a peak iff
 * z[i] > z[i-1] and z[i] >= z[i+1] (a plateau yields its lowest index); neighbours outside
 * [0, K) and NaN count as -infinity.  Peaks are ranked by z descending, then index ascending;
 * the first k indices go to idx_out[0..k-1]; unused slots are -1.  Bit-exact in indices.
 * Returns the number of peaks written (0..k), or a negative error code.
 *   z [K] input;  1 <= k <= min(K, FREDEC_TOPK_MAX);  idx_out [k].
 * Batched form: z [B][K], idx_out [B][k]; returns FREDEC_OK.
 */
int fredec_topk(const double* z, int64_t K, int32_t k, int64_t* idx_out);
int fredec_topk_batched(const double* z, int64_t B, int64_t K, int32_t k, int64_t* idx_out);

/*
 * fredec_topk_noalloc -- fredec_topk for callers that must not allocate device memory (same operation:
 * PAPER.md:201-206, reading S7; same indices bit for bit).
 *
 * Why it exists.  fredec_topk keeps a library-owned workspace that it grows with cudaMalloc when a larger
 * problem arrives, and pinned host memory for the count it returns.  That is wrong for a program that has
 * given the whole GPU to its own memory pool (the library's cudaMalloc then reports out-of-memory while the
 * pool sits half empty), for a service that cannot take the device-wide stall a cudaMalloc / cudaFree
 * causes on all its streams, and for code running where the CUDA allocator is off limits.  This entry point
 * never calls cudaMalloc, cudaFree, cudaMallocHost or any allocating library routine.  Its only scratch
 * memory is an array compiled into the library: fredec_topk_noalloc_scratch_bytes() bytes (about 1.2 MB)
 * that every GPU which loads libfredec_b200.so holds until the process exits.
 *
 *   z [K]          DEVICE pointer (device or managed memory of the current device), input, not modified
 *   K >= 1;  1 <= k <= min(K, FREDEC_TOPK_NOALLOC_K_MAX)
 *   idx_out [k]    DEVICE pointer: indices of the k highest peaks, z descending then index ascending,
 *                  unused slots -1
 *   count_out [1]  DEVICE pointer (int32): number of peaks written, 0..k
 *   cuda_stream    a cudaStream_t passed as void* (NULL: the default stream); fredec_set_stream does not
 *                  apply here.  The work (one 256-byte memset and one kernel) is enqueued on it and the
 *                  call returns without waiting: the outputs are ready once the caller has synchronised
 *                  with that stream.
 *
 * Returns FREDEC_OK; FREDEC_EINVAL for a NULL pointer, K < 1, k < 1, k > K, or a pointer that is not
 * device-accessible (host buffers would need staging memory, which this call may not allocate);
 * FREDEC_ELIMIT for k > FREDEC_TOPK_NOALLOC_K_MAX -- use fredec_topk for longer lists;
 * FREDEC_ECUDA for a CUDA error, whose cudaError_t fredec_topk_noalloc_cuda_error() returns.
 * There is no limit on K.
 *
 * Rules that follow from the shared, fixed array:
 *   - The first call on each device looks up the array's address on that device (the device must be the
 *     current one, as for every call).  Make that first call during start-up, outside any stream capture.
 *   - All calls on a device use the same array.  Each call clears the part that has to start at zero
 *     itself (on cuda_stream, before its kernel), so calls issued one after another on one stream are
 *     safe.  Two calls that can run on the GPU at the same time (different streams without an ordering
 *     between them, or two host threads) race on the array and give wrong peaks: order them.
 */
int fredec_topk_noalloc(const double* z, int64_t K, int32_t k, int64_t* idx_out, int32_t* count_out,
                        void* cuda_stream);
int fredec_topk_noalloc_cuda_error(void);        /* the cudaError_t behind its last FREDEC_ECUDA, else 0 */
int64_t fredec_topk_noalloc_scratch_bytes(void); /* size of the built-in scratch array, per GPU */

/*
 * fredec_scan_topk -- the whole hot path in one call: fredec_scan followed by fredec_topk on
 * the periodogram while it is still in device memory (one phase-1 iteration of PAPER.md:201).
 * z_out may be NULL when only the peaks are wanted.  Then, for d <= 9 and k <= 32, NO periodogram is
 * written anywhere: the peak test runs in the scan kernel's epilogue on the values it has just solved
 * for (per-warp sorted lists plus one edge record per tile of frequencies, merged by a second small
 * kernel), so B x K x 8 bytes of device memory and their traffic are not needed; the indices are the
 * same, bit for bit, as with a periodogram.  For larger d or k the periodogram goes to a
 * library-owned device buffer instead and is not copied out.  Other arguments as above.
 * Returns the number of peaks written (single series) / FREDEC_OK (batched), or an error.
 */
int fredec_scan_topk(const double* t, const double* x, const double* w, int64_t N,
                     const double* base_funcs, int32_t d, double f0, double df, int64_t K,
                     double* z_out, int32_t k, int64_t* idx_out);
int fredec_scan_topk_batched(const double* t, const double* x, const double* w, int64_t B, int64_t N,
                             const double* base_funcs, int32_t d, double f0, double df, int64_t K,
                             double* z_out, int32_t k, int64_t* idx_out);

/* ------------------------------------------- statistic, FAP and the phase-1 driver */

/*
 * fredec_zstat -- the paper's statistic from the chi-square reduction (eq. 8,
 * PAPER.md:106 eq. 10; reading G1: the printed ratio is read as the likelihood ratio
 * l_base / l_alt):   z_out[k] = (N_H / 2) ln(chi2_base / (chi2_base - dchi2[k])).
 *   dchi2 [K]   output of fredec_scan;  chi2_base > 0 from fredec_chi2_base;
 *   N_H         N - dim H of the alternative: N - 3(m+1) - 1 when the base is a
 *               constant + m sinusoids; in general N - d - (fitted base frequencies) - 3.  N_H > 0.
 *   z_out [K]   may alias dchi2.  +inf where dchi2 == chi2_base (perfect fit).
 */
int fredec_zstat(const double* dchi2, int64_t K, double chi2_base, double N_H, double* z_out);

/*
 * fredec_fap1 -- single-frequency false alarm probability bound (eq. 13, n = 1):
 *   fap_out[k] = min(1, A1 * W * exp(-z[k]) * sqrt(z[k]));  1 where z[k] <= 0.
 *   W   = f_max * T_eff (fredec_bandwidth);  A1 = the coefficient A~_1, which this paper does not
 *   print ("some numeric coefficients that we do not detail here"): the caller
 *   supplies it (A1 > 0; 1.0 is the single-frequency bound of the Paper-I series).  fap_out may alias z.
 */
int fredec_fap1(const double* z, int64_t K, double W, double A1, double* fap_out);

/*
 * fredec_bandwidth -- T_eff = sqrt(4 pi Var(t_i)) with the weighted variance of the times, and
 * W = f_max * T_eff.  t, w [N]; f_max >= 0; either output may be NULL.
 */
int fredec_bandwidth(const double* t, const double* w, int64_t N, double f_max, double* T_eff_out, double* W_out);

/*
 * fredec_phase1 -- phase 1 of FREDEC, the preliminary scan that builds the pool of candidate
 * frequencies (section 4.2; SLICK + QUICK):
 *   repeat: base model = constant + cos/sin pairs at the base frequencies found so far (all linear
 *   coefficients refitted at every trial frequency, frequencies fixed: reading S4) -> residual
 *   periodogram on the grid -> its k_peaks highest peaks -> statistic (fredec_zstat with
 *   N_H = N - 3(m+1) - 1, m = base frequencies) and FAP (fredec_fap1, W from the grid's f_max).
 *   Stop when the FAP of the highest peak exceeds fap0.  Otherwise every peak with FAP < fap1 AND
 *   height >= half of the highest goes to the pool (a grid point already in the
 *   pool keeps its smaller FAP), and the highest peak's frequency joins the base.
 *   Finally the pool is cut to N/10 entries of smallest FAP.
 * fredec_phase1 adds the GRID frequency of the peak to the base; fredec_phase1_refined (below) refits the
 * base frequencies after every addition.  DESIGN.md section 11 lists the readings.
 *
 *   t, x, w [N], f0, df, K        as fredec_scan (the base model is built internally)
 *   fap0 <= fap1 in (0, 1]        thresholds (PAPER.md:228 defaults: 0.05 and 0.1);  A1 as fredec_fap1
 *   max_base                      at most this many residual periodograms / base frequencies (>= 1,
 *                                 2*max_base + 1 <= FREDEC_D_MAX)
 *   k_peaks                       peaks examined per periodogram (1..FREDEC_TOPK_MAX)
 *   pool_idx, pool_z, pool_fap [pool_cap]   HOST arrays: grid index, statistic and FAP of the pool,
 *                                 sorted by FAP ascending then index; pool_cap >= 1
 *   base_idx [max_base]           HOST array: grid indices of the base frequencies in the order found
 *   n_base_out                    number of base frequencies
 * Returns the pool size (<= min(pool_cap, N/10)), or a negative error code.
 */
int fredec_phase1(const double* t, const double* x, const double* w, int64_t N,
                  double f0, double df, int64_t K,
                  double fap0, double fap1, double A1, int32_t max_base, int32_t k_peaks,
                  int64_t* pool_idx, double* pool_z, double* pool_fap, int32_t pool_cap,
                  int64_t* base_idx, int32_t* n_base_out);

/*
 * fredec_phase1_refined -- phase 1 with the base model fitted as the paper fits such models: after the
 * grid frequency of the highest peak has joined the base, ALL base frequencies are refitted
 * together by the local multifrequency fit of PAPER.md:177-185 (eq. 17; the device Gauss-Newton of
 * fredec_refine, started from the current values), and the next residual periodogram is computed against
 * constant + sinusoids at the refitted, off-grid frequencies (reading P5).  A signal
 * up to df/2 away from the nearest grid point is then removed whole, instead of leaving a residue that
 * re-enters the base and the pool at the neighbouring grid point a few iterations later.
 *   refine_iter >= 0, refine_tol > 0   as max_iter, tol of fredec_refine (20 and 1e-9 are sensible)
 *   max_base <= 25                     (the limit of fredec_refine)
 *   base_idx [max_base]                HOST: grid index of each iteration's highest peak, in the order found
 *   base_freq [max_base]               HOST: the frequencies the base model ends with (refitted)
 * Everything else as fredec_phase1, including the pool (grid indices of periodogram peaks).  If a refit
 * fails (singular normal equations) that iteration keeps its unrefined frequencies.
 */
int fredec_phase1_refined(const double* t, const double* x, const double* w, int64_t N,
                          double f0, double df, int64_t K,
                          double fap0, double fap1, double A1, int32_t max_base, int32_t k_peaks,
                          int32_t refine_iter, double refine_tol,
                          int64_t* pool_idx, double* pool_z, double* pool_fap, int32_t pool_cap,
                          int64_t* base_idx, double* base_freq, int32_t* n_base_out);

/*
 * fredec_trig_averages -- the trigonometric averages behind the gradient and Fisher matrix of the
 * local multifrequency fit (section 5, systems (19) and (20)) at an ARBITRARY list
 * of M frequencies f_j (omega_j = 2 pi f_j; for system (20) the caller passes the sums and
 * differences f_k +- f_m).  out [M][10], row j, in the paper's order:
 *   system (19):  <cos wt> <sin wt> <t cos wt> <t sin wt> <x cos wt> <x sin wt> <x t cos wt> <x t sin wt>
 *   system (20):  columns 0..3 again, then  <t^2 cos wt> <t^2 sin wt>   (columns 8, 9)
 * with <phi> = sum_i w_i phi(t_i) and t used as given (the paper centres it so that
 * <t> = 0).  t, x, w [N]; freqs [M], finite; M <= 2^31 - 1.
 */
int fredec_trig_averages(const double* t, const double* x, const double* w, int64_t N,
                         const double* freqs, int64_t M, double* out);

/*
 * fredec_subset_fits -- the linear multifrequency fit (section 3: Q = L L^T,
 * a = L^{-1} g, l = D - |a|^2 with g, Q of eqs. 15-16; reading G2) for EVERY subset of a pool of n
 * frequencies, as phase 2 needs them (2^n - 1 values), the frequencies held fixed
 * (the l_m(f') of eq. 7, PAPER.md:81 -- not the locally refitted l_{m,loc}):
 *   l_out[mask] = min over theta of <(x - theta_0 - sum_{j in mask} (a_j cos 2 pi f_j t + b_j sin 2 pi f_j t))^2>
 * for mask = 0 .. 2^n - 1 (bit j selects freqs[j]); l_out[0] is the chi-square of the constant alone.
 * A function that the preceding ones of its subset already span (equal frequencies) is dropped
 * (rule S6).  t, x, w [N]; freqs [n], 1 <= n <= 25, N >= 2n + 2; l_out [2^n].
 */
int fredec_subset_fits(const double* t, const double* x, const double* w, int64_t N,
                       const double* freqs, int32_t n, double* l_out);

/*
 * fredec_refine -- the local multifrequency fit l_{n,loc} (section 3, eq. 17): starting
 * from preliminary frequencies (periodogram peaks), iterate { exact linear fit of theta (eq. 14) ->
 * quadratic model of chi2 in (theta, f) with g_f, Q_f (their theta-part vanishes / equals Q) -> step
 * Q_f^{-1} g_f -> update f }, and finish with one more linear fit.  Model: eq. 2, constant +
 * n sinusoids; times are centred on their weighted mean.  Q_f is the Gauss-Newton
 * (Fisher) matrix <J J^T>, J = (model functions, d mu / d f_k).  Readings (R1-R2):
 * a frequency step is clamped to +-0.5 / T_eff so that the fit stays inside its periodogram peak
 * ("local"); iteration stops when max_k |step_k| * T_eff <= tol.
 *   t, x, w [N];  freqs [n] in: start, out: refined (host or device);  1 <= n <= 25, N >= 3n + 2
 *   max_iter >= 0 frequency updates at most;  tol > 0 (cycles of phase drift over T_eff)
 *   l_out      HOST double: min chi2 at the returned frequencies;  iters_out  HOST int32 (may be NULL)
 * Returns FREDEC_OK, or FREDEC_ESINGULAR when the normal equations are singular (equal frequencies).
 */
int fredec_refine(const double* t, const double* x, const double* w, int64_t N,
                  double* freqs, int32_t n, int32_t max_iter, double tol,
                  double* l_out, int32_t* iters_out);

/*
 * fredec_refine_batched -- the local fit of fredec_refine for T tuples drawn from one pool of n_pool
 * frequencies, in one call: the table of l_{m,loc} that phase 2 builds for the subsets of the pool
 * (PAPER.md:214), computed as "many entirely independent instances of the fitting subroutine"
 * -- one thread block per tuple, all Gauss-Newton iterations on the device.
 *   t, x, w [N];  pool_freqs [n_pool], finite, 1 <= n_pool <= 25: the start frequencies
 *   masks [T]     bit j of masks[i] selects pool_freqs[j] for tuple i (0 <= masks[i] < 2^n_pool; the empty
 *                 tuple is the constant alone); NULL: every tuple is the whole pool.  N >= 3m + 2 for the
 *                 largest tuple size m.  Host or device; a mask out of range is FREDEC_EINVAL either way
 *                 (device masks are checked, and m found, by a small kernel before the fits start)
 *   max_iter, tol as fredec_refine
 *   freqs_out [T][n_pool]  refined frequencies of the selected entries, pool_freqs[j] for the others
 *   l_out [T]              min chi2 at the returned frequencies
 *   iters_out, status_out [T] int32 (either may be NULL): frequency updates made; 0 or FREDEC_ESINGULAR
 *                 (singular normal equations, e.g. two equal frequencies in the tuple; l_out is then 0)
 * Returns the number of tuples whose status is not 0 (so 0 = every fit succeeded), or a negative error
 * code (FREDEC_EDATA: non-finite frequency or bad t / w).
 */
int fredec_refine_batched(const double* t, const double* x, const double* w, int64_t N,
                          const double* pool_freqs, int32_t n_pool, const int64_t* masks, int64_t T,
                          int32_t max_iter, double tol,
                          double* freqs_out, double* l_out, int32_t* iters_out, int32_t* status_out);

/* ----------------------------------------------------------------- runtime control */

/* Stream on which all work is enqueued (a cudaStream_t passed as void*); NULL = default. */
int fredec_set_stream(void* cuda_stream);

/*
 * fredec_set_async -- enable != 0: fredec_scan, fredec_scan_batched, fredec_topk, fredec_topk_batched,
 * fredec_scan_topk and fredec_scan_topk_batched return FREDEC_OK as soon as their work is enqueued on
 * the library's stream, PROVIDED every data pointer of the call is a device pointer (a call with a host
 * pointer stays synchronous: the library may keep no host pointer after return).  Argument errors are
 * still returned at once.  Data errors (FREDEC_EDATA, FREDEC_ESINGULAR) and the peak count are then
 * obtained with fredec_last_status().  The next compute call waits for a pending one before it enqueues
 * anything (their status buffers are shared), so at most one call is ever pending and consecutive calls are
 * NOT pipelined: the mode defers the host's wait to the next call, it does not remove it.  If that wait finds
 * a data error, the error is kept and the next fredec_last_status() reports it (the first such error wins).
 * enable == 0 (default): synchronous.
 */
int fredec_set_async(int32_t enable);

/*
 * fredec_last_status -- waits for the pending asynchronous call, if any (synchronises the stream), and
 * returns the status the synchronous form would have returned: FREDEC_OK or a negative code; *count_out
 * (may be NULL) receives the number of peaks of series 0 when the call extracted peaks.  Without a
 * pending call it repeats the status of the last resolved one.  An error of an earlier asynchronous call
 * that a later call had to wait for is reported here first, once.
 */
int fredec_last_status(int32_t* count_out);

/* 1 while an asynchronous call is enqueued and its status has not been read, else 0. */
int fredec_pending(void);

/* Device-side durations (ms, CUDA events on the library's stream) of the kernels of the LAST
 * compute call: out[0] = base orthogonalisation + packing kernel(s), out[1] = scan kernel(s),
 * out[2] = top-k kernel(s), out[3] = whole call including staging copies. Unused = 0. */
int fredec_last_timing(double out[4]);

/*
 * fredec_set_timing -- enable == 0: the scan / top-k calls stop recording the per-stage CUDA events behind
 * fredec_last_timing (seven event records per call, about 25 microseconds of host time: what a call on a
 * small series costs otherwise); fredec_last_timing then reports zeros.  enable != 0 (default): recorded.
 */
int fredec_set_timing(int32_t enable);

/* Number of kernels the LAST compute call launched. */
int fredec_last_launches(void);

/* Frees all library-owned device memory, events and staging buffers. */
int fredec_shutdown(void);

const char* fredec_strerror(int code);
int fredec_last_cuda_error(void);   /* the cudaError_t behind the last FREDEC_ECUDA, else 0 */
int fredec_version(void);           /* 100*major + minor */

#ifdef __cplusplus
}
#endif
#endif /* FREDEC_H */
