// fredec_api.cu -- host side of libfredec_b200.so: the C-ABI of include/fredec.h.
// Argument validation, host/device pointer staging, library-owned workspace, launch
// configuration and device-side timing.  All arithmetic of the method runs in the kernels.
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <vector>
#include <cuda_runtime.h>

#include "fredec.h"
#include "prep_kernel.cuh"
#include "scan_mma_kernel.cuh"
#include "refine_kernel.cuh"
#include "stat_kernel.cuh"
#include "subset_kernel.cuh"
#include "trig_kernel.cuh"
#include "topk_kernel.cuh"

using namespace fredec;

namespace {

struct DevBuf {
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t n)
    {
        if (n <= cap) return cudaSuccess;
        if (p) {
            cudaError_t e = cudaFree(p);
            p = nullptr;
            cap = 0;
            if (e != cudaSuccess) return e;
        }
        size_t want = n + n / 8 + 256;
        cudaError_t e = cudaMalloc(&p, want);
        if (e == cudaSuccess) cap = want;
        return e;
    }
    void release()
    {
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
    }
    template <class T>
    T* as() const { return static_cast<T*>(p); }
};

struct HostBuf {
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t n)
    {
        if (n <= cap) return cudaSuccess;
        if (p) cudaFreeHost(p);
        p = nullptr;
        cap = 0;
        cudaError_t e = cudaMallocHost(&p, n + 256);
        if (e == cudaSuccess) cap = n + 256;
        return e;
    }
    void release()
    {
        if (p) cudaFreeHost(p);
        p = nullptr;
        cap = 0;
    }
};

constexpr int kNumEvents = 7;

struct State {
    bool ready = false;
    int device = -1;
    int sm_count = 0;
    cudaStream_t stream = nullptr;
    cudaEvent_t ev[kNumEvents] = {};
    DevBuf in_t, in_x, in_w, in_base, in_z, out_z, out_idx, out_chi2;
    DevBuf fz, fi, fedge, fthr;  // fused peak extraction: lists, edge records, group thresholds
    DevBuf gram, rf, part, p1_base, p1_freq, p1_z, p1_idx, p1_stats, tab, srec, psi, xt, info, ws, red, part_z, part_i, count, sink;
    HostBuf h_info, h_count, h_flag, h_p1;
    DevBuf flag;
    int last_cuda = 0;
    double timing[4] = {0, 0, 0, 0};
    int launches = 0;
    // asynchronous form (fredec_set_async): a scan / top-k call whose pointers are all device pointers
    // returns after enqueueing; its status is resolved by fredec_last_status()
    bool async_mode = false;
    bool pending = false;        // a call has been enqueued and not yet resolved
    bool pend_series = false, pend_topk = false;
    int64_t pend_B = 0;
    int last_status = 0, last_count = 0;
    int unread_status = 0;  // first error of a pending call that was settled by a later call, not yet reported
    // the per-stage timing events of the scan / top-k calls; off inside fredec_phase1, whose iterations are
    // short enough for seven event records each to show
    bool timing_on = true;
};
State g;

cudaError_t record_event(int i) { return g.timing_on ? cudaEventRecord(g.ev[i], g.stream) : cudaSuccess; }
struct TimingOff {
    bool before;
    TimingOff() : before(g.timing_on) { g.timing_on = false; }
    ~TimingOff() { g.timing_on = before; }
};

// Error path of every entry point: copies or kernels that touch the caller's buffers may still be
// queued on the stream; wait for them so that "the library keeps no pointer after return" also holds
// when a call fails (the result of the wait itself is ignored).
void drain_stream()
{
    if (g.ready) (void)cudaStreamSynchronize(g.stream);
    (void)cudaGetLastError();
}

#define CK(expr)                                \
    do {                                        \
        cudaError_t e__ = (expr);               \
        if (e__ != cudaSuccess) {               \
            g.last_cuda = (int)e__;             \
            (void)cudaGetLastError();           \
            drain_stream();                     \
            return FREDEC_ECUDA;                \
        }                                       \
    } while (0)

int ensure_ready()
{
    if (g.ready) return FREDEC_OK;
    int n = 0;
    CK(cudaGetDeviceCount(&n));
    if (n < 1) {
        g.last_cuda = (int)cudaErrorNoDevice;
        return FREDEC_ECUDA;
    }
    CK(cudaGetDevice(&g.device));
    CK(cudaDeviceGetAttribute(&g.sm_count, cudaDevAttrMultiProcessorCount, g.device));
    for (int i = 0; i < kNumEvents; ++i) CK(cudaEventCreate(&g.ev[i]));
    g.ready = true;
    return FREDEC_OK;
}

// true if p is usable from device code as is
bool on_device(const void* p)
{
    cudaPointerAttributes a;
    cudaError_t e = cudaPointerGetAttributes(&a, p);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// device view of an input: the pointer itself, or a staged copy
template <class T>
int stage_in(const T* src, size_t count, DevBuf& buf, const T** out)
{
    if (src == nullptr || count == 0) {
        *out = nullptr;
        return FREDEC_OK;
    }
    if (on_device(src)) {
        *out = src;
        return FREDEC_OK;
    }
    CK(buf.reserve(count * sizeof(T)));
    CK(cudaMemcpyAsync(buf.p, src, count * sizeof(T), cudaMemcpyHostToDevice, g.stream));
    *out = buf.as<T>();
    return FREDEC_OK;
}

// device view of an output; *host_dst != nullptr means "copy back to there afterwards"
template <class T>
int stage_out(T* dst, size_t count, DevBuf& buf, T** out, T** host_dst)
{
    if (on_device(dst)) {
        *out = dst;
        *host_dst = nullptr;
        return FREDEC_OK;
    }
    CK(buf.reserve(count * sizeof(T)));
    *out = buf.as<T>();
    *host_dst = dst;
    return FREDEC_OK;
}

int check_series_args(const double* t, const double* x, const double* w, int64_t B, int64_t N,
                      const double* base_funcs, int32_t d)
{
    if (!t || !x || !w) return FREDEC_EINVAL;
    if (B < 1 || d < 0 || d > FREDEC_D_MAX || N < (int64_t)d + 3) return FREDEC_EINVAL;
    if (d > 0 && !base_funcs) return FREDEC_EINVAL;
    if (B > 65535 || N > (int64_t)1 << 31) return FREDEC_EINVAL;
    return FREDEC_OK;
}

float ev_ms(int a, int b)
{
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, g.ev[a], g.ev[b]) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0.f;
    }
    return ms;
}

// ---------------------------------------------------------------------------------------
// A compute call is assembled from three enqueue steps on g.stream and one finish:
//   begin_call -> [enqueue_series] -> [enqueue_topk] -> finish_call (copies out, one sync)
// Events: 0 start | 1 prep | 2 scan | 3 (scan done) | 4 topk | 5 (topk done) | 6 end.
// ---------------------------------------------------------------------------------------
struct Call {
    int64_t B = 0;
    bool has_series = false, has_topk = false;
    double* dz = nullptr;     // device periodogram [B][K]
    double* hz = nullptr;     // host destination of z, if any
    size_t z_count = 0;
    int64_t* didx = nullptr;  // device peak indices [B][k]
    int64_t* hidx = nullptr;
    size_t idx_count = 0;
    bool staged_inputs = false;  // an input was a host pointer (copied through library memory)
    bool fused = false;          // the scan kept per-warp peak lists instead of writing z (fm = merge parameters)
    FusedMergeParams fm;
};

int resolve_pending();
void settle_pending();

int begin_call()
{
    int rc = ensure_ready();
    if (rc) return rc;
    settle_pending();  // its events and pinned status buffers are about to be reused
    g.launches = 0;
    for (double& v : g.timing) v = 0.0;
    CK(record_event(0));
    return FREDEC_OK;
}

// orthogonalise (prep kernel), table kernel, MMA scan; inputs already on the device
// fused_k > 0 (peaks only, z_out == nullptr): a11 runs in the scan's epilogue when the scan is a single pass
// and k <= kFusedMaxK; no periodogram is written then.
int enqueue_series_mma(Call& c, const double* dt, const double* dx, const double* dw, const double* dbase, int64_t B,
                       int64_t N, int32_t d, double f0, double df, int64_t K, double* z_out, int32_t fused_k,
                       bool prepped = false)
{
    cudaStream_t st = g.stream;
    int rc;
    const size_t BN = (size_t)B * N;
    const int NB = d <= kMmaMaxNB ? d : 8;
    const int n_pass = d <= kMmaMaxNB ? 1 : (d + 7) / 8;
    const MmaScanConfig cfg = mma_scan_config(NB);
    const int R = 2 * cfg.H;
    const int64_t G4 = (N + 3) / 4;
    const int64_t U = (K + 8 * R - 1) / (8 * R);

    CK(g.psi.reserve(BN * (size_t)(d > 0 ? d : 1) * 8));
    CK(g.xt.reserve(BN * 8));
    CK(g.info.reserve((size_t)B * sizeof(SeriesInfo)));
    CK(g.h_info.reserve((size_t)B * sizeof(SeriesInfo)));
    CK(g.tab.reserve((size_t)B * n_pass * G4 * mma_group_doubles(cfg.H, NB) * 8));
    CK(g.srec.reserve((size_t)B * G4 * 4 * sizeof(SeedRec)));

    PrepParams pp;
    pp.t = dt; pp.x = dx; pp.w = dw; pp.base = dbase;
    pp.psi = g.psi.as<double>(); pp.xt = g.xt.as<double>();
    pp.info = g.info.as<SeriesInfo>();
    pp.N = N; pp.d = d;
    CK(record_event(1));
    if (!prepped) CK(launch_prep(pp, B, st));  // prepped: psi, x~ and the series record are already in place
    TableParams tp;
    tp.t = dt; tp.w = dw; tp.psi = g.psi.as<double>(); tp.xt = g.xt.as<double>();
    tp.info = g.info.as<SeriesInfo>();
    tp.tab = g.tab.as<double>(); tp.srec = g.srec.as<SeedRec>();
    tp.N = N; tp.G4 = G4; tp.d = d; tp.NB = NB; tp.n_pass = n_pass; tp.H = cfg.H; tp.df = df;
    CK(launch_table(tp, B, st));
    g.launches += prepped ? 1 : 2;
    CK(record_event(2));

    c.z_count = (size_t)B * K;
    const bool fused = z_out == nullptr && fused_k > 0 && fused_k <= kFusedMaxK && n_pass == 1;
    if (fused) {
        c.dz = nullptr;
        c.hz = nullptr;
    } else if (z_out == nullptr) {
        CK(g.out_z.reserve(c.z_count * 8));
        c.dz = g.out_z.as<double>();
        c.hz = nullptr;
    } else if ((rc = stage_out(z_out, c.z_count, g.out_z, &c.dz, &c.hz))) {
        return rc;
    }
    MmaScanParams sp;
    sp.tab = g.tab.as<double>(); sp.srec = g.srec.as<SeedRec>();
    sp.info = g.info.as<SeriesInfo>();
    sp.z = c.dz;
    sp.N = N; sp.K = K; sp.Kpad = U * 8 * R;
    sp.G4 = G4; sp.U = U; sp.T = B * U;
    sp.f0 = f0; sp.df = df;
    sp.n_pass = n_pass;
    sp.grid = (int)(sp.T < (int64_t)g.sm_count ? sp.T : (int64_t)g.sm_count);
    // ring of (table tile, seeds) slots: as many observations per slot (at most 32: two groups of 4
    // per seed warp) as leave room for three slots in shared memory; short series take 16
    constexpr size_t kSmemBudget = 221000;  // of the 232448 B a CTA may have: the kernel adds 8 KB behind the ring and ~1.3 KB static
    sp.TI = 32;
    while (sp.TI > 16 && 3 * mma_scan_slot_bytes(NB, sp.TI) > kSmemBudget) sp.TI -= 4;
    if (G4 <= 4) sp.TI = 16;
    sp.NS = (int)(kSmemBudget / mma_scan_slot_bytes(NB, sp.TI));
    if (sp.NS > kMmaMaxSlots) sp.NS = kMmaMaxSlots;
    if (sp.NS < 2) return FREDEC_EINVAL;
    sp.ws = nullptr;
    if (n_pass > 1) {
        CK(g.ws.reserve((size_t)B * 7 * sp.Kpad * 8));
        sp.ws = g.ws.as<double>();
    }
    CK(g.red.reserve((size_t)sp.grid * cfg.NW * mma_red_doubles(NB) * 8));
    sp.red = g.red.as<double>();
    // one series in one pass: full rounds per CTA + left-over rounds cut across the observations
    sp.shared = (B == 1 && n_pass == 1 && U >= (int64_t)cfg.NW * cfg.NOCT * g.sm_count) ? 1 : 0;  // >= 1 full round per CTA
    sp.F = 0;
    sp.Rt = 0;
    sp.part = nullptr;
    if (sp.shared) {
        const int64_t cap = (int64_t)cfg.NW * cfg.NOCT;
        sp.grid = g.sm_count;
        sp.F = (int)(U / (cap * sp.grid));
        sp.Rt = (int)((U - (int64_t)sp.F * cap * sp.grid + cap - 1) / cap);
        CK(g.part.reserve((size_t)2 * sp.grid * cfg.NW * mma_part_doubles(NB) * 8));
        sp.part = g.part.as<double>();
    }
    sp.fused_k = 0;
    sp.tail_group0 = 0;
    sp.list_z = nullptr;
    sp.list_i = nullptr;
    sp.edges = nullptr;
    sp.group_thr = nullptr;
    if (fused) {
        // one list group per (series, CTA) pair -- group = series + CTA -- and one per left-over round
        const size_t groups = (size_t)B + sp.grid + sp.Rt;
        const size_t entries = groups * cfg.NW * fused_k;
        CK(g.fz.reserve(entries * 8));
        CK(g.fi.reserve(entries * 8));
        CK(g.fedge.reserve((size_t)B * U * 4 * 8));
        CK(g.fthr.reserve(groups * 8));
        CK(cudaMemsetAsync(g.fi.p, 0xFF, entries * 8, st));  // every entry empty
        CK(cudaMemsetAsync(g.fthr.p, 0, groups * 8, st));    // no threshold yet
        sp.group_thr = g.fthr.as<unsigned long long>();
        sp.fused_k = fused_k;
        sp.tail_group0 = (int)(B + sp.grid);
        sp.list_z = g.fz.as<double>();
        sp.list_i = g.fi.as<int64_t>();
        sp.edges = g.fedge.as<double>();
        c.fused = true;
        c.fm.list_z = sp.list_z;
        c.fm.list_i = sp.list_i;
        c.fm.edges = sp.edges;
        c.fm.info = sp.info;
        c.fm.K = K;
        c.fm.U = U;
        c.fm.T = sp.T;
        c.fm.unit_points = 8 * R;
        c.fm.k = fused_k;
        c.fm.nw = cfg.NW;
        c.fm.grid = sp.grid;
        c.fm.shared = sp.shared;
        c.fm.Rt = sp.Rt;
        c.fm.tail_group0 = sp.tail_group0;
    }
    for (int pass = 0; pass < n_pass; ++pass) {
        sp.pass = pass;
        CK(launch_mma_scan(NB, sp, st));
        g.launches += (sp.shared && sp.Rt > 0) ? 2 : 1;  // + the tail-solve kernel
    }
    CK(record_event(3));
    c.B = B;
    c.has_series = true;
    return FREDEC_OK;
}

// stage inputs, orthogonalise + pack (prep kernel), scan.  z_out may be a host pointer, a
// device pointer, or nullptr (library-owned device buffer, e.g. when only peaks are wanted).
int enqueue_series(Call& c, const double* t, const double* x, const double* w, int64_t B, int64_t N,
                   const double* base_funcs, int32_t d, double f0, double df, int64_t K, double* z_out,
                   bool with_scan, int32_t fused_k = 0)
{
    cudaStream_t st = g.stream;
    int rc;
    const double *dt, *dx, *dw, *dbase;
    const size_t BN = (size_t)B * N;
    if ((rc = stage_in(t, BN, g.in_t, &dt))) return rc;
    if ((rc = stage_in(x, BN, g.in_x, &dx))) return rc;
    if ((rc = stage_in(w, BN, g.in_w, &dw))) return rc;
    if ((rc = stage_in(base_funcs, BN * d, g.in_base, &dbase))) return rc;
    c.staged_inputs = dt != t || dx != x || dw != w || dbase != base_funcs;

    if (with_scan) return enqueue_series_mma(c, dt, dx, dw, dbase, B, N, d, f0, df, K, z_out, fused_k);

    // base fit only (chi2_base): the prep kernel alone
    CK(g.psi.reserve(BN * (size_t)(d > 0 ? d : 1) * 8));
    CK(g.xt.reserve(BN * 8));
    CK(g.info.reserve((size_t)B * sizeof(SeriesInfo)));
    CK(g.h_info.reserve((size_t)B * sizeof(SeriesInfo)));
    PrepParams pp;
    pp.t = dt; pp.x = dx; pp.w = dw; pp.base = dbase;
    pp.psi = g.psi.as<double>(); pp.xt = g.xt.as<double>();
    pp.info = g.info.as<SeriesInfo>();
    pp.N = N; pp.d = d;
    CK(record_event(1));
    CK(launch_prep(pp, B, st));
    g.launches += 1;
    CK(record_event(2));
    CK(record_event(3));
    c.B = B;
    c.has_series = true;
    return FREDEC_OK;
}

// peaks of the DEVICE array dz [B][K]
int enqueue_topk(Call& c, const double* dz, int64_t B, int64_t K, int32_t k, int64_t* idx_out)
{
    cudaStream_t st = g.stream;
    int rc;
    c.idx_count = (size_t)B * k;
    if ((rc = stage_out(idx_out, c.idx_count, g.out_idx, &c.didx, &c.hidx))) return rc;
    TopkParams tp;
    tp.z = dz; tp.idx_out = c.didx; tp.K = K; tp.k = k;
    tp.nblk = topk_pick_nblk(B, K, g.sm_count);
    CK(g.count.reserve((size_t)B * sizeof(int)));
    CK(g.h_count.reserve((size_t)B * sizeof(int)));
    tp.count_out = g.count.as<int>();
    tp.part_z = nullptr; tp.part_i = nullptr;
    if (tp.nblk > 1) {
        CK(g.part_z.reserve((size_t)B * tp.nblk * k * 8));
        CK(g.part_i.reserve((size_t)B * tp.nblk * k * 8));
        tp.part_z = g.part_z.as<double>();
        tp.part_i = g.part_i.as<int64_t>();
    }
    CK(record_event(4));
    int nl = 0;
    CK(launch_topk(tp, B, st, &nl));
    g.launches += nl;
    CK(record_event(5));
    c.B = B;
    c.has_topk = true;
    return FREDEC_OK;
}

// second stage of the fused peak extraction: merges the scan's lists into idx_out
int enqueue_fused_merge(Call& c, int64_t B, int32_t k, int64_t* idx_out)
{
    cudaStream_t st = g.stream;
    int rc;
    c.idx_count = (size_t)B * k;
    if ((rc = stage_out(idx_out, c.idx_count, g.out_idx, &c.didx, &c.hidx))) return rc;
    CK(g.count.reserve((size_t)B * sizeof(int)));
    CK(g.h_count.reserve((size_t)B * sizeof(int)));
    c.fm.idx_out = c.didx;
    c.fm.count_out = g.count.as<int>();
    CK(record_event(4));
    CK(launch_fused_merge(c.fm, B, st));
    g.launches += 1;
    CK(record_event(5));
    c.has_topk = true;
    return FREDEC_OK;
}

// Waits for the enqueued call and reads its statuses: the first series status that is not 0, else 0;
// g.last_count = peaks of series 0.
int resolve_pending()
{
    if (!g.pending) return g.last_status;
    g.pending = false;
    g.last_status = FREDEC_ECUDA;
    g.last_count = 0;
    CK(cudaStreamSynchronize(g.stream));
    if (g.timing_on) {
        if (g.pend_series) {
            g.timing[0] = ev_ms(1, 2);
            g.timing[1] = ev_ms(2, 3);
        }
        if (g.pend_topk) g.timing[2] = ev_ms(4, 5);
        g.timing[3] = ev_ms(0, 6);
    }
    g.last_status = FREDEC_OK;
    if (g.pend_series) {
        const SeriesInfo* hi = static_cast<const SeriesInfo*>(g.h_info.p);
        for (int64_t b = 0; b < g.pend_B; ++b)
            if (hi[b].status != 0) {
                g.last_status = hi[b].status;
                break;
            }
    }
    if (g.pend_topk && g.last_status == FREDEC_OK) g.last_count = static_cast<const int*>(g.h_count.p)[0];
    return g.last_status;
}

// A pending call that something other than fredec_last_status has to wait for: its error, if any, is kept
// for the next fredec_last_status instead of being lost.
void settle_pending()
{
    if (!g.pending) return;
    const int rc = resolve_pending();
    if (rc < 0 && g.unread_status == 0) g.unread_status = rc;
}

// Copies results out and either synchronises and reads the statuses (*first_count = peaks of series 0),
// or -- `defer`, or the asynchronous mode with nothing to copy to the host -- leaves the call pending.
int finish_call(Call& c, int* first_count, bool defer = false)
{
    cudaStream_t st = g.stream;
    if (c.hz) CK(cudaMemcpyAsync(c.hz, c.dz, c.z_count * 8, cudaMemcpyDeviceToHost, st));
    if (c.hidx) CK(cudaMemcpyAsync(c.hidx, c.didx, c.idx_count * 8, cudaMemcpyDeviceToHost, st));
    if (c.has_series)
        CK(cudaMemcpyAsync(g.h_info.p, g.info.p, (size_t)c.B * sizeof(SeriesInfo), cudaMemcpyDeviceToHost, st));
    if (c.has_topk)
        CK(cudaMemcpyAsync(g.h_count.p, g.count.p, (size_t)c.B * sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(record_event(6));
    g.pending = true;
    g.pend_series = c.has_series;
    g.pend_topk = c.has_topk;
    g.pend_B = c.B;
    if (defer || (g.async_mode && !c.hz && !c.hidx && !c.staged_inputs)) return FREDEC_OK;
    const int rc = resolve_pending();
    if (first_count) *first_count = g.last_count;
    return rc;
}

int check_grid_args(double f0, double df, int64_t K)
{
    if (K < 1 || !(df > 0.0) || !(f0 >= 0.0) || !std::isfinite(f0) || !std::isfinite(df)) return FREDEC_EINVAL;
    if (!std::isfinite(f0 + df * (double)K)) return FREDEC_EINVAL;
    return FREDEC_OK;
}

int check_topk_args(int64_t B, int64_t K, int32_t k)
{
    if (B < 1 || B > 65535 || K < 1 || k < 1 || (int64_t)k > K || k > FREDEC_TOPK_MAX) return FREDEC_EINVAL;
    return FREDEC_OK;
}

int do_scan(const double* t, const double* x, const double* w, int64_t B, int64_t N, const double* base_funcs,
            int32_t d, double f0, double df, int64_t K, double* z_out, int32_t k, int64_t* idx_out, bool want_topk,
            bool defer = false)
{
    int rc = check_series_args(t, x, w, B, N, base_funcs, d);
    if (rc) return rc;
    if ((rc = check_grid_args(f0, df, K))) return rc;
    if (want_topk) {
        if (!idx_out) return FREDEC_EINVAL;
        if ((rc = check_topk_args(B, K, k))) return rc;
    } else if (!z_out) {
        return FREDEC_EINVAL;
    }
    if ((rc = begin_call())) return rc;
    Call c;
    if ((rc = enqueue_series(c, t, x, w, B, N, base_funcs, d, f0, df, K, z_out, true, want_topk ? k : 0))) return rc;
    if (want_topk && (rc = c.fused ? enqueue_fused_merge(c, B, k, idx_out) : enqueue_topk(c, c.dz, B, K, k, idx_out)))
        return rc;
    int count = 0;
    if ((rc = finish_call(c, &count, defer))) return rc;
    return (want_topk && B == 1) ? count : FREDEC_OK;
}

// One SLICK iteration after the first (fredec_phase1): the base was extended in place by launch_prep_append,
// so the scan starts at the table kernel.  Single series, device pointers, left pending (deferred).
int do_scan_prepped(const double* dt, const double* dx, const double* dw, int64_t N, int32_t d, double f0, double df,
                    int64_t K, double* dz, int32_t k, int64_t* didx)
{
    int rc = begin_call();
    if (rc) return rc;
    Call c;
    if ((rc = enqueue_series_mma(c, dt, dx, dw, nullptr, 1, N, d, f0, df, K, dz, 0, true))) return rc;
    if ((rc = enqueue_topk(c, c.dz, 1, K, k, didx))) return rc;
    return finish_call(c, nullptr, true);
}

int do_chi2(const double* t, const double* x, const double* w, int64_t B, int64_t N, const double* base_funcs,
            int32_t d, double* chi2_out)
{
    int rc = check_series_args(t, x, w, B, N, base_funcs, d);
    if (rc) return rc;
    if (!chi2_out) return FREDEC_EINVAL;
    if ((rc = begin_call())) return rc;
    Call c;
    if ((rc = enqueue_series(c, t, x, w, B, N, base_funcs, d, 0.0, 1.0, 1, nullptr, false))) return rc;
    if ((rc = finish_call(c, nullptr))) return rc;
    // chi2 is read from the pinned status records below: in the asynchronous mode finish_call may have left
    // the call pending (fredec.h: only the scan / top-k calls are asynchronous), so wait for it here
    if (g.pending && (rc = resolve_pending())) return rc;
    const SeriesInfo* hi = static_cast<const SeriesInfo*>(g.h_info.p);
    if (on_device(chi2_out)) {
        double* tmp = static_cast<double*>(std::malloc((size_t)B * 8));
        if (!tmp) return FREDEC_EINVAL;
        for (int64_t b = 0; b < B; ++b) tmp[b] = hi[b].chi2_base;
        cudaError_t e = cudaMemcpy(chi2_out, tmp, (size_t)B * 8, cudaMemcpyHostToDevice);
        std::free(tmp);
        CK(e);
    } else {
        for (int64_t b = 0; b < B; ++b) chi2_out[b] = hi[b].chi2_base;
    }
    return FREDEC_OK;
}

int do_topk(const double* z, int64_t B, int64_t K, int32_t k, int64_t* idx_out, int* first_count)
{
    if (!z || !idx_out) return FREDEC_EINVAL;
    int rc = check_topk_args(B, K, k);
    if (rc) return rc;
    if ((rc = begin_call())) return rc;
    const double* dz;
    if ((rc = stage_in(z, (size_t)B * K, g.in_z, &dz))) return rc;
    Call c;
    c.staged_inputs = dz != z;
    if ((rc = enqueue_topk(c, dz, B, K, k, idx_out))) return rc;
    return finish_call(c, first_count);
}

// element-wise map of a [K] array (zstat / fap1): stage, launch, copy out, one sync
template <class Launch>
int do_map(const double* in, int64_t K, double* out, Launch launch)
{
    if (!in || !out || K < 1) return FREDEC_EINVAL;
    int rc = begin_call();
    if (rc) return rc;
    const double* din;
    if ((rc = stage_in(in, (size_t)K, g.in_z, &din))) return rc;
    double *dout, *hout;
    if ((rc = stage_out(out, (size_t)K, g.out_z, &dout, &hout))) return rc;
    CK(launch(din, dout, g.stream));
    g.launches += 1;
    if (hout) CK(cudaMemcpyAsync(hout, dout, (size_t)K * 8, cudaMemcpyDeviceToHost, g.stream));
    CK(cudaEventRecord(g.ev[6], g.stream));
    CK(cudaStreamSynchronize(g.stream));
    g.timing[3] = ev_ms(0, 6);
    return FREDEC_OK;
}

// T_eff, weighted variance and mean of t; dt, dw device pointers
int device_bandwidth(const double* dt, const double* dw, int64_t N, double out4[4])
{
    CK(g.sink.reserve(64));
    CK(launch_bandwidth(dt, dw, N, g.sink.as<double>(), g.stream));
    CK(cudaMemcpyAsync(out4, g.sink.p, 32, cudaMemcpyDeviceToHost, g.stream));
    CK(cudaStreamSynchronize(g.stream));
    return out4[3] != 0.0 ? FREDEC_EDATA : FREDEC_OK;
}

// enqueues the "all finite" check of a device array; the flag is read by flag_status() after the
// call's final synchronisation
int enqueue_finite_check(const double* dv, int64_t n)
{
    CK(g.flag.reserve(sizeof(int)));
    CK(g.h_flag.reserve(sizeof(int)));
    CK(launch_finite_flag(dv, n, g.flag.as<int>(), g.stream));
    CK(cudaMemcpyAsync(g.h_flag.p, g.flag.p, sizeof(int), cudaMemcpyDeviceToHost, g.stream));
    return FREDEC_OK;
}
int flag_status() { return *static_cast<const int*>(g.h_flag.p) != 0 ? FREDEC_EDATA : FREDEC_OK; }

struct PoolEntry {
    int64_t idx;
    double z, fap;
};

}  // namespace

extern "C" {

int fredec_scan(const double* t, const double* x, const double* w, int64_t N, const double* base_funcs,
                int32_t d, double f0, double df, int64_t K, double* z_out)
{
    return do_scan(t, x, w, 1, N, base_funcs, d, f0, df, K, z_out, 0, nullptr, false);
}

int fredec_scan_batched(const double* t, const double* x, const double* w, int64_t B, int64_t N,
                        const double* base_funcs, int32_t d, double f0, double df, int64_t K, double* z_out)
{
    return do_scan(t, x, w, B, N, base_funcs, d, f0, df, K, z_out, 0, nullptr, false);
}

int fredec_scan_topk(const double* t, const double* x, const double* w, int64_t N, const double* base_funcs,
                     int32_t d, double f0, double df, int64_t K, double* z_out, int32_t k, int64_t* idx_out)
{
    return do_scan(t, x, w, 1, N, base_funcs, d, f0, df, K, z_out, k, idx_out, true);
}

int fredec_scan_topk_batched(const double* t, const double* x, const double* w, int64_t B, int64_t N,
                             const double* base_funcs, int32_t d, double f0, double df, int64_t K,
                             double* z_out, int32_t k, int64_t* idx_out)
{
    return do_scan(t, x, w, B, N, base_funcs, d, f0, df, K, z_out, k, idx_out, true);
}

int fredec_chi2_base(const double* t, const double* x, const double* w, int64_t N, const double* base_funcs,
                     int32_t d, double* chi2_base_out)
{
    return do_chi2(t, x, w, 1, N, base_funcs, d, chi2_base_out);
}

int fredec_chi2_base_batched(const double* t, const double* x, const double* w, int64_t B, int64_t N,
                             const double* base_funcs, int32_t d, double* chi2_base_out)
{
    return do_chi2(t, x, w, B, N, base_funcs, d, chi2_base_out);
}

int fredec_topk(const double* z, int64_t K, int32_t k, int64_t* idx_out)
{
    int count = 0;
    int rc = do_topk(z, 1, K, k, idx_out, &count);
    return rc < 0 ? rc : count;
}

int fredec_topk_batched(const double* z, int64_t B, int64_t K, int32_t k, int64_t* idx_out)
{
    return do_topk(z, B, K, k, idx_out, nullptr);
}

int fredec_zstat(const double* dchi2, int64_t K, double chi2_base, double N_H, double* z_out)
{
    if (!(chi2_base > 0.0) || !std::isfinite(chi2_base) || !(N_H > 0.0) || !std::isfinite(N_H)) return FREDEC_EINVAL;
    return do_map(dchi2, K, z_out, [&](const double* in, double* out, cudaStream_t st) {
        return launch_zstat(in, K, chi2_base, N_H, out, st);
    });
}

int fredec_fap1(const double* z, int64_t K, double W, double A1, double* fap_out)
{
    if (!(W >= 0.0) || !std::isfinite(W) || !(A1 > 0.0) || !std::isfinite(A1)) return FREDEC_EINVAL;
    return do_map(z, K, fap_out, [&](const double* in, double* out, cudaStream_t st) {
        return launch_fap1(in, K, W, A1, out, st);
    });
}

int fredec_bandwidth(const double* t, const double* w, int64_t N, double f_max, double* T_eff_out, double* W_out)
{
    if (!t || !w || N < 2 || !(f_max >= 0.0) || !std::isfinite(f_max)) return FREDEC_EINVAL;
    int rc = begin_call();
    if (rc) return rc;
    const double *dt, *dw;
    if ((rc = stage_in(t, (size_t)N, g.in_t, &dt))) return rc;
    if ((rc = stage_in(w, (size_t)N, g.in_w, &dw))) return rc;
    double out4[4];
    if ((rc = device_bandwidth(dt, dw, N, out4))) return rc;
    g.launches += 1;
    if (T_eff_out) *T_eff_out = out4[0];
    if (W_out) *W_out = f_max * out4[0];
    return FREDEC_OK;
}

// Phase 1 in both forms.  refine == false: fredec_phase1 (the peak's GRID frequency joins the base, which
// grows in place).  refine == true: fredec_phase1_refined (after every addition all base frequencies are
// refitted by the device Gauss-Newton of fredec_refine and the base is rebuilt from the refitted values).
static int phase1_impl(const double* t, const double* x, const double* w, int64_t N, double f0, double df, int64_t K,
                       double fap0, double fap1, double A1, int32_t max_base, int32_t k_peaks, int64_t* pool_idx,
                       double* pool_z, double* pool_fap, int32_t pool_cap, int64_t* base_idx, int32_t* n_base_out,
                       bool refine, int32_t refine_iter, double refine_tol, double* base_freq_out)
{
    if (!t || !x || !w || !pool_idx || !pool_z || !pool_fap || !base_idx || !n_base_out) return FREDEC_EINVAL;
    if (N < 4 || pool_cap < 1 || max_base < 1 || 2 * max_base + 1 > FREDEC_D_MAX) return FREDEC_EINVAL;
    if (refine && (max_base > 25 || refine_iter < 0 || !(refine_tol > 0.0) || !base_freq_out || on_device(base_freq_out)))
        return FREDEC_EINVAL;
    if (!(fap0 > 0.0) || !(fap1 <= 1.0) || !(fap0 <= fap1) || !(A1 > 0.0) || !std::isfinite(A1)) return FREDEC_EINVAL;
    int rc = check_grid_args(f0, df, K);
    if (rc) return rc;
    if ((rc = check_topk_args(1, K, k_peaks))) return rc;
    if (on_device(pool_idx) || on_device(pool_z) || on_device(pool_fap) || on_device(base_idx)) return FREDEC_EINVAL;
    if ((rc = ensure_ready())) return rc;
    cudaStream_t st = g.stream;
    TimingOff no_stage_timing;

    // the series stays on the device for all iterations
    const double *dt, *dx, *dw;
    if ((rc = stage_in(t, (size_t)N, g.in_t, &dt))) return rc;
    if ((rc = stage_in(x, (size_t)N, g.in_x, &dx))) return rc;
    if ((rc = stage_in(w, (size_t)N, g.in_w, &dw))) return rc;
    double bw[4];
    if ((rc = device_bandwidth(dt, dw, N, bw))) return rc;
    const double f_max = f0 + df * (double)(K - 1);
    const double W = f_max * bw[0];  // W = f_max T_eff

    CK(g.p1_base.reserve((size_t)(refine ? 2 * max_base + 1 : 1) * N * 8));
    // the orthonormal base grows in place from iteration to iteration: room for the last one now
    CK(g.psi.reserve((size_t)(2 * max_base + 1) * N * 8));
    CK(g.xt.reserve((size_t)N * 8));
    CK(g.p1_freq.reserve((size_t)max_base * 8));
    CK(g.p1_z.reserve((size_t)K * 8));
    CK(g.p1_idx.reserve((size_t)k_peaks * 8));
    CK(g.p1_stats.reserve((size_t)k_peaks * 16));
    CK(g.h_p1.reserve((size_t)k_peaks * 24));  // pinned: peak indices, then (z, FAP) pairs
    int64_t* idx = static_cast<int64_t*>(g.h_p1.p);
    double* stats = reinterpret_cast<double*>(idx + k_peaks);
    std::vector<double> base_f;
    std::vector<PoolEntry> pool;
    int launches = 1;
    *n_base_out = 0;

    for (int m = 0; m < max_base; ++m) {
        const int d = 2 * m + 1;
        const double NH = (double)N - 3.0 * (m + 1) - 1.0;  // N - dim H_{m+1}
        if (NH <= 0.0 || N < (int64_t)d + 3) break;
        // one host round trip per iteration: the scan and the peak search are enqueued without a
        // synchronisation, the peak statistics read chi2_base from device memory, and the statuses,
        // indices and statistics come back together
        int rc1;
        if (m == 0) {
            // the constant alone: orthogonalisation from scratch (the prep kernel)
            CK(launch_sin_base(dt, N, g.p1_freq.as<double>(), 0, g.p1_base.as<double>(), st));
            rc1 = do_scan(dt, dx, dw, 1, N, g.p1_base.as<double>(), d, f0, df, K, g.p1_z.as<double>(), k_peaks,
                          g.p1_idx.as<int64_t>(), true, true);
        } else if (refine) {
            // every base frequency moved in the refit: constant + m sinusoids rebuilt and orthogonalised anew
            CK(cudaMemcpyAsync(g.p1_freq.as<double>(), base_f.data(), (size_t)m * 8, cudaMemcpyHostToDevice, st));
            CK(launch_sin_base(dt, N, g.p1_freq.as<double>(), m, g.p1_base.as<double>(), st));
            rc1 = do_scan(dt, dx, dw, 1, N, g.p1_base.as<double>(), d, f0, df, K, g.p1_z.as<double>(), k_peaks,
                          g.p1_idx.as<int64_t>(), true, true);
        } else {
            // the base of the previous iteration plus one sinusoid: the two new functions are appended to
            // the orthonormal base in place, O(N d) instead of O(N d^2)
            CK(cudaMemcpyAsync(g.p1_freq.as<double>() + (m - 1), &base_f[m - 1], 8, cudaMemcpyHostToDevice, st));
            PrepAppendParams ap;
            ap.t = dt; ap.w = dw; ap.freq = g.p1_freq.as<double>() + (m - 1);
            ap.psi = g.psi.as<double>(); ap.xt = g.xt.as<double>(); ap.info = g.info.as<SeriesInfo>();
            ap.N = N; ap.d0 = d - 2;
            CK(launch_prep_append(ap, st));
            rc1 = do_scan_prepped(dt, dx, dw, N, d, f0, df, K, g.p1_z.as<double>(), k_peaks, g.p1_idx.as<int64_t>());
        }
        launches += 1 + g.launches;
        if (rc1 < 0) return rc1;
        CK(launch_peak_stats(g.p1_z.as<double>(), g.p1_idx.as<int64_t>(), k_peaks, g.info.as<SeriesInfo>(), NH, W, A1,
                             g.p1_stats.as<double>(), st));
        launches += 1;
        CK(cudaMemcpyAsync(idx, g.p1_idx.p, (size_t)k_peaks * 8, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(stats, g.p1_stats.p, (size_t)k_peaks * 16, cudaMemcpyDeviceToHost, st));
        if ((rc1 = resolve_pending()) < 0) return rc1;
        const int count = g.last_count;
        if (count == 0) break;
        const double chi2_base = static_cast<const SeriesInfo*>(g.h_info.p)[0].chi2_base;
        if (!(chi2_base > 0.0)) break;  // the base model already fits exactly
        const double z_top = stats[0], fap_top = stats[1];
        if (fap_top > fap0) break;
        for (int j = 0; j < count; ++j) {
            const double zj = stats[2 * j], fj = stats[2 * j + 1];
            const bool take = j == 0 || (fj < fap1 && zj >= 0.5 * z_top);
            if (!take) continue;
            auto it = std::find_if(pool.begin(), pool.end(), [&](const PoolEntry& e) { return e.idx == idx[j]; });
            if (it == pool.end()) {
                pool.push_back(PoolEntry{idx[j], zj, fj});
            } else if (fj < it->fap) {
                it->z = zj;
                it->fap = fj;
            }
        }
        base_idx[m] = idx[0];
        base_f.push_back(std::fma((double)idx[0], df, f0));
        *n_base_out = m + 1;
        if (refine && N >= 3 * (int64_t)(m + 1) + 2) {
            // PAPER.md:177-185 (eq. 17): joint local fit of all base frequencies, the new one included; when
            // the normal equations are singular the unrefined values stay (reading P5)
            std::vector<double> fr(base_f);
            double l_loc = 0.0;
            const int rr = fredec_refine(dt, dx, dw, N, fr.data(), m + 1, refine_iter, refine_tol, &l_loc, nullptr);
            launches += g.launches;
            if (rr == FREDEC_OK) base_f.swap(fr);
            else if (rr != FREDEC_ESINGULAR) return rr;
        }
    }
    if (base_freq_out)
        for (size_t i = 0; i < base_f.size(); ++i) base_freq_out[i] = base_f[i];
    std::sort(pool.begin(), pool.end(), [](const PoolEntry& a, const PoolEntry& b) {
        return a.fap < b.fap || (a.fap == b.fap && a.idx < b.idx);
    });
    size_t n = pool.size();
    if (n > (size_t)(N / 10)) n = (size_t)(N / 10);
    if (n > (size_t)pool_cap) n = (size_t)pool_cap;
    for (size_t i = 0; i < n; ++i) {
        pool_idx[i] = pool[i].idx;
        pool_z[i] = pool[i].z;
        pool_fap[i] = pool[i].fap;
    }
    g.launches = launches;
    return (int)n;
}

int fredec_phase1(const double* t, const double* x, const double* w, int64_t N, double f0, double df, int64_t K,
                  double fap0, double fap1, double A1, int32_t max_base, int32_t k_peaks, int64_t* pool_idx,
                  double* pool_z, double* pool_fap, int32_t pool_cap, int64_t* base_idx, int32_t* n_base_out)
{
    return phase1_impl(t, x, w, N, f0, df, K, fap0, fap1, A1, max_base, k_peaks, pool_idx, pool_z, pool_fap, pool_cap,
                       base_idx, n_base_out, false, 0, 0.0, nullptr);
}

int fredec_phase1_refined(const double* t, const double* x, const double* w, int64_t N, double f0, double df,
                          int64_t K, double fap0, double fap1, double A1, int32_t max_base, int32_t k_peaks,
                          int32_t refine_iter, double refine_tol, int64_t* pool_idx, double* pool_z,
                          double* pool_fap, int32_t pool_cap, int64_t* base_idx, double* base_freq,
                          int32_t* n_base_out)
{
    return phase1_impl(t, x, w, N, f0, df, K, fap0, fap1, A1, max_base, k_peaks, pool_idx, pool_z, pool_fap, pool_cap,
                       base_idx, n_base_out, true, refine_iter, refine_tol, base_freq);
}

int fredec_trig_averages(const double* t, const double* x, const double* w, int64_t N, const double* freqs, int64_t M,
                         double* out)
{
    if (!t || !x || !w || !freqs || !out || N < 1 || M < 1 || M > 0x7fffffff) return FREDEC_EINVAL;
    int rc = begin_call();
    if (rc) return rc;
    const double *dt, *dx, *dw, *dfr;
    if ((rc = stage_in(t, (size_t)N, g.in_t, &dt))) return rc;
    if ((rc = stage_in(x, (size_t)N, g.in_x, &dx))) return rc;
    if ((rc = stage_in(w, (size_t)N, g.in_w, &dw))) return rc;
    if ((rc = stage_in(freqs, (size_t)M, g.in_z, &dfr))) return rc;
    double *dout, *hout;
    if ((rc = stage_out(out, (size_t)M * kTrigCols, g.out_z, &dout, &hout))) return rc;
    if ((rc = enqueue_finite_check(dfr, M))) return rc;
    CK(launch_trig_averages(dt, dx, dw, N, dfr, M, dout, g.stream));
    g.launches += 2;
    if (hout) CK(cudaMemcpyAsync(hout, dout, (size_t)M * kTrigCols * 8, cudaMemcpyDeviceToHost, g.stream));
    CK(cudaEventRecord(g.ev[6], g.stream));
    CK(cudaStreamSynchronize(g.stream));
    g.timing[3] = ev_ms(0, 6);
    return flag_status();
}

int fredec_subset_fits(const double* t, const double* x, const double* w, int64_t N, const double* freqs, int32_t n,
                       double* l_out)
{
    if (!t || !x || !w || !freqs || !l_out || n < 1 || n > 25 || N < 2 * (int64_t)n + 2) return FREDEC_EINVAL;
    int rc = begin_call();
    if (rc) return rc;
    cudaStream_t st = g.stream;
    const int M = 2 * n + 1;
    const size_t total = (size_t)1 << n;
    const double *dt, *dx, *dw, *dfr;
    if ((rc = stage_in(t, (size_t)N, g.in_t, &dt))) return rc;
    if ((rc = stage_in(x, (size_t)N, g.in_x, &dx))) return rc;
    if ((rc = stage_in(w, (size_t)N, g.in_w, &dw))) return rc;
    if ((rc = stage_in(freqs, (size_t)n, g.p1_freq, &dfr))) return rc;
    double *dl, *hl;
    if ((rc = stage_out(l_out, total, g.out_z, &dl, &hl))) return rc;
    CK(g.p1_base.reserve((size_t)M * N * 8));
    CK(g.gram.reserve((size_t)(M + 1) * (M + 1) * 8));
    if ((rc = enqueue_finite_check(dfr, n))) return rc;
    CK(launch_sin_base(dt, N, dfr, n, g.p1_base.as<double>(), st));
    CK(launch_gram(g.p1_base.as<double>(), dx, dw, N, M, g.gram.as<double>(), st));
    CK(cudaEventRecord(g.ev[2], st));
    CK(launch_subset_fits(g.gram.as<double>(), n, dl, g.sm_count, st));
    CK(cudaEventRecord(g.ev[3], st));
    g.launches += 4;
    if (hl) CK(cudaMemcpyAsync(hl, dl, total * 8, cudaMemcpyDeviceToHost, st));
    CK(cudaEventRecord(g.ev[6], st));
    CK(cudaStreamSynchronize(st));
    g.timing[1] = ev_ms(2, 3);
    g.timing[3] = ev_ms(0, 6);
    return flag_status();
}

int fredec_refine_batched(const double* t, const double* x, const double* w, int64_t N, const double* pool_freqs,
                          int32_t n_pool, const int64_t* masks, int64_t T, int32_t max_iter, double tol,
                          double* freqs_out, double* l_out, int32_t* iters_out, int32_t* status_out)
{
    if (!t || !x || !w || !pool_freqs || !freqs_out || !l_out || n_pool < 1 || n_pool > 25 || T < 1 ||
        T > 0x7fffffff)
        return FREDEC_EINVAL;
    if (max_iter < 0 || !(tol > 0.0)) return FREDEC_EINVAL;
    int rc = begin_call();
    if (rc) return rc;
    cudaStream_t st = g.stream;
    // the largest tuple sizes the shared memory (hence the CTAs resident per SM) and the N >= 3m + 2
    // requirement; masks on the device are measured by a small kernel whose two counters are read back
    int m_max = n_pool;
    if (masks && !on_device(masks)) {
        m_max = 0;
        for (int64_t i = 0; i < T; ++i) {
            if (masks[i] < 0 || masks[i] >= ((int64_t)1 << n_pool)) return FREDEC_EINVAL;
            int c = 0;
            for (int j = 0; j < n_pool; ++j) c += (int)((masks[i] >> j) & 1);
            m_max = c > m_max ? c : m_max;
        }
    } else if (masks) {
        int stats[2] = {0, 0};
        CK(g.sink.reserve(64));
        int* dstats = reinterpret_cast<int*>(g.sink.as<double>() + 6);  // bytes 48..55; bandwidth uses 0..31
        CK(launch_mask_stats(masks, T, n_pool, dstats, st));
        CK(cudaMemcpyAsync(stats, dstats, sizeof(stats), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        g.launches += 1;
        if (stats[1] != 0) return FREDEC_EINVAL;
        m_max = stats[0];
    }
    if (N < 3 * (int64_t)m_max + 2) return FREDEC_EINVAL;
    const double *dt, *dx, *dw, *dpool;
    const int64_t* dmask;
    if ((rc = stage_in(t, (size_t)N, g.in_t, &dt))) return rc;
    if ((rc = stage_in(x, (size_t)N, g.in_x, &dx))) return rc;
    if ((rc = stage_in(w, (size_t)N, g.in_w, &dw))) return rc;
    if ((rc = stage_in(pool_freqs, (size_t)n_pool, g.p1_freq, &dpool))) return rc;
    if ((rc = stage_in(masks, masks ? (size_t)T : 0, g.in_base, &dmask))) return rc;
    double *dfo, *hfo, *dlo, *hlo;
    if ((rc = stage_out(freqs_out, (size_t)T * n_pool, g.out_z, &dfo, &hfo))) return rc;
    if ((rc = stage_out(l_out, (size_t)T, g.rf, &dlo, &hlo))) return rc;
    // iteration counts and statuses always go through library buffers (they are read here for the return code)
    CK(g.part_i.reserve((size_t)T * 2 * sizeof(int32_t)));
    int32_t* dit = g.part_i.as<int32_t>();
    int32_t* dstat = dit + T;
    CK(g.h_count.reserve((size_t)T * 2 * sizeof(int32_t)));
    if ((rc = enqueue_finite_check(dpool, n_pool))) return rc;
    CK(g.sink.reserve(64));
    CK(launch_bandwidth(dt, dw, N, g.sink.as<double>(), st));
    RefineParams rp;
    rp.t = dt; rp.x = dx; rp.w = dw; rp.bw = g.sink.as<double>(); rp.pool = dpool; rp.masks = dmask;
    rp.freqs_out = dfo; rp.l_out = dlo; rp.iters_out = dit; rp.status_out = dstat;
    rp.N = N; rp.n_pool = n_pool; rp.max_iter = max_iter; rp.tol = tol;
    CK(cudaEventRecord(g.ev[2], st));
    CK(launch_refine_batched(rp, T, m_max, st));
    CK(cudaEventRecord(g.ev[3], st));
    g.launches += 3;
    if (hfo) CK(cudaMemcpyAsync(hfo, dfo, (size_t)T * n_pool * 8, cudaMemcpyDeviceToHost, st));
    if (hlo) CK(cudaMemcpyAsync(hlo, dlo, (size_t)T * 8, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(g.h_count.p, dit, (size_t)T * 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    if (iters_out && on_device(iters_out))
        CK(cudaMemcpyAsync(iters_out, dit, (size_t)T * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    if (status_out && on_device(status_out))
        CK(cudaMemcpyAsync(status_out, dstat, (size_t)T * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    CK(cudaEventRecord(g.ev[6], st));
    CK(cudaStreamSynchronize(st));
    g.timing[1] = ev_ms(2, 3);
    g.timing[3] = ev_ms(0, 6);
    if ((rc = flag_status())) return rc;
    const int32_t* hit = static_cast<const int32_t*>(g.h_count.p);
    const int32_t* hstat = hit + T;
    if (iters_out && !on_device(iters_out)) std::memcpy(iters_out, hit, (size_t)T * sizeof(int32_t));
    if (status_out && !on_device(status_out)) std::memcpy(status_out, hstat, (size_t)T * sizeof(int32_t));
    int failed = 0;
    for (int64_t i = 0; i < T; ++i) {
        if (hstat[i] == FREDEC_EDATA) return FREDEC_EDATA;
        failed += hstat[i] != 0;
    }
    return failed;
}

int fredec_refine(const double* t, const double* x, const double* w, int64_t N, double* freqs, int32_t n,
                  int32_t max_iter, double tol, double* l_out, int32_t* iters_out)
{
    if (!freqs || !l_out || on_device(l_out) || (iters_out && on_device(iters_out))) return FREDEC_EINVAL;
    if (n < 1 || n > 25 || N < 3 * (int64_t)n + 2) return FREDEC_EINVAL;
    // one tuple: the whole "pool"; the refined frequencies overwrite the start values
    int32_t status = 0, iters = 0;
    const int rc = fredec_refine_batched(t, x, w, N, freqs, n, nullptr, 1, max_iter, tol, freqs, l_out, &iters, &status);
    if (rc < 0) return rc;
    if (iters_out) *iters_out = iters;
    return status == 0 ? FREDEC_OK : status;
}

int fredec_set_stream(void* cuda_stream)
{
    settle_pending();  // the pending call was enqueued on the old stream: wait on that one
    g.stream = static_cast<cudaStream_t>(cuda_stream);
    return FREDEC_OK;
}

int fredec_set_async(int32_t enable)
{
    settle_pending();
    g.async_mode = enable != 0;
    return FREDEC_OK;
}

int fredec_last_status(int32_t* count_out)
{
    int rc = resolve_pending();
    if (g.unread_status != 0) {  // an earlier asynchronous call failed and nobody has been told yet
        rc = g.unread_status;
        g.unread_status = 0;
    }
    if (count_out) *count_out = rc == FREDEC_OK ? g.last_count : 0;
    return rc;
}

int fredec_pending(void) { return g.pending ? 1 : 0; }

int fredec_last_timing(double out[4])
{
    if (!out) return FREDEC_EINVAL;
    settle_pending();
    for (int i = 0; i < 4; ++i) out[i] = g.timing[i];
    return FREDEC_OK;
}

int fredec_set_timing(int32_t enable)
{
    settle_pending();
    g.timing_on = enable != 0;
    return FREDEC_OK;
}

int fredec_last_launches(void) { return g.launches; }

int fredec_shutdown(void)
{
    settle_pending();  // it reads the pinned status buffers released below
    DevBuf* bufs[] = {&g.fz, &g.fi, &g.fedge, &g.fthr, &g.in_t, &g.in_x, &g.in_w, &g.in_base, &g.in_z, &g.out_z, &g.out_idx, &g.out_chi2, &g.gram, &g.rf, &g.part, &g.p1_base, &g.p1_freq, &g.p1_z, &g.p1_idx, &g.p1_stats, &g.tab, &g.srec,
                      &g.psi,  &g.xt,   &g.info, &g.ws, &g.red,     &g.part_z, &g.part_i, &g.count, &g.sink};
    for (DevBuf* b : bufs) b->release();
    g.h_info.release();
    g.h_flag.release();
    g.h_p1.release();
    g.flag.release();
    g.h_count.release();
    if (g.ready)
        for (int i = 0; i < kNumEvents; ++i) cudaEventDestroy(g.ev[i]);
    g.ready = false;
    g.pending = g.pend_series = g.pend_topk = false;
    g.last_status = FREDEC_OK;
    g.last_count = 0;
    g.unread_status = 0;
    (void)cudaGetLastError();
    return FREDEC_OK;
}

const char* fredec_strerror(int code)
{
    switch (code) {
        case FREDEC_OK: return "ok";
        case FREDEC_EINVAL: return "invalid argument";
        case FREDEC_EDATA: return "invalid data (non-finite value, negative weight or zero total weight)";
        case FREDEC_ESINGULAR: return "base functions are linearly dependent";
        case FREDEC_ECUDA: return "CUDA error (see fredec_last_cuda_error)";
        case FREDEC_ELIMIT: return "size exceeds the fixed capacity of a no-allocation entry point";
        default: return code > 0 ? "ok (count)" : "unknown error";
    }
}

int fredec_last_cuda_error(void) { return g.last_cuda; }

int fredec_version(void) { return 100; }

}  // extern "C"
