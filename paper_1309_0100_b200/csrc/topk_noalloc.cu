// topk_noalloc.cu -- fredec_topk_noalloc: peak extraction (step a11, reading S7) for
// callers that must not allocate device memory.
//
// Who this is for.  fredec_topk grows a library-owned workspace with cudaMalloc the first time it sees a
// larger problem, and allocates pinned host memory for the peak count.  Some programs that want the peaks
// of a periodogram cannot afford that:
//   * a survey pipeline that has handed the whole device to its own memory pool (a framework's caching
//     allocator, a fixed arena sized at start-up): a cudaMalloc from inside this library then fails with
//     out-of-memory although the pool has room;
//   * a service with a latency budget: cudaMalloc and cudaFree synchronise the whole device, so a call that
//     happens to grow the workspace stalls every other stream of the process;
//   * code that runs where the CUDA allocator may not be called at all (inside a region another component
//     has marked allocation-free, or under a memory quota that is already spent).
// For them this file holds its scratch memory in a file-scope device array.  The array is part of the
// loaded library image: every GPU that loads libfredec_b200.so reserves it (about 1.2 MB) until the
// process exits, whether or not the entry point is ever called.  In exchange the entry point calls no
// cudaMalloc, cudaFree, cudaMallocHost or allocating library routine, ever.
//
// The kernel is a single-launch variant of topk_scan_kernel + topk_merge_kernel (topk_kernel.cu): every CTA
// writes its partial top-k list to the scratch array, takes a ticket, and the CTA that draws the last ticket
// merges all partial lists.  Same peak rule, same total order (z descending, index ascending), hence the
// same indices bit for bit as fredec_topk.
#include <cmath>
#include <cstdint>
#include <cuda_runtime.h>
#include "fredec.h"
#include "topk_list.cuh"

namespace fredec {
namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kMaxK = FREDEC_TOPK_NOALLOC_K_MAX;  // 128
constexpr int kMaxCtas = 592;                      // 4 CTAs per SM on a 148-SM B200; the grid is clamped to this
constexpr int kHeaderBytes = 256;                  // ticket counter (the only part that must start at zero)
constexpr size_t kEntries = (size_t)kMaxCtas * kMaxK;
constexpr size_t kScratchBytes = kHeaderBytes + kEntries * (sizeof(double) + sizeof(int64_t));

// The scratch memory.  Layout: [ticket counter, padded to 256 B][part_z: kEntries doubles][part_i: kEntries
// int64].  In host code this NAME is only a handle for cudaGetSymbolAddress -- it is not a device address and
// must never be passed to a kernel or to cudaMemset as a pointer; device_state() below obtains the real
// address once per device.
static __device__ __align__(256) unsigned char g_topk_scratch[kScratchBytes];

struct Params {
    const double* z;         // [K]
    int64_t* idx_out;        // [k]
    int* count_out;          // [1]
    unsigned char* scratch;  // device address of g_topk_scratch (from cudaGetSymbolAddress)
    int64_t K;
    int k;
    int nblk;
};

__device__ __forceinline__ double2 load_pair(const double* __restrict__ z, int64_t i, int64_t K)
{
    if (i + 1 < K) return *reinterpret_cast<const double2*>(z + i);
    return make_double2(i < K ? z[i] : -INFINITY, -INFINITY);
}

// Warp lists -> shared memory -> warp 0's list holds the CTA's top k.  Returns true in warp 0 only.
template <int SLOTS>
__device__ bool cta_merge(WarpList<SLOTS>& L, int k, double* sz, int64_t* si)
{
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    L.store(sz + wid * k, si + wid * k);
    __syncthreads();
    if (wid != 0) return false;
    const int total = kWarps * k;
    for (int e = k + lane; e - lane < total; e += 32) {  // entries [0, k) are warp 0's own
        const bool valid = e < total && si[e < total ? e : 0] != kEmptyIdx;
        L.offer(valid ? sz[e] : -INFINITY, valid ? si[e] : kEmptyIdx, valid);
    }
    return true;
}

template <int SLOTS>
__device__ void write_final(const WarpList<SLOTS>& L, const Params& p)
{
    const int lane = threadIdx.x & 31;
    int found = 0;
#pragma unroll
    for (int s = 0; s < SLOTS; ++s) {
        const int r = s * 32 + lane;
        const bool has = r < p.k && L.id[s] != kEmptyIdx;
        if (r < p.k) p.idx_out[r] = has ? L.id[s] : -1;
        found += __popc(__ballot_sync(0xffffffffu, has));
    }
    if (lane == 0) *p.count_out = found;
}

template <int SLOTS>
__global__ void __launch_bounds__(kThreads) topk_noalloc_kernel(Params p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ unsigned s_ticket;
    double* sz = reinterpret_cast<double*>(smem_raw);
    int64_t* si = reinterpret_cast<int64_t*>(sz + kWarps * p.k);
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t K = p.K;
    const double* z = p.z;
    unsigned* ticket = reinterpret_cast<unsigned*>(p.scratch);
    double* part_z = reinterpret_cast<double*>(p.scratch + kHeaderBytes);
    int64_t* part_i = reinterpret_cast<int64_t*>(p.scratch + kHeaderBytes + kEntries * sizeof(double));

    // this CTA's contiguous chunk, one contiguous segment per warp, in steps of 64 points
    constexpr int64_t kStep = 64;
    int64_t chunk = (K + p.nblk - 1) / p.nblk;
    chunk = (chunk + kStep * kWarps - 1) / (kStep * kWarps) * (kStep * kWarps);
    const int64_t begin = (int64_t)blockIdx.x * chunk;
    const int64_t end = min(K, begin + chunk);
    const int64_t seg = chunk / kWarps;
    const int64_t s0 = begin + wid * seg, s1 = min(end, s0 + seg);

    WarpList<SLOTS> L;
    L.init(p.k, lane);
    if ((reinterpret_cast<uintptr_t>(z) & 15) == 0) {
        // 16-byte loads, four steps in flight.  A step is examined only if one of its points could enter the
        // list (z >= the k-th entry so far); the neighbours of the few survivors are re-read from L1/L2.
        constexpr int kUnroll = 4;
        for (int64_t base = s0; base < s1; base += kStep * kUnroll) {
            double2 v[kUnroll];
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) v[u] = load_pair(z, base + u * kStep + 2 * lane, K);
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                const int64_t sb = base + u * kStep;
                if (sb >= s1) break;  // warp-uniform
                if (__any_sync(0xffffffffu, v[u].x >= L.thr_z || v[u].y >= L.thr_z)) {
                    const int64_t i0 = sb + 2 * lane;
                    const double a = sanitize(v[u].x), c = sanitize(v[u].y);
                    const double l = (i0 > 0 && i0 - 1 < K) ? sanitize(z[i0 - 1]) : -INFINITY;
                    const double r = (i0 + 2 < K) ? sanitize(z[i0 + 2]) : -INFINITY;
                    L.offer(a, i0, i0 < s1 && a > l && a >= c);
                    L.offer(c, i0 + 1, i0 + 1 < s1 && c > a && c >= r);
                }
            }
        }
    } else {
        for (int64_t base = s0 + lane; base - lane < s1; base += 32) {
            const int64_t i = base;
            bool peak = false;
            double v = -INFINITY;
            if (i < s1) {
                v = sanitize(z[i]);
                const double l = i > 0 ? sanitize(z[i - 1]) : -INFINITY;
                const double r = i + 1 < K ? sanitize(z[i + 1]) : -INFINITY;
                peak = v > l && v >= r;
            }
            L.offer(v, i, peak);
        }
    }

    const bool w0 = cta_merge<SLOTS>(L, p.k, sz, si);
    if (p.nblk == 1) {
        if (w0) write_final<SLOTS>(L, p);
        return;
    }
    // partial list -> scratch; fence; ticket.  The CTA that draws ticket nblk - 1 sees every partial list.
    if (w0) {
        L.store(part_z + (int64_t)blockIdx.x * p.k, part_i + (int64_t)blockIdx.x * p.k);
        __threadfence();
        __syncwarp();
        if (lane == 0) s_ticket = atomicAdd(ticket, 1u);
    }
    __syncthreads();
    if (s_ticket != (unsigned)p.nblk - 1u) return;
    __threadfence();
    const int64_t total = (int64_t)p.nblk * p.k;
    L.init(p.k, lane);
    for (int64_t base = (int64_t)wid * 32; base < total; base += kThreads) {
        const int64_t e = base + lane;
        int64_t ic = kEmptyIdx;
        double zc = -INFINITY;
        if (e < total) {
            ic = __ldcg(part_i + e);
            if (ic != kEmptyIdx) zc = __ldcg(part_z + e);
        }
        L.offer(zc, ic, ic != kEmptyIdx);
    }
    __syncthreads();  // the first merge's shared lists are dead: every warp has left cta_merge's reads
    if (cta_merge<SLOTS>(L, p.k, sz, si)) write_final<SLOTS>(L, p);
}

// ---------------------------------------------------------------------------------- host side
struct DeviceState {
    unsigned char* scratch = nullptr;  // device address of g_topk_scratch on this device
    int sm_count = 0;
    bool ready = false;
};
constexpr int kMaxDevices = 64;
DeviceState g_dev[kMaxDevices];
int g_last_cuda = 0;

// Set-up, once per device, with that device current: the symbol's address on THIS device.
cudaError_t device_state(int dev, DeviceState** out)
{
    DeviceState& s = g_dev[dev];
    if (!s.ready) {
        void* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_topk_scratch);
        if (e != cudaSuccess) return e;
        if (ptr == nullptr) return cudaErrorInvalidSymbol;
        e = cudaDeviceGetAttribute(&s.sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        s.scratch = static_cast<unsigned char*>(ptr);
        s.ready = true;
    }
    *out = &s;
    return cudaSuccess;
}

// device-accessible memory of the current device (plain device or managed memory)?
cudaError_t is_device_pointer(const void* p, int dev, bool* ok)
{
    cudaPointerAttributes a;
    const cudaError_t e = cudaPointerGetAttributes(&a, p);
    if (e != cudaSuccess) return e;
    *ok = (a.type == cudaMemoryTypeDevice && a.device == dev) || a.type == cudaMemoryTypeManaged;
    return cudaSuccess;
}

template <int SLOTS>
cudaError_t launch(const Params& p, cudaStream_t stream)
{
    const size_t smem = (size_t)kWarps * p.k * 16;  // <= 16 KB for k <= 128: no opt-in needed
    topk_noalloc_kernel<SLOTS><<<(unsigned)p.nblk, kThreads, smem, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace
}  // namespace fredec

extern "C" {

int fredec_topk_noalloc(const double* z, int64_t K, int32_t k, int64_t* idx_out, int32_t* count_out,
                        void* cuda_stream)
{
    using namespace fredec;
    if (z == nullptr || idx_out == nullptr || count_out == nullptr || K < 1 || k < 1 || (int64_t)k > K)
        return FREDEC_EINVAL;
    if (k > FREDEC_TOPK_NOALLOC_K_MAX) return FREDEC_ELIMIT;  // the fixed scratch array has no room for longer lists
#define NOALLOC_CUDA(call)                   \
    do {                                     \
        const cudaError_t e__ = (call);      \
        if (e__ != cudaSuccess) {            \
            g_last_cuda = (int)e__;          \
            (void)cudaGetLastError();        \
            return FREDEC_ECUDA;             \
        }                                    \
    } while (0)
    int dev = -1;
    NOALLOC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) {
        g_last_cuda = (int)cudaErrorInvalidDevice;
        return FREDEC_ECUDA;
    }
    bool ok_z = false, ok_i = false, ok_c = false;
    NOALLOC_CUDA(is_device_pointer(z, dev, &ok_z));
    NOALLOC_CUDA(is_device_pointer(idx_out, dev, &ok_i));
    NOALLOC_CUDA(is_device_pointer(count_out, dev, &ok_c));
    if (!ok_z || !ok_i || !ok_c) return FREDEC_EINVAL;  // host buffers would need a staging allocation
    DeviceState* s = nullptr;
    NOALLOC_CUDA(device_state(dev, &s));
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);

    Params p;
    p.z = z;
    p.idx_out = idx_out;
    p.count_out = count_out;
    p.scratch = s->scratch;
    p.K = K;
    p.k = k;
    int64_t nblk = 4 * (int64_t)s->sm_count, most = (K + 4095) / 4096;  // >= ~4096 points per CTA
    if (nblk > most) nblk = most;
    if (nblk > kMaxCtas) nblk = kMaxCtas;
    if (nblk < 1) nblk = 1;
    p.nblk = (int)nblk;
    // The array keeps whatever the previous call (or an aborted one) left behind.  Only the ticket counter
    // must start at zero; the partial lists are fully rewritten by this launch before they are read.
    if (p.nblk > 1) NOALLOC_CUDA(cudaMemsetAsync(s->scratch, 0, kHeaderBytes, stream));
    if (k <= 32) NOALLOC_CUDA(launch<1>(p, stream));
    else if (k <= 64) NOALLOC_CUDA(launch<2>(p, stream));
    else NOALLOC_CUDA(launch<4>(p, stream));
#undef NOALLOC_CUDA
    return FREDEC_OK;
}

int fredec_topk_noalloc_cuda_error(void) { return fredec::g_last_cuda; }

int64_t fredec_topk_noalloc_scratch_bytes(void) { return (int64_t)fredec::kScratchBytes; }

}  // extern "C"
