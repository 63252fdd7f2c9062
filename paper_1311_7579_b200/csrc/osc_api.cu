// osc_api.cu -- the C ABI of libosc_b200 (include/osc.h): argument checks, host precompute, launches.
// No torch types, no exceptions across the boundary; every failure sets the thread's error message.
#include <cuda_runtime.h>

#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <array>
#include <complex>
#include <limits>
#include <map>
#include <memory>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "../../include/osc.h"
#include "osc_host.cuh"
#include "osc_kernels.cuh"
#include "osc_like.cuh"
#include "osc_scan.cuh"
#include "osc_precompute.h"

using namespace oscb;

namespace {

thread_local char t_err[512] = "";
std::mutex g_mu;
HostSet g_state;
bool g_configured = false;
std::atomic<unsigned long long> g_launches{0};

// Measurement / test overrides (osc_set_batch_path, osc_set_k2_tuning); 0 = the library chooses.  Never read from
// the environment: a stray variable must not change launch shapes in a fitter that calls the library 1e6 times.
std::atomic<int> g_batch_path{0};                       // 0 auto, 2 k2, 4 k4, 41 / 42 k4 with the slice / constant-bank kernel, 5 k5
std::atomic<int> g_tune_threads{0}, g_tune_slots{0}, g_tune_nsub{0}, g_tune_bps{0};
#ifndef OSC_SORT_CHUNK
#define OSC_SORT_CHUNK 2048
#endif
std::atomic<size_t> g_sort_chunk{OSC_SORT_CHUNK};                 // events per block-local sort chunk (multiple of 512)

int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                                   \
    do {                                                                                                 \
        cudaError_t e_ = (expr);                                                                         \
        if (e_ != cudaSuccess) return fail(OSC_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_));        \
    } while (0)

bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

int sm_count(int* out)
{
    static int cached[64] = {0};
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(OSC_ERR_CUDA, "device index %d out of range", dev);
    if (cached[dev] == 0) {
        int v = 0;
        CUDA_TRY(cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev));
        cached[dev] = v;
    }
    *out = cached[dev];
    return OSC_OK;
}

int snapshot(HostSet& h)
{
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_configured) return fail(OSC_ERR_NOT_CONFIGURED, "osc_set_params has not been called");
    h = g_state;
    return OSC_OK;
}

int check_flavour(int f, const char* what)
{
    if (f < 0 || f > 2) return fail(OSC_ERR_INVALID_ARG, "%s = %d is not a flavour index (0, 1, 2)", what, f);
    return OSC_OK;
}

// Blocks per SM the persistent kernels are sized for (register budget: see DESIGN.md "Kernels").
constexpr int kBlocksPerSM = 4;

int grid_for(size_t work_items, int* grid, int blocks_per_sm = kBlocksPerSM)
{
    int sms = 0;
    int rc = sm_count(&sms);
    if (rc) return rc;
    size_t g = (size_t)sms * blocks_per_sm;
    if (work_items < g) g = work_items;
    if (g < 1) g = 1;
    *grid = (int)g;
    return OSC_OK;
}

int post_launch(const char* what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(OSC_ERR_CUDA, "%s launch failed: %s", what, cudaGetErrorString(e));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return OSC_OK;
}

constexpr int kMaxBins = 768; // 4 warps x 2 slots x 4 channels x 768 bins x 8 B = 196 KB of sub-histograms
constexpr size_t kSmemBudget = 220 * 1024;

size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

size_t k2_smem_bytes(int nb, int threads, int n_sub, int slots = kSlots)
{
    return sizeof(double) * kBinArgsDoubles + bin_table_bytes(nb) +
           sizeof(double) * (size_t)(threads / 32) * slots * n_sub * kChannels * (size_t)nb;
}

int check_bin_args(const double* E_true, const double* E_reco, const double* w0, const int8_t* channel, size_t n,
                   double energy_scale, const double* bin_edges, int n_bins, const void* out)
{
    if (n_bins < 1 || n_bins > kMaxBins)
        return fail(OSC_ERR_INVALID_ARG, "n_bins = %d outside [1, %d]", n_bins, kMaxBins);
    if (!(energy_scale > 0.0) || !std::isfinite(energy_scale))
        return fail(OSC_ERR_INVALID_ARG, "energy_scale must be finite and > 0");
    if (!bin_edges || !out) return fail(OSC_ERR_INVALID_ARG, "null bin_edges or output pointer");
    if (n > 0 && (!E_true || !E_reco || !channel)) return fail(OSC_ERR_INVALID_ARG, "null event array with n > 0");
    (void)w0;
    if (!aligned(E_true, 8) || !aligned(E_reco, 8) || !aligned(w0, 8) || !aligned(bin_edges, 8))
        return fail(OSC_ERR_ALIGNMENT, "fp64 array not 8-byte aligned");
    return OSC_OK;
}

// The stream-ordered allocator returns freed memory to the driver at the next synchronisation unless the pool is told to
// keep some: with the default threshold of zero every batched call would pay for fresh device allocations (hundreds of
// microseconds on the host).  Once per device, the default pool is allowed to retain up to 512 MB.
int keep_pool_memory()
{
    static std::atomic<bool> done[64];
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64 || done[dev].load(std::memory_order_relaxed)) return OSC_OK;
    cudaMemPool_t pool = nullptr;
    CUDA_TRY(cudaDeviceGetDefaultMemPool(&pool, dev));
    unsigned long long current = 0, keep = 512ull << 20;
    CUDA_TRY(cudaMemPoolGetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &current));
    if (current < keep) CUDA_TRY(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
    done[dev].store(true, std::memory_order_relaxed);
    return OSC_OK;
}

// Stream-ordered scratch of one call; freed (stream-ordered) when it goes out of scope.
struct Scratch {
    char* p = nullptr;
    cudaStream_t st = nullptr;
    int alloc(size_t bytes, cudaStream_t s)
    {
        st = s;
        int rc = keep_pool_memory();
        if (rc) return rc;
        CUDA_TRY(cudaMallocAsync((void**)&p, bytes, s));
        return OSC_OK;
    }
    ~Scratch()
    {
        if (p) cudaFreeAsync(p, st);
    }
};

// Device scratch the library keeps per (device, stream) for osc_reweight_bin: merge tickets (kept at zero
// between kernels by the kernels themselves) and the per-block partial histograms.  Work on one stream is
// ordered, so consecutive calls can share the buffer; it is allocated, zeroed and (when it has to grow)
// freed in stream order.
constexpr size_t kCounterBytes = 4096;
constexpr size_t kTableCacheBytes = 12 * 1024;          // >= bin_table_bytes(kMaxBins): image of the last bin table (osc_bins.cuh)
constexpr size_t kScratchHead = kCounterBytes + kTableCacheBytes;   // zeroed at allocation; the per-call areas follow
static_assert(bin_table_bytes(768) <= kTableCacheBytes, "bin-table cache too small for the largest binning");
struct StreamScratch {
    char* buf = nullptr;
    size_t cap = 0;
    std::mutex mu;            // held from the hand-out of the buffer until the launch that uses it is enqueued
};
std::mutex g_scratch_mu;
std::map<std::pair<int, cudaStream_t>, std::unique_ptr<StreamScratch>> g_scratch;

// The buffer of (current device, stream) with at least `bytes` bytes.  The lease keeps the entry locked: a second host
// thread that enqueues on the same stream waits until the first one has launched, so a buffer that is about to be
// replaced (grown) is never handed to a launch that has not been enqueued yet.
struct ScratchLease {
    std::unique_lock<std::mutex> lk;
    char* p = nullptr;
};

int stream_scratch(size_t bytes, cudaStream_t st, ScratchLease& lease)
{
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    StreamScratch* sp = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_scratch_mu);
        std::unique_ptr<StreamScratch>& e = g_scratch[std::make_pair(dev, st)];
        if (!e) e.reset(new StreamScratch);
        sp = e.get();
    }
    lease.lk = std::unique_lock<std::mutex>(sp->mu);
    StreamScratch& s = *sp;
    if (s.cap < bytes) {
        if (s.buf) CUDA_TRY(cudaFreeAsync(s.buf, st));
        s.buf = nullptr;
        s.cap = 0;
        const size_t cap = round_up(bytes + bytes / 2, 1 << 16);
        char* p = nullptr;
        CUDA_TRY(cudaMallocAsync((void**)&p, cap, st));
        cudaError_t e = cudaMemsetAsync(p, 0, kScratchHead, st);
        if (e != cudaSuccess) {
            cudaFreeAsync(p, st);
            return fail(OSC_ERR_CUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
        }
        s.buf = p;
        s.cap = cap;
    }
    lease.p = s.buf;
    return OSC_OK;
}

// The per-call areas of a stream scratch: ticket counter and bin-table cache in the zeroed head, block partials behind.
struct CallScratch {
    MergeScratch ms;
    unsigned char* table_cache;
};

// One merge level while the partial sums of a launch are at most 512 kB (one SM reads them in the shadow of a few
// microseconds), two levels above that (osc_hist.cuh, block_merge).
int merge_groups(int grid, size_t nh)
{
    return (size_t)grid * nh * sizeof(double) <= (size_t)512 * 1024 ? 1 : (grid + kGroup - 1) / kGroup;
}

size_t merge_scratch_bytes(int grid, size_t nh)
{
    return kScratchHead + ((size_t)grid + (size_t)merge_groups(grid, nh)) * nh * sizeof(double);
}

CallScratch call_scratch(char* scratch, int grid, size_t nh)
{
    CallScratch c;
    c.ms.counters = reinterpret_cast<unsigned int*>(scratch);
    c.ms.partial = reinterpret_cast<double*>(scratch + kScratchHead);
    c.ms.gpartial = c.ms.partial + (size_t)grid * nh;
    c.ms.ngroups = merge_groups(grid, nh);
    c.table_cache = reinterpret_cast<unsigned char*>(scratch + kCounterBytes);
    return c;
}

// Launch with the programmatic-stream-serialization attribute (programmatic dependent launch): the set-up of this launch
// may overlap the tail of the kernel before it on the stream; the kernels call griddepcontrol.wait before they touch
// global memory (osc_kernels.cuh, pdl_wait).  After a kernel that never triggers, the launch is ordered as usual.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t st, Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

template <bool VEC, int THREADS, int SLOTS = kSlots>
int launch_k2(int grid, size_t smem, cudaStream_t st, const BinArgs& args, const double* E_true, const double* E_reco,
              const double* w0, const int8_t* channel, size_t n, double energy_scale, const double* bin_edges,
              int n_bins, int n_sub, const CallScratch& cs, double* hist_out)
{
    // the attribute is set once per instantiation and size (the call costs a microsecond of host time otherwise)
    static std::atomic<size_t> configured{0};
    if (smem > 48 * 1024 && configured.load(std::memory_order_relaxed) < smem) {
        CUDA_TRY(cudaFuncSetAttribute(reweight_bin_kernel<VEC, THREADS, SLOTS>,
                                      cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured.store(smem, std::memory_order_relaxed);
    }
    CUDA_TRY(launch_pdl(reweight_bin_kernel<VEC, THREADS, SLOTS>, grid, THREADS, smem, st, args, E_true, E_reco, w0, channel, n,
                        energy_scale, bin_edges, n_bins, n_sub, cs.ms, cs.table_cache, hist_out));
    return post_launch("osc_reweight_bin");
}

// Enqueue bin_setup + k2 for one parameter block.  hist_out is overwritten.
int launch_reweight(const BinArgs& args, const double* E_true, const double* E_reco, const double* w0,
                    const int8_t* channel, size_t n, double energy_scale, const double* bin_edges, int n_bins,
                    double* hist_out, cudaStream_t st)
{
    const size_t nh = (size_t)kChannels * n_bins;
    if (n == 0) {
        CUDA_TRY(cudaMemsetAsync(hist_out, 0, nh * sizeof(double), st));
        return OSC_OK;
    }
    int sms = 0;
    int rc = sm_count(&sms);
    if (rc) return rc;
    // ONE block per SM, as many warps as the sub-histograms leave room for (us per 1e7 events on a B200, end of round 2;
    // in brackets: round 1):
    //   up to ~140 bins   768 threads, a sub-histogram per (warp, event of the lane)   118-121 (129-138)
    //   up to ~213 bins   512 threads, same layout (122 registers, 5 % fewer instructions)   118-119 (138-140)
    //   up to ~425 bins   512 threads, ONE sub-histogram per warp (SLOTS = 1, lane_hist_single)   118-142 (139-155)
    //   up to ~570 bins   384 threads, one sub-histogram per warp   159-160 (170-174)
    //   up to 768 bins    256 threads, one sub-histogram per warp   224-228 (245-251)
    // (1 and 10 bins: 137 and 126 us -- every lane of a warp hits the same few cells.  The step from 118 us at 250 bins to
    // 133 us at 300 is not the launch shape: above ~280 uniform bins some cells of the 2048-cell look-up table straddle two
    // edges and the bin search takes its two-step form.)
    // Warp counts that are not a multiple of four per scheduler lose (576, 640, 704 threads: 145, 135, 138 us against
    // 129).  Why one block: co-resident blocks do not run at the same speed -- the warp schedulers favour the warps
    // that arrived first: with three blocks of 256 and equal shares of 44 tiles the first block of an SM needed
    // 85 us, the second 102 us and the third 127 us, and the SM spent the end of the kernel on 8 warps.  The warps of
    // ONE block are all the same age and finish together (measured: 137 -> 129 us per 1e7 events); a static
    // re-weighting of the shares does not work, the slot of a block on its SM is not known in advance.  (Several
    // blocks of 256 or 128 threads with two-slot sub-histograms remain reachable through
    // osc_set_k2_tuning for measurements: 147-230 us and 150-420 us over the same range of binnings.)
    int threads = 256, slots = 1;
    if (k2_smem_bytes(n_bins, 768, 1) + 1024 <= kSmemBudget) {
        threads = 768;
        slots = kSlots;
    } else if (k2_smem_bytes(n_bins, 512, 1) + 1024 <= kSmemBudget) {
        threads = 512;
        slots = kSlots;
    } else if (k2_smem_bytes(n_bins, 512, 1, 1) + 1024 <= kSmemBudget) {
        threads = 512;
    } else if (k2_smem_bytes(n_bins, 384, 1, 1) + 1024 <= kSmemBudget) {
        threads = 384;
    }
    const int t_threads = g_tune_threads.load(), t_slots = g_tune_slots.load(), t_nsub = g_tune_nsub.load();
    const int t_bps = g_tune_bps.load();
    if (t_slots) slots = t_slots == 1 ? 1 : kSlots;
    if (t_threads) {
        threads = t_threads;
        if (threads == 384) slots = 1;
    }
    // 256 threads: two sub-histograms per slot halve the collisions inside a warp; taken when 3 blocks still fit
    const int n_sub = (slots == kSlots && threads == 256 && 3 * (k2_smem_bytes(n_bins, 256, 2) + 1024) <= kSmemBudget) ? 2 : 1;
    int n_sub_t = n_sub;
    if (t_nsub) n_sub_t = slots == kSlots ? t_nsub : 1;
    const size_t smem = k2_smem_bytes(n_bins, threads, n_sub_t, slots);
    if (smem + 1024 > (size_t)227 * 1024)
        return fail(OSC_ERR_INVALID_ARG, "%d bins with %d threads and %d slot(s) need %zu bytes of shared memory", n_bins,
                    threads, slots, smem);
    size_t per_sm = kSmemBudget / (smem + 1024);
    if (t_bps) per_sm = (size_t)t_bps;
    if (per_sm < 1) per_sm = 1;
    const size_t max_per_sm = threads >= 384 ? 1 : threads == 256 ? 3 : 6;   // __launch_bounds__(THREADS, 768 / THREADS) of k2
    if (per_sm > max_per_sm && !t_bps) per_sm = max_per_sm;
    const size_t ntiles = (n + 2 * threads - 1) / (2 * (size_t)threads);
    if (ntiles > 0xFFFFFFFFull) return fail(OSC_ERR_INVALID_ARG, "n = %zu events is more than one call takes (2^32 tiles)", n);
    size_t g = (size_t)sms * per_sm;
    if (ntiles < g) g = ntiles;
    const int grid = (int)g;

    ScratchLease lease;
    if ((rc = stream_scratch(merge_scratch_bytes(grid, nh), st, lease))) return rc;
    const CallScratch ms = call_scratch(lease.p, grid, nh);

    const bool vec = aligned(E_true, 16) && aligned(E_reco, 16) && aligned(w0, 16) && aligned(channel, 2);
#define OSC_K2_SINGLE(T)                                                                                               \
    if (slots == 1 && threads == T)                                                                                    \
        return vec ? launch_k2<true, T, 1>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale,         \
                                           bin_edges, n_bins, 1, ms, hist_out)                                         \
                   : launch_k2<false, T, 1>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale,        \
                                            bin_edges, n_bins, 1, ms, hist_out);
    OSC_K2_SINGLE(512) OSC_K2_SINGLE(384) OSC_K2_SINGLE(256)
#undef OSC_K2_SINGLE
    if (slots == 1) return fail(OSC_ERR_INVALID_ARG, "single-slot k2 is built for 256, 384 and 512 threads");
    if (threads == 768)
        return vec ? launch_k2<true, 768>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                          n_bins, n_sub_t, ms, hist_out)
                   : launch_k2<false, 768>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                           n_bins, n_sub_t, ms, hist_out);
    if (threads == 512)
        return vec ? launch_k2<true, 512>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                          n_bins, n_sub_t, ms, hist_out)
                   : launch_k2<false, 512>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                           n_bins, n_sub_t, ms, hist_out);
    if (threads == 256)
        return vec ? launch_k2<true, 256>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                          n_bins, n_sub_t, ms, hist_out)
                   : launch_k2<false, 256>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                           n_bins, n_sub_t, ms, hist_out);
    return vec ? launch_k2<true, 128>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                      n_bins, n_sub_t, ms, hist_out)
               : launch_k2<false, 128>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                       n_bins, n_sub_t, ms, hist_out);
}

// Threads per block of k2s, 512 / kScalesThreads blocks per SM (126-128 registers either way).  1e7 events x 3 scales, in
// the order the kernel changed: as round 2 began 2 x 256 threads 242.5 us, 1 x 512 268.3 us; with the loop constants in
// registers 198.0 / 193.9; with gridDim.x in a register as well 190.0 / 182.2 (1e8 events: 1753 / 1694 us, 1e6: 32.8 /
// 30.4) -- once the warps no longer wait for constants, one block (half the partial sums to merge, all warps the same age)
// is ahead, as it is for k2.  2 x 320 and 1 x 640 threads (96 registers): 198.1 / 195.4 us.
constexpr int kScalesThreads = 512;
constexpr int kScalesBlocksPerSM = 512 / kScalesThreads;

template <bool VEC, int NS>
int launch_k2s(int grid, size_t smem, cudaStream_t st, const BinArgs& args, const ScaleArgs& sc, const double* E_true,
               const double* E_reco, const double* w0, const int8_t* channel, size_t n, const double* bin_edges,
               int n_bins, int n_sub, const CallScratch& cs, double* hist_out)
{
    static std::atomic<size_t> configured{0};
    if (configured.load(std::memory_order_relaxed) < smem) {
        CUDA_TRY(cudaFuncSetAttribute(reweight_bin_scales_kernel<VEC, kScalesThreads, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)smem));
        configured.store(smem, std::memory_order_relaxed);
    }
    CUDA_TRY(launch_pdl(reweight_bin_scales_kernel<VEC, kScalesThreads, NS>, grid, kScalesThreads, smem, st, args, sc, E_true, E_reco, w0, channel, n,
                        bin_edges, n_bins, n_sub, cs.ms, cs.table_cache, hist_out));
    return post_launch("osc_reweight_bin_scales");
}

// k2s for n_scales in [2, kMaxScales]; returns 1 (not an error code) when the sub-histograms of all scales do not
// fit the shared memory of one SM twice, in which case the caller runs one k2 pass per scale.
int launch_reweight_scales(const BinArgs& args, const double* E_true, const double* E_reco, const double* w0,
                           const int8_t* channel, size_t n, const double* scales, int n_scales,
                           const double* bin_edges, int n_bins, double* hist_out, cudaStream_t st)
{
    const size_t nht = (size_t)n_scales * kChannels * n_bins;
    const size_t fixed = sizeof(double) * kBinArgsDoubles + bin_table_bytes(n_bins);
    const size_t sub1 = sizeof(double) * (kScalesThreads / 32) * kSlots * nht;
    if (kScalesBlocksPerSM * (fixed + sub1 + 1024) > kSmemBudget) return 1;
    const int n_sub = kScalesBlocksPerSM * (fixed + 2 * sub1 + 1024) <= kSmemBudget ? 2 : 1;
    const size_t smem = fixed + n_sub * sub1;
    int sms = 0;
    int rc = sm_count(&sms);
    if (rc) return rc;
    const size_t ntiles = (n + 2 * kScalesThreads - 1) / (2 * kScalesThreads);
    if (ntiles > 0xFFFFFFFFull) return fail(OSC_ERR_INVALID_ARG, "n = %zu events is more than one call takes (2^32 tiles)", n);
    size_t g = (size_t)sms * kScalesBlocksPerSM;
    if (ntiles < g) g = ntiles;
    const int grid = (int)g;
    ScratchLease lease;
    if ((rc = stream_scratch(merge_scratch_bytes(grid, nht), st, lease))) return rc;
    const CallScratch ms = call_scratch(lease.p, grid, nht);
    ScaleArgs sc;
    for (int k = 0; k < kMaxScales; ++k) sc.s[k] = k < n_scales ? scales[k] : 1.0;
    const bool vec = aligned(E_true, 16) && aligned(E_reco, 16) && aligned(w0, 16) && aligned(channel, 2);
#define OSC_K2S(NS)                                                                                                  \
    return vec ? launch_k2s<true, NS>(grid, smem, st, args, sc, E_true, E_reco, w0, channel, n, bin_edges, n_bins, \
                                      n_sub, ms, hist_out)                                                           \
               : launch_k2s<false, NS>(grid, smem, st, args, sc, E_true, E_reco, w0, channel, n, bin_edges, n_bins, \
                                       n_sub, ms, hist_out)
    switch (n_scales) {
    case 2: OSC_K2S(2);
    case 3: OSC_K2S(3);
    default: OSC_K2S(4);
    }
#undef OSC_K2S
}

// Device staging buffers of the *_host entry points (grown on demand, reused between calls).
constexpr int kHostChunks = 8;                 // chunks a host call's events cross PCIe in, at most
constexpr size_t kHostChunkMin = 1u << 20;     // events per chunk, at least (a kernel launch per chunk: 7 us of fixed cost)
struct HostPath {
    std::mutex mu;
    cudaStream_t stream = nullptr;             // kernels, small copies
    cudaStream_t copy_stream = nullptr;        // the event arrays, chunk after chunk
    cudaEvent_t chunk_ready[kHostChunks] = {};
    char* buf = nullptr;
    size_t cap = 0;
    int ensure(size_t bytes)
    {
        if (!stream) CUDA_TRY(cudaStreamCreateWithFlags(&stream, cudaStreamNonBlocking));
        if (!copy_stream) {
            CUDA_TRY(cudaStreamCreateWithFlags(&copy_stream, cudaStreamNonBlocking));
            for (int c = 0; c < kHostChunks; ++c) CUDA_TRY(cudaEventCreateWithFlags(&chunk_ready[c], cudaEventDisableTiming));
        }
        if (bytes > cap) {
            if (buf) CUDA_TRY(cudaFree(buf));
            buf = nullptr;
            cap = 0;
            CUDA_TRY(cudaMalloc((void**)&buf, bytes));
            cap = bytes;
        }
        return OSC_OK;
    }
};
HostPath g_hosts[64];          // one per device: a stream and a cudaMalloc'd buffer belong to the device they were made on

int host_path(HostPath** out)
{
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(OSC_ERR_CUDA, "device index %d out of range", dev);
    *out = &g_hosts[dev];
    return OSC_OK;
}

} // namespace

extern "C" {

int osc_set_params(double sin2_th12, double sin2_th23, double sin2_th13, double dm2_32, double dm2_21,
                   double delta_cp, double rho_g_cm3, double L_km, int hierarchy)
{
    osc_params p;
    p.sin2_th12 = sin2_th12;
    p.sin2_th23 = sin2_th23;
    p.sin2_th13 = sin2_th13;
    p.dm2_32 = dm2_32;
    p.dm2_21 = dm2_21;
    p.delta_cp = delta_cp;
    p.rho_g_cm3 = rho_g_cm3;
    p.L_km = L_km;
    p.hierarchy = hierarchy;
    if (const char* msg = check_params(p)) return fail(OSC_ERR_INVALID_ARG, "osc_set_params: %s", msg);
    HostSet h;
    precompute(p, h);
    std::lock_guard<std::mutex> lk(g_mu);
    g_state = h;
    g_configured = true;
    return OSC_OK;
}

int osc_prob(const double* E_true, size_t n, int flavour_in, int flavour_out, int antinu, double* P_out, void* stream)
{
    int rc;
    if ((rc = check_flavour(flavour_in, "flavour_in")) || (rc = check_flavour(flavour_out, "flavour_out"))) return rc;
    if (antinu != 0 && antinu != 1) return fail(OSC_ERR_INVALID_ARG, "antinu must be 0 or 1");
    HostSet h;
    if ((rc = snapshot(h))) return rc;
    if (n == 0) return OSC_OK;
    if (!E_true || !P_out) return fail(OSC_ERR_INVALID_ARG, "null array with n > 0");
    if (!aligned(E_true, 8) || !aligned(P_out, 8)) return fail(OSC_ERR_ALIGNMENT, "fp64 array not 8-byte aligned");
    ProbArgs a;
    a.set = h.set;
    a.tr = make_trans(h, flavour_in, flavour_out, antinu);
    const size_t npairs = (n + 1) / 2;
    // one block of kBlockProb threads per SM once every SM gets two full iterations of it; below that, blocks of
    // kBlock threads spread the events over more SMs (configs[0]: 1e5 events)
    int sms = 0;
    if ((rc = sm_count(&sms))) return rc;
    const bool big = npairs >= (size_t)2 * sms * kBlockProb;
    int grid = 1;
    if ((rc = big ? grid_for((npairs + kBlockProb - 1) / kBlockProb, &grid, 1)
                  : grid_for((npairs + kBlock - 1) / kBlock, &grid)))
        return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // the element of S that is asked for is known here: 1 (e, e), 2 another diagonal element, 3 off-diagonal
    const int kind = flavour_in != flavour_out ? 3 : (flavour_in == 0 ? 1 : 2);
#define OSC_K1(VEC, T)                                                                    \
    switch (kind) {                                                                       \
    case 1: prob_kernel<VEC, 1, T><<<grid, T, 0, st>>>(a, E_true, n, P_out); break;       \
    case 2: prob_kernel<VEC, 2, T><<<grid, T, 0, st>>>(a, E_true, n, P_out); break;       \
    default: prob_kernel<VEC, 3, T><<<grid, T, 0, st>>>(a, E_true, n, P_out); break;      \
    }
    const bool vec = aligned(E_true, 16) && aligned(P_out, 16);
    if (big) {
        if (vec) { OSC_K1(true, kBlockProb) } else { OSC_K1(false, kBlockProb) }
    } else {
        if (vec) { OSC_K1(true, kBlock) } else { OSC_K1(false, kBlock) }
    }
#undef OSC_K1
    return post_launch("osc_prob");
}

int osc_prob_all(const double* E_true, size_t n, int antinu, double* P_out, void* stream)
{
    int rc;
    if (antinu != 0 && antinu != 1) return fail(OSC_ERR_INVALID_ARG, "antinu must be 0 or 1");
    HostSet h;
    if ((rc = snapshot(h))) return rc;
    if (n == 0) return OSC_OK;
    if (!E_true || !P_out) return fail(OSC_ERR_INVALID_ARG, "null array with n > 0");
    if (!aligned(E_true, 8) || !aligned(P_out, 8)) return fail(OSC_ERR_ALIGNMENT, "fp64 array not 8-byte aligned");
    ProbAllArgs a;
    a.set = h.set;
    for (int beta = 0; beta < 2; ++beta)
        for (int alpha = 0; alpha < 2; ++alpha) a.tr[2 * beta + alpha] = make_trans(h, alpha, beta, antinu);
    // launch shape as osc_prob: one block of kBlockProbAll threads per SM once every SM gets two full iterations of it,
    // blocks of kBlock threads below that; 128-bit accesses when E_true and every row of P_out are 16-byte aligned
    const size_t npairs = (n + 1) / 2;
    int sms = 0;
    if ((rc = sm_count(&sms))) return rc;
    constexpr int kT = kBlockProbAll;
    const bool big = npairs >= (size_t)2 * sms * kT;
    int grid = 1;
    if ((rc = big ? grid_for((npairs + kT - 1) / kT, &grid, 1)
                  : grid_for((npairs + kBlock - 1) / kBlock, &grid)))
        return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const bool vec = aligned(E_true, 16) && aligned(P_out, 16) && n % 2 == 0;
    if (big) {
        if (vec) CUDA_TRY(launch_pdl(prob_all_kernel<true, kT>, grid, kT, 0, st, a, E_true, n, P_out));
        else CUDA_TRY(launch_pdl(prob_all_kernel<false, kT>, grid, kT, 0, st, a, E_true, n, P_out));
    } else {
        if (vec) CUDA_TRY(launch_pdl(prob_all_kernel<true, kBlock>, grid, kBlock, 0, st, a, E_true, n, P_out));
        else CUDA_TRY(launch_pdl(prob_all_kernel<false, kBlock>, grid, kBlock, 0, st, a, E_true, n, P_out));
    }
    return post_launch("osc_prob_all");
}

int osc_reweight_bin(const double* E_true, const double* E_reco, const double* w0, const int8_t* channel, size_t n,
                     double energy_scale, const double* bin_edges, int n_bins, double* hist_out, void* stream)
{
    int rc = check_bin_args(E_true, E_reco, w0, channel, n, energy_scale, bin_edges, n_bins, hist_out);
    if (rc) return rc;
    if (n > 0 && !w0) return fail(OSC_ERR_INVALID_ARG, "null w0 with n > 0");
    if (!aligned(hist_out, 8)) return fail(OSC_ERR_ALIGNMENT, "hist_out not 8-byte aligned");
    HostSet h;
    if ((rc = snapshot(h))) return rc;
    BinArgs args;
    make_bin_args(h, args);
    return launch_reweight(args, E_true, E_reco, w0, channel, n, energy_scale, bin_edges, n_bins, hist_out,
                           static_cast<cudaStream_t>(stream));
}

// ------------------------------------------------------------------------------------------------
// osc_reweight_bin_static: osc_reweight_bin for callers that must not allocate (stream capture, serving loops,
// harnesses that forbid cudaMalloc).  The scratch of k2 -- ticket counters, bin-table cache, block partials -- lives in
// a file-scope __device__ array instead of the per-stream scratch the library otherwise allocates on first use.  Every
// GPU that loads the library holds the array (1.08 MB) until the process exits; every call shares it.
// ------------------------------------------------------------------------------------------------
namespace {

constexpr int kStaticMaxBins = 128;    // the binnings k2 takes with its widest block (768 threads, two slots per warp)
constexpr int kStaticMaxGrid = 256;    // blocks: one per SM, clamped
constexpr size_t kStaticScratchBytes =
    kScratchHead + (size_t)(kStaticMaxGrid + (kStaticMaxGrid + kGroup - 1) / kGroup) * kChannels * kStaticMaxBins * sizeof(double);

} // namespace

// In host code this name is a host-side stand-in for the symbol, not a device address: the address the kernels get is
// taken with cudaGetSymbolAddress below.  Zero-initialised when the module is loaded.
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

namespace {

// Device address of g_static_scratch on the current device (taken once per device, with that device current).
int static_scratch(char** out)
{
    static std::atomic<char*> ptr[64];
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(OSC_ERR_CUDA, "device index %d out of range", dev);
    char* p = ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        void* q = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&q, g_static_scratch);
        if (e != cudaSuccess || !q)
            return fail(OSC_ERR_CUDA, "cudaGetSymbolAddress(g_static_scratch) on device %d: %s", dev, cudaGetErrorString(e));
        p = static_cast<char*>(q);
        ptr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return OSC_OK;
}

} // namespace

int osc_reweight_bin_static(const double* E_true, const double* E_reco, const double* w0, const int8_t* channel, size_t n,
                            double energy_scale, const double* bin_edges, int n_bins, double* hist_out, void* stream)
{
    int rc = check_bin_args(E_true, E_reco, w0, channel, n, energy_scale, bin_edges, n_bins, hist_out);
    if (rc) return rc;
    if (n_bins > kStaticMaxBins)
        return fail(OSC_ERR_INVALID_ARG, "osc_reweight_bin_static: n_bins = %d is more than the %d bins its static scratch "
                                         "(%zu bytes per GPU) is laid out for; use osc_reweight_bin", n_bins, kStaticMaxBins,
                    kStaticScratchBytes);
    if (n > 0 && !w0) return fail(OSC_ERR_INVALID_ARG, "null w0 with n > 0");
    if (!aligned(hist_out, 8)) return fail(OSC_ERR_ALIGNMENT, "hist_out not 8-byte aligned");
    HostSet h;
    if ((rc = snapshot(h))) return rc;
    BinArgs args;
    make_bin_args(h, args);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t nh = (size_t)kChannels * n_bins;
    if (n == 0) {
        CUDA_TRY(cudaMemsetAsync(hist_out, 0, nh * sizeof(double), st));
        return OSC_OK;
    }
    constexpr int THREADS = 768;
    const size_t smem = k2_smem_bytes(n_bins, THREADS, 1);
    if (smem + 1024 > kSmemBudget)
        return fail(OSC_ERR_INVALID_ARG, "internal: %d bins do not fit the 768-thread layout of k2", n_bins);
    int sms = 0;
    if ((rc = sm_count(&sms))) return rc;
    const size_t ntiles = (n + 2 * THREADS - 1) / (2 * (size_t)THREADS);
    if (ntiles > 0xFFFFFFFFull) return fail(OSC_ERR_INVALID_ARG, "n = %zu events is more than one call takes (2^32 tiles)", n);
    size_t g = std::min<size_t>((size_t)sms, (size_t)kStaticMaxGrid);
    if (ntiles < g) g = ntiles;
    const int grid = (int)g;
    if (merge_scratch_bytes(grid, nh) > kStaticScratchBytes)
        return fail(OSC_ERR_INVALID_ARG, "internal: static scratch too small for %d blocks x %zu cells", grid, nh);
    char* scratch = nullptr;
    if ((rc = static_scratch(&scratch))) return rc;
    // the array keeps what the last call left: the ticket counters must start at zero (a call that failed on the device
    // may have left them set); the bin-table cache is validated against the edges by the kernel, the partials are
    // written before they are read
    CUDA_TRY(cudaMemsetAsync(scratch, 0, kCounterBytes, st));
    const CallScratch cs = call_scratch(scratch, grid, nh);
    const bool vec = aligned(E_true, 16) && aligned(E_reco, 16) && aligned(w0, 16) && aligned(channel, 2);
    return vec ? launch_k2<true, THREADS>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                          n_bins, 1, cs, hist_out)
               : launch_k2<false, THREADS>(grid, smem, st, args, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                           n_bins, 1, cs, hist_out);
}

namespace {

// Pinned staging for host-built tables that a batched call uploads: a small ring of page-locked buffers, each
// fenced by an event recorded after the copy that reads it, so that the upload is a true asynchronous copy (a
// pageable source makes cudaMemcpyAsync wait for the stream) and the call returns while earlier work still runs.
struct PinnedRing {
    static constexpr int kSlots = 4;
    struct Slot {
        void* host = nullptr;
        size_t cap = 0;
        cudaEvent_t ev = nullptr;
        bool in_flight = false;
    };
    Slot slot[kSlots];
    int next = 0;
    std::mutex mu;

    // `lk` stays locked until the caller has filled the slot, enqueued the copy that reads it and called fence():
    // a concurrent caller cannot be handed a slot that is still being filled.
    int acquire(size_t bytes, Slot** out, std::unique_lock<std::mutex>& lk)
    {
        lk = std::unique_lock<std::mutex>(mu);
        Slot& s = slot[next];
        next = (next + 1) % kSlots;
        if (s.in_flight) {
            CUDA_TRY(cudaEventSynchronize(s.ev));
            s.in_flight = false;
        }
        if (!s.ev) CUDA_TRY(cudaEventCreateWithFlags(&s.ev, cudaEventDisableTiming));
        if (s.cap < bytes) {
            if (s.host) CUDA_TRY(cudaFreeHost(s.host));
            s.host = nullptr;
            s.cap = 0;
            const size_t cap = round_up(bytes + bytes / 2, 1 << 16);
            CUDA_TRY(cudaMallocHost(&s.host, cap));
            s.cap = cap;
        }
        *out = &s;
        return OSC_OK;
    }
    int fence(Slot* s, cudaStream_t st)
    {
        CUDA_TRY(cudaEventRecord(s->ev, st));
        s->in_flight = true;
        return OSC_OK;
    }
};
PinnedRing g_rings[64];        // one per device: an event belongs to the device it was created on

int ring_for_device(PinnedRing** out)
{
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(OSC_ERR_CUDA, "device index %d out of range", dev);
    *out = &g_rings[dev];
    return OSC_OK;
}

} // namespace

// ------------------------------------------------------------------------------------------------
// k4 (osc_scan.cuh): host side of the factorised batched call.
// ------------------------------------------------------------------------------------------------
namespace {

typedef std::array<unsigned long long, 7> GroupKey;

unsigned long long bits_of(double v)
{
    unsigned long long b;
    std::memcpy(&b, &v, sizeof b);
    return b;
}

// Everything S' depends on; theta23 and delta_cp are what may differ inside a group.
GroupKey group_key(const osc_params& p)
{
    return GroupKey{bits_of(p.sin2_th12), bits_of(p.sin2_th13), bits_of(p.dm2_32), bits_of(p.dm2_21),
                    bits_of(p.rho_g_cm3), bits_of(p.L_km), (unsigned long long)(long long)p.hierarchy};
}

struct ScanPlan {
    std::vector<ScanGroup> groups;
    std::vector<ScanSub> subs;
    std::vector<ScanConstArgs> consts;   // subs[s] as the parameter block of scan_const_kernel (when const_ok)
    bool const_ok = false;               // every channel of every group is one of the two kinds that kernel is built for
    std::vector<std::array<std::complex<double>, kChannels * kScanElems>> coef;   // c_k of every point and channel
};

// Index sets of the rows of W = R23 D: row e touches column 0 only, rows mu and tau columns 1 and 2.
int w_cols(int flavour, int out[2])
{
    if (flavour == 0) {
        out[0] = 0;
        return 1;
    }
    out[0] = 1;
    out[1] = 2;
    return 2;
}

// Sub-group s of the plan as the parameter block of scan_const_kernel (osc_scan.cuh).  The rows of W have unit length,
// which takes one term off each kind of channel:
//   three entries (numu -> numu): coefficients a, b on two diagonal entries z_a, z_b of S' and c on an off-diagonal
//     entry z_c, all real, a + b = 1:  |a z_a + b z_b + c z_c|^2 = |s + a u + c v|^2 with s = z_b, u = z_a - z_b, v = z_c
//     = |s|^2 + a^2 |u|^2 + c^2 |v|^2 + 2a Re(s u*) + 2c Re(s v*) + 2ac Re(u v*);  u is the amplitude of the
//     pseudo-entry el_a - el_b (every field of ScanElem enters the amplitude linearly, and its delta is 0);
//   two entries (numu -> nue): |c0|^2 + |c1|^2 = 1:  |c0 z0 + c1 z1|^2
//     = |z1|^2 + |c0|^2 (|z0|^2 - |z1|^2) + 2 Re(c0 c1*) Re(z0 z1*) - 2 Im(c0 c1*) Im(z0 z1*).
// The first term of each does not depend on the point: the kernel sums it once per event.  false: a channel is of
// neither kind (the caller keeps to scan_main_kernel, which takes any term list).
bool make_const_args(const ScanPlan& plan, size_t s, ScanConstArgs& a)
{
    const ScanSub& sub = plan.subs[s];
    const ScanGroup& g = plan.groups[(size_t)sub.group];
    std::memset(&a, 0, sizeof a);
    a.set = g.set;
    for (int l = 0; l < kScanLanes; ++l) a.pt[l] = sub.pt[l];
    const double UNIT = 8 * std::numeric_limits<double>::epsilon();
    for (int c = 0; c < kChannels; ++c) {
        const ScanChan& gc = g.ch[c];
        ScanChan& ac = a.ch[c];
        ac.sa = gc.sa;
        ac.nk = gc.nk;
        for (int k = 0; k < gc.nk; ++k)
            if (gc.el[k].ee != 0.0) return false;
        if (gc.nk == 3) {
            int d[3], nd = 0, o = -1;
            for (int k = 0; k < 3; ++k) {
                if (gc.el[k].delta != 0.0) d[nd++] = k;
                else o = k;
            }
            if (nd != 2 || o < 0) return false;
            a.mm |= 1 << c;
            ac.el[0] = gc.el[d[1]];                                         // s = z_b
            ac.el[1].delta = 0.0;                                           // u = z_a - z_b
            ac.el[1].ee = 0.0;
            ac.el[1].Tr0 = gc.el[d[0]].Tr0 - gc.el[d[1]].Tr0;
            ac.el[1].T2r0 = gc.el[d[0]].T2r0 - gc.el[d[1]].T2r0;
            ac.el[1].T2r1 = gc.el[d[0]].T2r1 - gc.el[d[1]].T2r1;
            ac.el[2] = gc.el[o];                                            // v = z_c
            for (int l = 0; l < kScanLanes; ++l) {
                if (sub.pt[l] < 0) continue;
                const std::complex<double>* ck = &plan.coef[(size_t)sub.pt[l]][(size_t)c * kScanElems];
                if (ck[0].imag() != 0.0 || ck[1].imag() != 0.0 || ck[2].imag() != 0.0) return false;
                const double ca = ck[d[0]].real(), cb = ck[d[1]].real(), cc = ck[o].real();
                if (std::fabs(ca + cb - 1.0) > UNIT) return false;
                a.mono[c][0][l] = ca * ca;
                a.mono[c][1][l] = cc * cc;
                a.mono[c][2][l] = 2.0 * ca;
                a.mono[c][3][l] = 2.0 * cc;
                a.mono[c][4][l] = 2.0 * ca * cc;
            }
        } else if (gc.nk == 2) {
            if (gc.el[0].delta != 0.0 || gc.el[1].delta != 0.0) return false;
            ac.el[0] = gc.el[0];
            ac.el[1] = gc.el[1];
            for (int l = 0; l < kScanLanes; ++l) {
                if (sub.pt[l] < 0) continue;
                const std::complex<double>* ck = &plan.coef[(size_t)sub.pt[l]][(size_t)c * kScanElems];
                if (std::fabs(std::norm(ck[0]) + std::norm(ck[1]) - 1.0) > UNIT) return false;
                const std::complex<double> x = ck[0] * std::conj(ck[1]);
                a.mono[c][0][l] = std::norm(ck[0]);
                a.mono[c][1][l] = 2.0 * x.real();
                a.mono[c][2][l] = -2.0 * x.imag();
            }
        } else {
            return false;
        }
        for (int t = 0; t < kConstTerms; ++t)
            for (int l = 0; l < kScanLanes; ++l)
                if (a.mono[c][t][l] != 0.0) ac.tmask |= 1 << t;
    }
    return true;
}

void build_scan_plan(const osc_params* points, int n_points, ScanPlan& plan)
{
    typedef std::complex<double> cd;
    std::map<GroupKey, int> index;
    std::vector<std::vector<int>> members;
    for (int p = 0; p < n_points; ++p) {
        const GroupKey k = group_key(points[p]);
        auto it = index.find(k);
        if (it == index.end()) {
            it = index.emplace(k, (int)members.size()).first;
            members.emplace_back();
        }
        members[(size_t)it->second].push_back(p);
    }
    plan.groups.assign(members.size(), ScanGroup());
    plan.subs.clear();
    plan.coef.assign((size_t)n_points, {});
    for (size_t g = 0; g < members.size(); ++g) {
        // T' of the group: the precompute with theta23 = 0, delta = 0 gives U = R13 R12
        osc_params q = points[members[g][0]];
        q.sin2_th23 = 0.0;
        q.delta_cp = 0.0;
        HostSet h;
        precompute(q, h);
        ScanGroup& sg = plan.groups[g];
        std::memset(&sg, 0, sizeof sg);
        sg.set = h.set;
        int el_i[kChannels][kScanElems], el_j[kChannels][kScanElems];
        for (int c = 0; c < kChannels; ++c) {
            int fin, fout, anti;
            channel_def(c, fin, fout, anti);
            int ci[2], cj[2];
            const int ni = w_cols(fout, ci), nj = w_cols(fin, cj);
            int nk = 0;
            for (int a = 0; a < ni; ++a)
                for (int b = 0; b < nj; ++b) {
                    const int i = ci[a] < cj[b] ? ci[a] : cj[b], j = ci[a] < cj[b] ? cj[b] : ci[a];
                    bool seen = false;
                    for (int k = 0; k < nk; ++k) seen = seen || (el_i[c][k] == i && el_j[c][k] == j);
                    if (!seen) {
                        el_i[c][nk] = i;
                        el_j[c][nk] = j;
                        ++nk;
                    }
                }
            ScanChan& sc = sg.ch[c];
            sc.nk = nk;
            sc.tmask = 0;
            for (int k = 0; k < nk; ++k) {
                const OscTrans t = make_trans(h, el_j[c][k], el_i[c][k], anti);   // entry (i, j): alpha = j, beta = i
                sc.sa = t.sa;
                sc.el[k].delta = t.delta;
                sc.el[k].ee = t.ee;
                sc.el[k].Tr0 = t.Tr0;
                sc.el[k].T2r0 = t.T2r0;
                sc.el[k].T2r1 = t.T2r1;
            }
        }
        // coefficients c_k = C_ij = W_{beta i} conj(W_{alpha j}) (+ C_ji for i != j) of every point, and from them the
        // monomials of |sum_k c_k z_k|^2 in the canonical term order of osc_scan.cuh
        const std::vector<int>& mem = members[g];
        std::vector<std::array<double, kChannels * kScanTerms>> mono(mem.size());
        for (size_t q = 0; q < mem.size(); ++q) {
            const osc_params& pp = points[mem[q]];
            const double s23 = std::sqrt(pp.sin2_th23), c23 = std::sqrt(1.0 - pp.sin2_th23);
            for (int c = 0; c < kChannels; ++c) {
                int fin, fout, anti;
                channel_def(c, fin, fout, anti);
                const double d = anti ? -pp.delta_cp : pp.delta_cp;          // antineutrinos: W -> conj(W)
                const cd ep(std::cos(d), std::sin(d));
                const cd W[3][3] = {{cd(1.0), cd(0.0), cd(0.0)}, {cd(0.0), cd(c23), s23 * ep}, {cd(0.0), cd(-s23), c23 * ep}};
                cd ck[kScanElems] = {cd(0.0), cd(0.0), cd(0.0)};
                for (int k = 0; k < sg.ch[c].nk; ++k) {
                    const int i = el_i[c][k], j = el_j[c][k];
                    ck[k] = W[fout][i] * std::conj(W[fin][j]);
                    if (i != j) ck[k] += W[fout][j] * std::conj(W[fin][i]);
                }
                for (int k = 0; k < kScanElems; ++k) plan.coef[(size_t)mem[q]][(size_t)c * kScanElems + k] = ck[k];
                double* mo = &mono[q][(size_t)c * kScanTerms];
                static const int PK[3] = {0, 0, 1}, PL[3] = {1, 2, 2};
                for (int k = 0; k < 3; ++k) mo[k] = std::norm(ck[k]);
                for (int r = 0; r < 3; ++r) {
                    const cd x = ck[PK[r]] * std::conj(ck[PL[r]]);
                    mo[3 + r] = 2.0 * x.real();
                    mo[6 + r] = -2.0 * x.imag();
                }
                for (int t = 0; t < kScanTerms; ++t)
                    if (mo[t] != 0.0) sg.ch[c].tmask |= 1 << t;
            }
        }
        // sub-groups of at most 32 points; the used terms of a channel are stored compacted, in canonical order
        for (size_t first = 0; first < mem.size(); first += kScanLanes) {
            plan.subs.emplace_back();
            ScanSub& sub = plan.subs.back();
            std::memset(&sub, 0, sizeof sub);
            sub.group = (int)g;
            for (int l = 0; l < kScanLanes; ++l) sub.pt[l] = -1;
            for (int l = 0; l < kScanLanes && first + l < mem.size(); ++l) {
                sub.pt[l] = mem[first + l];
                for (int c = 0; c < kChannels; ++c) {
                    int tt = 0;
                    for (int t = 0; t < kScanTerms; ++t)
                        if (sg.ch[c].tmask & (1 << t)) sub.mono[c][tt++][l] = mono[first + l][(size_t)c * kScanTerms + t];
                }
            }
        }
    }
    plan.consts.resize(plan.subs.size());
    plan.const_ok = true;
    for (size_t s = 0; s < plan.subs.size() && plan.const_ok; ++s) plan.const_ok = make_const_args(plan, s, plan.consts[s]);
}

// Events sorted by histogram cell and cut into pieces (osc_scan.cuh): what k4 and k5 work on.  The buffers belong
// either to the stream-ordered scratch of one batched call or to an osc_plan.
struct SortedEvents {
    ScanGeom geo;              // range, nranges, piece, max_units, ncells (nsubs / subs_per_slot are set per run)
    int n_bins = 0;
    size_t n = 0;
    unsigned int* cell_begin = nullptr;
    unsigned int* unit_begin = nullptr;
    unsigned short* unit_cell = nullptr;   // [max_units]
    double* sEt = nullptr;
    double* sW = nullptr;
};

size_t sorted_bytes_cells(int ncells) { return round_up((size_t)(ncells + 1) * sizeof(unsigned int), 256); }
size_t sorted_bytes_events(size_t n) { return round_up(n * sizeof(double), 256); }
size_t sorted_bytes_units(unsigned max_units) { return round_up((size_t)max_units * sizeof(unsigned short), 256); }

// Geometry of the sort for n events; `piece` as the caller wants it (multiple of 64).
int sorted_geometry(size_t n, int n_bins, size_t piece, ScanGeom& geo)
{
    if (n >= 0xFFFFFFFFull - 64) return fail(OSC_ERR_INVALID_ARG, "n = %zu events is more than one batched call takes", n);
    geo.ncells = kChannels * n_bins;
    geo.nsubs = 0;
    geo.subs_per_slot = 0;
    // warp ranges of the sort passes: short enough to give every SM dozens of warps (the passes are latency-bound),
    // long enough to keep the [ncells][nranges] count table below 64 MB
    const size_t max_ranges = std::min<size_t>(16384, (64u << 20) / (sizeof(unsigned int) * (size_t)geo.ncells));
    geo.range = round_up(std::max<size_t>(256, (n + max_ranges - 1) / max_ranges), 32);
    if (geo.ncells <= kSortMaxCells) {
        // block-local sort (sort_count_kernel / sort_scatter_kernel): a block sorts a chunk of `range` events in shared
        // memory; chunks short enough to give every SM a few blocks, long enough for runs of whole sectors per cell
        int sms = 0;
        int rc = sm_count(&sms);
        if (rc) return rc;
        // chunk = 512 * STEPS events with STEPS in {2, 4, 8} (sort_scatter_kernel<STEPS>)
        size_t chunk = g_sort_chunk.load();
        while (chunk > 1024 && n / chunk < (size_t)sms * 4) chunk /= 2;
        while (chunk < 4096 && (n + chunk - 1) / chunk > max_ranges) chunk *= 2;
        geo.range = chunk;
    }
    geo.nranges = (unsigned)((n + geo.range - 1) / geo.range);
    geo.piece = (unsigned)piece;
    geo.max_units = (unsigned)(n / piece + (size_t)geo.ncells + 1);
    return OSC_OK;
}

// Kind of the element of S each channel asks for (assemble_kind in osc_core.cuh): 1 (e, e), 2 another diagonal
// element, 3 off-diagonal.
ChannelKinds channel_kinds()
{
    ChannelKinds kinds;
    for (int c = 0; c < kChannels; ++c) {
        int fin, fout, anti;
        channel_def(c, fin, fout, anti);
        kinds.k[c] = fin != fout ? 3 : (fin == 0 ? 1 : 2);
    }
    return kinds;
}

// The three sort passes.  se's buffers are assigned by the caller; the temporaries come from a stream-ordered scratch.
int scan_sort(const SortedEvents& se, const double* E_true, const double* E_reco, const double* w0, const int8_t* channel,
              double energy_scale, const double* bin_edges, cudaStream_t st)
{
    int rc;
    const ScanGeom& geo = se.geo;
    const size_t b_cellid = round_up(se.n * sizeof(unsigned short), 256);
    const size_t b_count = round_up((size_t)geo.ncells * geo.nranges * sizeof(unsigned int), 256);
    Scratch tmp;
    if ((rc = tmp.alloc(b_cellid + b_count, st))) return rc;
    unsigned short* cellid = reinterpret_cast<unsigned short*>(tmp.p);
    unsigned int* count = reinterpret_cast<unsigned int*>(tmp.p + b_cellid);
    int sms = 0;
    if ((rc = sm_count(&sms))) return rc;
    if (geo.ncells <= kSortMaxCells) {
        // block-local sort: cell ids and per-(cell, chunk) counts, offsets, then the scatter through shared memory
        const size_t smem_c = bin_table_bytes(se.n_bins) + sizeof(unsigned int) * (size_t)geo.ncells;
        const size_t smem_s = round_up(((size_t)(kSortWarps + 2) * geo.ncells + 1) * sizeof(unsigned int), 16) +
                              geo.range * (sizeof(double2) + sizeof(unsigned short));
        if (smem_s + 1024 > (size_t)227 * 1024) return fail(OSC_ERR_INVALID_ARG, "internal: sort chunk of %zu events does not fit shared memory", geo.range);
        const unsigned per_sm = (unsigned)std::max<size_t>(1, std::min<size_t>(4, kSmemBudget / (smem_s + 1024)));
        const int steps = (int)(geo.range / (32 * kSortWarps));
        auto scatter = steps == 2 ? sort_scatter_kernel<2> : steps == 4 ? sort_scatter_kernel<4> : sort_scatter_kernel<8>;
        if (steps != 2 && steps != 4 && steps != 8)
            return fail(OSC_ERR_INVALID_ARG, "internal: sort chunk of %zu events is not 1024, 2048 or 4096", geo.range);
        if (smem_s > 48 * 1024) CUDA_TRY(cudaFuncSetAttribute(scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_s));
        sort_count_kernel<<<std::min<unsigned>(geo.nranges, (unsigned)sms * 4u), kSortThreads, smem_c, st>>>(
            E_true, E_reco, channel, se.n, energy_scale, bin_edges, se.n_bins, geo, cellid, count);
        if ((rc = post_launch("sort of the events: count"))) return rc;
        scan_offsets_cell_kernel<<<geo.ncells, 1024, 0, st>>>(count, geo, se.cell_begin);
        if ((rc = post_launch("sort of the events: offsets per cell"))) return rc;
        scan_offsets_kernel<<<1, 1024, 0, st>>>(geo, se.cell_begin, se.unit_begin, se.unit_cell);
        if ((rc = post_launch("sort of the events: offsets"))) return rc;
        scatter<<<std::min<unsigned>(geo.nranges, (unsigned)sms * per_sm), kSortThreads, smem_s, st>>>(
            E_true, w0, cellid, se.n, geo, count, se.cell_begin, se.sEt, se.sW);
        return post_launch("sort of the events: scatter");
    }
    // blocks per SM of the two event-ordered passes (measured at 1e7 events): the count pass is latency-bound and wants
    // all the warps an SM holds, the scatter pass is bound by its write pattern and gets slower with more of them
    const unsigned range_blocks = (geo.nranges + kScanWarps - 1) / kScanWarps;
    const unsigned count_blocks = std::min<unsigned>(range_blocks, (unsigned)sms * 16u);
    const unsigned sort_blocks = std::min<unsigned>(range_blocks, (unsigned)sms * 8u);
    const size_t smem_cnt = sizeof(unsigned int) * kScanWarps * (size_t)geo.ncells;
    const size_t smem_count = bin_table_bytes(se.n_bins) + smem_cnt;
    if (smem_count > 48 * 1024)
        CUDA_TRY(cudaFuncSetAttribute(scan_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_count));
    if (smem_cnt > 48 * 1024)
        CUDA_TRY(cudaFuncSetAttribute(scan_scatter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cnt));
    scan_count_kernel<<<count_blocks, 32 * kScanWarps, smem_count, st>>>(E_true, E_reco, channel, se.n, energy_scale,
                                                                         bin_edges, se.n_bins, geo, cellid, count);
    if ((rc = post_launch("sort of the events: count"))) return rc;
    scan_offsets_cell_kernel<<<geo.ncells, 1024, 0, st>>>(count, geo, se.cell_begin);
    if ((rc = post_launch("sort of the events: offsets per cell"))) return rc;
    scan_offsets_kernel<<<1, 1024, 0, st>>>(geo, se.cell_begin, se.unit_begin, se.unit_cell);
    if ((rc = post_launch("sort of the events: offsets"))) return rc;
    scan_scatter_kernel<<<sort_blocks, 32 * kScanWarps, smem_cnt, st>>>(E_true, w0, cellid, se.n, geo, count, se.cell_begin,
                                                                        se.sEt, se.sW);
    return post_launch("sort of the events: scatter");
}

// The plan of the last point list, kept: a scan is typically repeated over the same grid (other events, another energy
// scale, the next step of a fit), and building the plan is 0.2 ms of host time for 1024 points -- a quarter of what the
// GPU then needs for 1e6 events.  Compared bytewise (a list that differs only in padding bytes is rebuilt, never reused
// wrongly); thread-safe; the plan is immutable once built.
struct PlanCache {
    std::mutex mu;
    std::vector<unsigned char> key;
    std::shared_ptr<const ScanPlan> plan;
};
PlanCache g_plan_cache;

std::shared_ptr<const ScanPlan> scan_plan_for(const osc_params* points, int n_points)
{
    const size_t bytes = (size_t)n_points * sizeof(osc_params);
    {
        std::lock_guard<std::mutex> lk(g_plan_cache.mu);
        if (g_plan_cache.plan && g_plan_cache.key.size() == bytes && !std::memcmp(g_plan_cache.key.data(), points, bytes))
            return g_plan_cache.plan;
    }
    auto fresh = std::make_shared<ScanPlan>();
    build_scan_plan(points, n_points, *fresh);
    std::lock_guard<std::mutex> lk(g_plan_cache.mu);
    g_plan_cache.key.assign(reinterpret_cast<const unsigned char*>(points), reinterpret_cast<const unsigned char*>(points) + bytes);
    g_plan_cache.plan = fresh;
    return fresh;
}

int scan_merge(const double* partial, const SortedEvents& se, int n_points, double* hist_out, cudaStream_t st)
{
    if (n_points < 32)
        scan_merge_few_kernel<<<se.geo.ncells, 256, 0, st>>>(partial, se.unit_begin, se.geo.ncells, n_points, hist_out);
    else
        scan_merge_kernel<<<dim3((unsigned)se.geo.ncells, (unsigned)((n_points + 255) / 256)), 256, 0, st>>>(
            partial, se.unit_begin, se.geo.ncells, n_points, hist_out);
    return post_launch("batched reweighting on sorted events (merge)");
}

// k4 with the tables in the kernel parameters (scan_const_kernel): unless osc_set_batch_path("k4s") asks for the
// shared-memory slice kernel, whenever every channel is of one of the two kinds the kernel is built for.
// A launch per sub-group is 32 launches for 1024 points, about 5 us of host time each with 5.8 kB of parameters: below 1e5
// events the call is bound by that and the single launch of the slice kernel is ahead (1024 points in 32 sub-groups, plan
// of the point list kept, ms per call, slice kernel / this one: 1e4 events 0.084 / 0.217, 3e4 0.113 / 0.135, 1e5 0.178 /
// 0.177, 2e5 0.285 / 0.251, 4e5 0.491 / 0.392, 1e6 1.110 / 0.733, 3e6 3.159 / 1.950).  Dealing the launches round to eight
// side streams that fork from and join the caller's stream costs more host time than it saves (0.28 ms per call up to
// 2e5 events).  osc_set_batch_path("k4s" | "k4c") forces one of the two kernels.
constexpr size_t kConstMinEvents = 100000;
constexpr size_t kConstUnits = 4096;   // pieces per launch the events are cut into (pieces of 128 / 256 / 320 / 384 / 512
                                       // events at 1e6: 0.845 / 0.747 / 0.752 / 0.780 / 0.782 ms per call)
bool scan_uses_const(const ScanPlan& plan, size_t n)
{
    const int forced = g_batch_path.load();
    if (forced == 41 || !plan.const_ok) return false;
    return forced == 42 || n >= kConstMinEvents;
}

// One launch per sub-group, nothing uploaded.  The first launch is ordered after the sort as usual; the others carry
// the programmatic-serialization attribute: they start while their predecessor drains and, because every block waits
// for the predecessor before it exits, complete in order, so the merge behind them sees all of partial[][].
int scan_run_const(const SortedEvents& se, const ScanPlan& plan, int n_points, double* hist_out, cudaStream_t st)
{
    int rc;
    const ScanGeom& geo = se.geo;
    Scratch sc;
    if ((rc = sc.alloc(round_up((size_t)geo.max_units * n_points * sizeof(double), 256), st))) return rc;
    double* partial = reinterpret_cast<double*>(sc.p);
    const int grid = (int)((geo.max_units + kScanWarps - 1) / kScanWarps);
    for (size_t s = 0; s < plan.consts.size(); ++s) {
        if (s == 0)
            scan_const_kernel<<<grid, 32 * kScanWarps, 0, st>>>(plan.consts[s], se.sEt, se.sW, se.cell_begin, se.unit_begin,
                                                               se.unit_cell, geo, se.n_bins, n_points, partial);
        else
            CUDA_TRY(launch_pdl(scan_const_kernel, grid, 32 * kScanWarps, 0, st, plan.consts[s], se.sEt, se.sW, se.cell_begin,
                                se.unit_begin, se.unit_cell, geo, se.n_bins, n_points, partial));
        if ((rc = post_launch("batched reweighting on sorted events (k4, tables in the kernel parameters)"))) return rc;
    }
    return scan_merge(partial, se, n_points, hist_out, st);
}

// The point kernels on sorted events: k4 (plan != nullptr: sub-groups of a scan grid) or k5 (full != nullptr: one
// parameter block per point, every point its own eigen-problem), then the ordered merge of the pieces of every cell.
int scan_run(const SortedEvents& se, const ScanPlan* plan, const std::vector<BinArgs>* full, int n_points,
             double* hist_out, cudaStream_t st)
{
    int rc;
    ScanGeom geo = se.geo;
    if (plan && g_batch_path.load() == 42 && !plan->const_ok)
        return fail(OSC_ERR_INVALID_ARG, "osc_set_batch_path(\"k4c\"): a channel of this point list is of neither kind scan_const_kernel is built for");
    if (plan && scan_uses_const(*plan, se.n)) return scan_run_const(se, *plan, n_points, hist_out, st);
    geo.nsubs = plan ? (int)plan->subs.size() : n_points;      // items a warp walks per piece: sub-groups or points
    int slots = geo.nsubs < 8 ? geo.nsubs : 8;
    geo.subs_per_slot = (geo.nsubs + slots - 1) / slots;
    slots = (geo.nsubs + geo.subs_per_slot - 1) / geo.subs_per_slot;
    if (!plan && geo.piece > 512) return fail(OSC_ERR_INVALID_ARG, "internal: piece of %u events is too long for k5", geo.piece);

    const size_t b_groups = plan ? round_up(plan->groups.size() * sizeof(ScanGroup), 256)
                                 : round_up((size_t)n_points * sizeof(BinArgs), 256);
    const size_t b_subs = plan ? round_up(plan->subs.size() * sizeof(ScanSub), 256) : 0;
    const size_t b_partial = round_up((size_t)geo.max_units * n_points * sizeof(double), 256);
    Scratch sc;
    if ((rc = sc.alloc(b_groups + b_subs + b_partial, st))) return rc;
    ScanGroup* d_groups = reinterpret_cast<ScanGroup*>(sc.p);
    ScanSub* d_subs = reinterpret_cast<ScanSub*>(sc.p + b_groups);
    double* partial = reinterpret_cast<double*>(sc.p + b_groups + b_subs);
    // the host-built tables are contiguous on the device: one asynchronous copy from a pinned staging slot
    PinnedRing* ring = nullptr;
    if ((rc = ring_for_device(&ring))) return rc;
    PinnedRing::Slot* slot = nullptr;
    std::unique_lock<std::mutex> ring_lock;
    if ((rc = ring->acquire(b_groups + b_subs, &slot, ring_lock))) return rc;
    if (plan) {
        std::memcpy(slot->host, plan->groups.data(), plan->groups.size() * sizeof(ScanGroup));
        std::memcpy(static_cast<char*>(slot->host) + b_groups, plan->subs.data(), plan->subs.size() * sizeof(ScanSub));
    } else {
        std::memcpy(slot->host, full->data(), (size_t)n_points * sizeof(BinArgs));
    }
    CUDA_TRY(cudaMemcpyAsync(d_groups, slot->host, b_groups + b_subs, cudaMemcpyHostToDevice, st));
    if ((rc = ring->fence(slot, st))) return rc;
    ring_lock.unlock();

    const dim3 grid((geo.max_units + kScanWarps - 1) / kScanWarps, (unsigned)slots);
    if (plan) {
        scan_main_kernel<<<grid, 32 * kScanWarps, 0, st>>>(d_groups, d_subs, se.sEt, se.sW, se.cell_begin, se.unit_begin,
                                                           se.unit_cell, geo, se.n_bins, n_points, partial);
        if ((rc = post_launch("batched reweighting on sorted events (k4, factorised)"))) return rc;
    } else {
        const ChannelKinds kinds = channel_kinds();
        if (geo.subs_per_slot > 2) {          // a piece is staged in shared memory once and walked by many points
            const size_t smem_ev = sizeof(double) * kScanWarps * 3 * (size_t)geo.piece;  // <= 48 kB at piece = 512
            scan_full_kernel<true><<<grid, 32 * kScanWarps, smem_ev, st>>>(
                reinterpret_cast<const double*>(d_groups), n_points, geo.subs_per_slot, kinds, se.sEt, se.sW,
                se.cell_begin, se.unit_begin, se.unit_cell, geo, se.n_bins, partial);
        } else {                              // one or two points per piece: straight from the sorted arrays
            scan_full_kernel<false><<<grid, 32 * kScanWarps, 0, st>>>(
                reinterpret_cast<const double*>(d_groups), n_points, geo.subs_per_slot, kinds, se.sEt, se.sW,
                se.cell_begin, se.unit_begin, se.unit_cell, geo, se.n_bins, partial);
        }
        if ((rc = post_launch("batched reweighting on sorted events (k5, one eigen-problem per point)"))) return rc;
    }
    return scan_merge(partial, se, n_points, hist_out, st);
}

// One batched call: sort into a stream-ordered scratch, then run.
int launch_batch_scan(const ScanPlan* plan, const std::vector<BinArgs>* full, int n_points, const double* E_true,
                      const double* E_reco, const double* w0, const int8_t* channel, size_t n, double energy_scale,
                      const double* bin_edges, int n_bins, double* hist_out, cudaStream_t st)
{
    int rc;
    const int nsubs = plan ? (int)plan->subs.size() : n_points;
    const int slots = nsubs < 8 ? nsubs : 8;
    size_t piece = round_up(n * (size_t)slots / 16384 + 1, 64);
    if (plan && scan_uses_const(*plan, n)) piece = round_up(n / kConstUnits + 1, 64);   // a launch per sub-group: its own grid
    if (piece < 128) piece = 128;
    if (piece > (plan ? 8192u : 512u)) piece = plan ? 8192 : 512;   // k5 stages the piece in shared memory
    SortedEvents se;
    se.n = n;
    se.n_bins = n_bins;
    if ((rc = sorted_geometry(n, n_bins, piece, se.geo))) return rc;
    const size_t b_cells = sorted_bytes_cells(se.geo.ncells), b_ev = sorted_bytes_events(n);
    const size_t b_units = sorted_bytes_units(se.geo.max_units);
    Scratch sc;
    if ((rc = sc.alloc(2 * b_cells + 2 * b_ev + b_units, st))) return rc;
    se.cell_begin = reinterpret_cast<unsigned int*>(sc.p);
    se.unit_begin = reinterpret_cast<unsigned int*>(sc.p + b_cells);
    se.sEt = reinterpret_cast<double*>(sc.p + 2 * b_cells);
    se.sW = reinterpret_cast<double*>(sc.p + 2 * b_cells + b_ev);
    se.unit_cell = reinterpret_cast<unsigned short*>(sc.p + 2 * b_cells + 2 * b_ev);
    if ((rc = scan_sort(se, E_true, E_reco, w0, channel, energy_scale, bin_edges, st))) return rc;
    return scan_run(se, plan, full, n_points, hist_out, st);
}

// An osc_plan: the sorted events of one (event sample, energy scale, binning), kept on the device.
struct PlanImpl {
    unsigned long long magic = 0x6F73635F706C616EULL;   // "osc_plan"
    int device = 0;
    SortedEvents se;
    char* buf = nullptr;
};

PlanImpl* plan_cast(const void* p)
{
    PlanImpl* q = static_cast<PlanImpl*>(const_cast<void*>(p));
    return (q && q->magic == 0x6F73635F706C616EULL) ? q : nullptr;
}

} // namespace

int osc_reweight_bin_scales(const double* E_true, const double* E_reco, const double* w0, const int8_t* channel,
                            size_t n, const double* energy_scales, int n_scales, const double* bin_edges, int n_bins,
                            double* hist_out, void* stream)
{
    if (n_scales < 1 || n_scales > kMaxScales)
        return fail(OSC_ERR_INVALID_ARG, "n_scales = %d outside [1, %d]", n_scales, kMaxScales);
    if (!energy_scales) return fail(OSC_ERR_INVALID_ARG, "null energy_scales");
    int rc = OSC_OK;
    for (int k = 0; k < n_scales; ++k)
        if ((rc = check_bin_args(E_true, E_reco, w0, channel, n, energy_scales[k], bin_edges, n_bins, hist_out))) return rc;
    if (n > 0 && !w0) return fail(OSC_ERR_INVALID_ARG, "null w0 with n > 0");
    if (!aligned(hist_out, 8)) return fail(OSC_ERR_ALIGNMENT, "hist_out not 8-byte aligned");
    HostSet h;
    if ((rc = snapshot(h))) return rc;
    BinArgs args;
    make_bin_args(h, args);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t nh = (size_t)kChannels * n_bins;
    if (n_scales > 1 && n > 0) {
        rc = launch_reweight_scales(args, E_true, E_reco, w0, channel, n, energy_scales, n_scales, bin_edges, n_bins,
                                    hist_out, st);
        if (rc != 1) return rc;
    }
    for (int k = 0; k < n_scales; ++k)          // one scale, no events, or histograms too large to fuse
        if ((rc = launch_reweight(args, E_true, E_reco, w0, channel, n, energy_scales[k], bin_edges, n_bins,
                                  hist_out + (size_t)k * nh, st)))
            return rc;
    return OSC_OK;
}

int osc_reweight_bin_batch(const osc_params* points, int n_points, const double* E_true, const double* E_reco,
                           const double* w0, const int8_t* channel, size_t n, double energy_scale,
                           const double* bin_edges, int n_bins, double* hist_out, void* stream)
{
    if (n_points < 0) return fail(OSC_ERR_INVALID_ARG, "n_points < 0");
    if (n_points == 0) return OSC_OK;
    if (!points) return fail(OSC_ERR_INVALID_ARG, "null points with n_points > 0");
    int rc = check_bin_args(E_true, E_reco, w0, channel, n, energy_scale, bin_edges, n_bins, hist_out);
    if (rc) return rc;
    if (n > 0 && !w0) return fail(OSC_ERR_INVALID_ARG, "null w0 with n > 0");
    if (!aligned(hist_out, 8)) return fail(OSC_ERR_ALIGNMENT, "hist_out not 8-byte aligned");
    for (int p = 0; p < n_points; ++p)
        if (const char* msg = check_params(points[p]))
            return fail(OSC_ERR_INVALID_ARG, "osc_reweight_bin_batch: point %d: %s", p, msg);
    const size_t nh = (size_t)kChannels * n_bins;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (n == 0) {
        CUDA_TRY(cudaMemsetAsync(hist_out, 0, (size_t)n_points * nh * sizeof(double), st));
        return OSC_OK;
    }
    // Points that differ only in theta23 and delta_cp share the eigen-problem: when the list has enough of that
    // structure (a scan grid), the factorised path k4 does the eigen-solve once per group (osc_scan.cuh).
    // osc_set_batch_path overrides the choice (tests exercise all paths on the same inputs).
    const int forced = g_batch_path.load();
    {
        const std::shared_ptr<const ScanPlan> held = scan_plan_for(points, n_points);
        const ScanPlan& plan = *held;
        bool use_scan = (size_t)n_points >= 8 * plan.subs.size();
        if (forced == 4 || forced == 41 || forced == 42) use_scan = true;
        if (forced == 2 || forced == 5) use_scan = false;
        if (use_scan)
            return launch_batch_scan(&plan, nullptr, n_points, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                     n_bins, hist_out, st);
    }
    // a1 for every point (host), packed as BinArgs
    std::vector<BinArgs> blocks((size_t)n_points);
    for (int p = 0; p < n_points; ++p) {
        HostSet h;
        precompute(points[p], h);
        make_bin_args(h, blocks[(size_t)p]);
    }
    // Point lists without scan structure.  The sort of the events costs about 20 ps per event (44 us at 1e6 events, 201 us at
    // 1e7) and then a point costs 9 ps per event in k5 against 12.4 ps (23 us per 1e6 events) for a pass of the fused
    // single-set kernel k2: k5 is ahead from 4 points on at 1e6 events and from 6 points on at 1e7.  Below that every
    // point gets its own k2 pass.
    bool use_full = n_points >= (n <= 2000000 ? 4 : 6);
    if (forced == 5) use_full = true;
    if (forced == 2) use_full = false;
    if (use_full)
        return launch_batch_scan(nullptr, &blocks, n_points, E_true, E_reco, w0, channel, n, energy_scale, bin_edges,
                                 n_bins, hist_out, st);
    for (int p = 0; p < n_points; ++p)
        if ((rc = launch_reweight(blocks[(size_t)p], E_true, E_reco, w0, channel, n, energy_scale, bin_edges, n_bins,
                                  hist_out + (size_t)p * nh, st)))
            return rc;
    return OSC_OK;
}

int osc_plan_create(const double* E_true, const double* E_reco, const double* w0, const int8_t* channel, size_t n,
                    double energy_scale, const double* bin_edges, int n_bins, void* stream, osc_plan** plan_out)
{
    if (!plan_out) return fail(OSC_ERR_INVALID_ARG, "null plan_out");
    *plan_out = nullptr;
    double dummy;
    int rc = check_bin_args(E_true, E_reco, w0, channel, n, energy_scale, bin_edges, n_bins, &dummy);
    if (rc) return rc;
    if (n > 0 && !w0) return fail(OSC_ERR_INVALID_ARG, "null w0 with n > 0");
    PlanImpl* pl = new (std::nothrow) PlanImpl;
    if (!pl) return fail(OSC_ERR_CUDA, "out of host memory");
    cudaError_t e = cudaGetDevice(&pl->device);
    if (e != cudaSuccess) {
        delete pl;
        return fail(OSC_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    }
    SortedEvents& se = pl->se;
    se.n = n;
    se.n_bins = n_bins;
    // pieces short enough for k5 (it stages a piece in shared memory) and for a single parameter set to fill the GPU
    size_t piece = round_up(n / 16384 + 1, 64);
    if (piece < 128) piece = 128;
    if (piece > 512) piece = 512;
    if ((rc = sorted_geometry(n, n_bins, piece, se.geo))) {
        delete pl;
        return rc;
    }
    const size_t b_cells = sorted_bytes_cells(se.geo.ncells), b_ev = sorted_bytes_events(n);
    const size_t b_units = sorted_bytes_units(se.geo.max_units);
    e = cudaMalloc((void**)&pl->buf, 2 * b_cells + 2 * b_ev + b_units + 256);
    if (e != cudaSuccess) {
        delete pl;
        return fail(OSC_ERR_CUDA, "cudaMalloc of the plan (%zu bytes): %s", 2 * b_cells + 2 * b_ev, cudaGetErrorString(e));
    }
    se.cell_begin = reinterpret_cast<unsigned int*>(pl->buf);
    se.unit_begin = reinterpret_cast<unsigned int*>(pl->buf + b_cells);
    se.sEt = reinterpret_cast<double*>(pl->buf + 2 * b_cells);
    se.sW = reinterpret_cast<double*>(pl->buf + 2 * b_cells + b_ev);
    se.unit_cell = reinterpret_cast<unsigned short*>(pl->buf + 2 * b_cells + 2 * b_ev);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (n == 0) {
        e = cudaMemsetAsync(pl->buf, 0, 2 * b_cells, st);       // no event, no piece
        rc = e == cudaSuccess ? OSC_OK : fail(OSC_ERR_CUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
    } else {
        rc = scan_sort(se, E_true, E_reco, w0, channel, energy_scale, bin_edges, st);
    }
    if (rc) {
        cudaFree(pl->buf);
        delete pl;
        return rc;
    }
    *plan_out = reinterpret_cast<osc_plan*>(pl);
    return OSC_OK;
}

int osc_plan_destroy(osc_plan* plan)
{
    if (!plan) return OSC_OK;
    PlanImpl* pl = plan_cast(plan);
    if (!pl) return fail(OSC_ERR_INVALID_ARG, "not an osc_plan");
    pl->magic = 0;
    cudaError_t e = cudaFree(pl->buf);              // synchronises with the work that still reads the plan
    delete pl;
    if (e != cudaSuccess) return fail(OSC_ERR_CUDA, "cudaFree: %s", cudaGetErrorString(e));
    return OSC_OK;
}

int osc_plan_reweight_bin_batch(const osc_plan* plan, const osc_params* points, int n_points, double* hist_out,
                                void* stream)
{
    PlanImpl* pl = plan_cast(plan);
    if (!pl) return fail(OSC_ERR_INVALID_ARG, "not an osc_plan");
    if (n_points < 0) return fail(OSC_ERR_INVALID_ARG, "n_points < 0");
    if (n_points == 0) return OSC_OK;
    if (!points || !hist_out) return fail(OSC_ERR_INVALID_ARG, "null points or hist_out");
    if (!aligned(hist_out, 8)) return fail(OSC_ERR_ALIGNMENT, "hist_out not 8-byte aligned");
    for (int p = 0; p < n_points; ++p)
        if (const char* msg = check_params(points[p]))
            return fail(OSC_ERR_INVALID_ARG, "osc_plan_reweight_bin_batch: point %d: %s", p, msg);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // same choice between the factorised kernel k4 and the one-eigen-problem-per-point kernel k5 as in
    // osc_reweight_bin_batch; the sort is already paid for, so there is no k2 branch
    const std::shared_ptr<const ScanPlan> held = scan_plan_for(points, n_points);
    const ScanPlan& sp = *held;
    bool use_scan = (size_t)n_points >= 8 * sp.subs.size();
    const int forced = g_batch_path.load();
    if (forced == 4 || forced == 41 || forced == 42) use_scan = true;
    if (forced == 5) use_scan = false;
    if (use_scan) return scan_run(pl->se, &sp, nullptr, n_points, hist_out, st);
    std::vector<BinArgs> blocks((size_t)n_points);
    for (int p = 0; p < n_points; ++p) {
        HostSet h;
        precompute(points[p], h);
        make_bin_args(h, blocks[(size_t)p]);
    }
    return scan_run(pl->se, nullptr, &blocks, n_points, hist_out, st);
}

int osc_plan_reweight_bin(const osc_plan* plan, double* hist_out, void* stream)
{
    PlanImpl* pl = plan_cast(plan);
    if (!pl) return fail(OSC_ERR_INVALID_ARG, "not an osc_plan");
    if (!hist_out) return fail(OSC_ERR_INVALID_ARG, "null hist_out");
    if (!aligned(hist_out, 8)) return fail(OSC_ERR_ALIGNMENT, "hist_out not 8-byte aligned");
    HostSet h;
    int rc = snapshot(h);
    if (rc) return rc;
    BinArgs args;
    make_bin_args(h, args);
    // one parameter set: parameter block by value, partial sums in the per-stream scratch of the library -- two
    // launches and nothing else on the stream
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const SortedEvents& se = pl->se;
    ScratchLease lease;
    if ((rc = stream_scratch(kScratchHead + (size_t)se.geo.max_units * sizeof(double), st, lease))) return rc;
    double* partial = reinterpret_cast<double*>(lease.p + kScratchHead);
    const ChannelKinds kinds = channel_kinds();
    scan_full_one_kernel<<<(se.geo.max_units + kScanWarps - 1) / kScanWarps, 32 * kScanWarps, 0, st>>>(
        args, kinds, se.sEt, se.sW, se.cell_begin, se.unit_begin, se.unit_cell, se.geo, se.n_bins, partial);
    if ((rc = post_launch("osc_plan_reweight_bin (k5, one parameter set)"))) return rc;
    scan_merge_few_kernel<<<se.geo.ncells, 256, 0, st>>>(partial, se.unit_begin, se.geo.ncells, 1, hist_out);
    return post_launch("osc_plan_reweight_bin (merge)");
}

int osc_bin_centre_compare(const double* E_true, const double* w0, const int8_t* channel, size_t n,
                           const double* bin_edges, int n_bins, double* hist_event_out, double* hist_centre_out,
                           void* stream)
{
    int rc = check_bin_args(E_true, E_true, w0, channel, n, 1.0, bin_edges, n_bins, hist_event_out);
    if (rc) return rc;
    if (!hist_centre_out) return fail(OSC_ERR_INVALID_ARG, "null hist_centre_out");
    if (n > 0 && !w0) return fail(OSC_ERR_INVALID_ARG, "null w0 with n > 0");
    if (!aligned(hist_event_out, 8) || !aligned(hist_centre_out, 8))
        return fail(OSC_ERR_ALIGNMENT, "histogram not 8-byte aligned");
    HostSet h;
    if ((rc = snapshot(h))) return rc;
    BinArgs args;
    make_bin_args(h, args);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int nh = kChannels * n_bins;
    // launch shape of the unit histogram, fixed before anything is enqueued: a sub-histogram per (warp, event of the
    // lane) while that fits, one per warp above (768 bins: 8 warps x 4 x 768 x 8 B = 196 kB)
    const size_t sub2 = sizeof(double) * (kBlock / 32) * kSlots * (size_t)nh;
    const bool two_slots = bin_table_bytes(n_bins) + sub2 + 1024 <= kSmemBudget;
    const size_t sub1 = two_slots ? sub2 : sub2 / kSlots;
    const int n_sub = two_slots && bin_table_bytes(n_bins) + 2 * sub1 <= 100 * 1024 ? 2 : 1;
    const size_t smem = bin_table_bytes(n_bins) + n_sub * sub1;
    if (smem + 1024 > (size_t)227 * 1024)
        return fail(OSC_ERR_INVALID_ARG, "n_bins = %d needs more shared memory than one SM has", n_bins);
    // event by event: the fused kernel with the true energy in the role of the binned energy
    if ((rc = launch_reweight(args, E_true, E_true, w0, channel, n, 1.0, bin_edges, n_bins, hist_event_out, st))) return rc;
    // bin centre: unoscillated content of every true-energy bin, times the probability at the centre
    if (n == 0) {
        CUDA_TRY(cudaMemsetAsync(hist_centre_out, 0, (size_t)nh * sizeof(double), st));
    } else {
        int sms = 0;
        if ((rc = sm_count(&sms))) return rc;
        const size_t ntiles = (n + 2 * kBlock - 1) / (2 * (size_t)kBlock);
        size_t g = (size_t)sms * (smem <= 100 * 1024 ? 2 : 1);
        if (ntiles < g) g = ntiles;
        const int grid = (int)g;
        ScratchLease lease;
        if ((rc = stream_scratch(merge_scratch_bytes(grid, (size_t)nh), st, lease))) return rc;
        const MergeScratch ms = call_scratch(lease.p, grid, (size_t)nh).ms;
        if (two_slots) {
            if (smem > 48 * 1024)
                CUDA_TRY(cudaFuncSetAttribute(unit_hist_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            unit_hist_kernel<2><<<grid, kBlock, smem, st>>>(E_true, w0, channel, n, bin_edges, n_bins, n_sub, ms, hist_centre_out);
        } else {
            CUDA_TRY(cudaFuncSetAttribute(unit_hist_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            unit_hist_kernel<1><<<grid, kBlock, smem, st>>>(E_true, w0, channel, n, bin_edges, n_bins, 1, ms, hist_centre_out);
        }
        if ((rc = post_launch("osc_bin_centre_compare (unit histogram)"))) return rc;
    }
    centre_weight_kernel<<<(nh + 255) / 256, 256, 0, st>>>(args, bin_edges, n_bins, hist_centre_out);
    return post_launch("osc_bin_centre_compare (centre weights)");
}

int osc_neg2lnl(const double* hist, int n_points, int n_cells, const double* data, double norm, double* out,
                void* stream)
{
    if (n_points < 0 || n_cells < 1) return fail(OSC_ERR_INVALID_ARG, "osc_neg2lnl: n_points < 0 or n_cells < 1");
    if (n_points == 0) return OSC_OK;
    if (!hist || !data || !out) return fail(OSC_ERR_INVALID_ARG, "osc_neg2lnl: null pointer");
    if (!(norm > 0.0) || !std::isfinite(norm)) return fail(OSC_ERR_INVALID_ARG, "osc_neg2lnl: norm must be finite and > 0");
    if (!aligned(hist, 8) || !aligned(data, 8) || !aligned(out, 8))
        return fail(OSC_ERR_ALIGNMENT, "osc_neg2lnl: fp64 array not 8-byte aligned");
    const int warps = 8;
    neg2lnl_kernel<<<(n_points + warps - 1) / warps, 32 * warps, 0, static_cast<cudaStream_t>(stream)>>>(
        hist, n_points, n_cells, data, norm, out);
    return post_launch("osc_neg2lnl");
}

int osc_bin_index(const double* E_true, const double* E_reco, const int8_t* channel, size_t n, double energy_scale,
                  const double* bin_edges, int n_bins, int32_t* bin_out, void* stream)
{
    int rc = check_bin_args(E_true, E_reco, E_true, channel, n, energy_scale, bin_edges, n_bins, bin_out);
    if (rc) return rc;
    if (n == 0) return OSC_OK;
    int grid = 1;
    if ((rc = grid_for((n + kBlock - 1) / kBlock, &grid))) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    bin_index_kernel<<<grid, kBlock, bin_table_bytes(n_bins), st>>>(E_true, E_reco, channel, n, energy_scale, bin_edges,
                                                                   n_bins, bin_out);
    return post_launch("osc_bin_index");
}

int osc_prob_host(const double* E_true_host, size_t n, int flavour_in, int flavour_out, int antinu,
                  double* P_out_host)
{
    if (n > 0 && (!E_true_host || !P_out_host)) return fail(OSC_ERR_INVALID_ARG, "null host array with n > 0");
    HostPath* hp = nullptr;
    int rc = host_path(&hp);
    if (rc) return rc;
    HostPath& g_host = *hp;
    std::lock_guard<std::mutex> lk(g_host.mu);
    const size_t bytes = round_up(n * sizeof(double), 256);
    if ((rc = g_host.ensure(2 * bytes + 256))) return rc;
    double* dE = reinterpret_cast<double*>(g_host.buf);
    double* dP = reinterpret_cast<double*>(g_host.buf + bytes);
    if (n) CUDA_TRY(cudaMemcpyAsync(dE, E_true_host, n * sizeof(double), cudaMemcpyHostToDevice, g_host.stream));
    rc = osc_prob(dE, n, flavour_in, flavour_out, antinu, dP, g_host.stream);
    if (rc) return rc;
    if (n) CUDA_TRY(cudaMemcpyAsync(P_out_host, dP, n * sizeof(double), cudaMemcpyDeviceToHost, g_host.stream));
    CUDA_TRY(cudaStreamSynchronize(g_host.stream));
    return OSC_OK;
}

int osc_reweight_bin_scales_host(const double* E_true_host, const double* E_reco_host, const double* w0_host,
                                 const int8_t* channel_host, size_t n, const double* energy_scales, int n_scales,
                                 const double* bin_edges_host, int n_bins, double* hist_out_host)
{
    if (n_bins < 1 || n_bins > kMaxBins) return fail(OSC_ERR_INVALID_ARG, "n_bins = %d outside [1, %d]", n_bins, kMaxBins);
    if (n_scales < 1 || n_scales > kMaxScales)
        return fail(OSC_ERR_INVALID_ARG, "n_scales = %d outside [1, %d]", n_scales, kMaxScales);
    if (!energy_scales || !bin_edges_host || !hist_out_host)
        return fail(OSC_ERR_INVALID_ARG, "null energy_scales, bin_edges or hist_out");
    if (n > 0 && (!E_true_host || !E_reco_host || !w0_host || !channel_host))
        return fail(OSC_ERR_INVALID_ARG, "null host array with n > 0");
    HostPath* hp = nullptr;
    int rc = host_path(&hp);
    if (rc) return rc;
    HostPath& g_host = *hp;
    std::lock_guard<std::mutex> lk(g_host.mu);
    const size_t nh = (size_t)kChannels * n_bins;
    const size_t nout = (size_t)n_scales * nh;
    // chunks of an even number of events (the 16-byte loads of the kernels), at most kHostChunks of at least kHostChunkMin
    size_t chunk = std::max<size_t>(kHostChunkMin, (n + kHostChunks - 1) / kHostChunks);
    chunk += chunk & 1;
    const int n_chunks = n ? (int)((n + chunk - 1) / chunk) : 1;
    const size_t b8 = round_up(n * sizeof(double), 256);
    const size_t b1 = round_up(n, 256);
    const size_t be = round_up((size_t)(n_bins + 1) * sizeof(double), 256);
    const size_t bh = round_up((size_t)(n_chunks + 1) * nout * sizeof(double), 256);
    if ((rc = g_host.ensure(3 * b8 + b1 + be + bh + 256))) return rc;
    char* p = g_host.buf;
    double* dEt = reinterpret_cast<double*>(p);
    double* dEr = reinterpret_cast<double*>(p + b8);
    double* dW = reinterpret_cast<double*>(p + 2 * b8);
    int8_t* dC = reinterpret_cast<int8_t*>(p + 3 * b8);
    double* dEdges = reinterpret_cast<double*>(p + 3 * b8 + b1);
    double* dH = reinterpret_cast<double*>(p + 3 * b8 + b1 + be);       // [0]: the result, [1 + c]: chunk c
    cudaStream_t st = g_host.stream, cs = g_host.copy_stream;
    CUDA_TRY(cudaMemcpyAsync(dEdges, bin_edges_host, (size_t)(n_bins + 1) * sizeof(double), cudaMemcpyHostToDevice, st));
    if (n_chunks == 1) {
        if (n) {
            CUDA_TRY(cudaMemcpyAsync(dEt, E_true_host, n * sizeof(double), cudaMemcpyHostToDevice, st));
            CUDA_TRY(cudaMemcpyAsync(dEr, E_reco_host, n * sizeof(double), cudaMemcpyHostToDevice, st));
            CUDA_TRY(cudaMemcpyAsync(dW, w0_host, n * sizeof(double), cudaMemcpyHostToDevice, st));
            CUDA_TRY(cudaMemcpyAsync(dC, channel_host, n, cudaMemcpyHostToDevice, st));
        }
        if ((rc = osc_reweight_bin_scales(dEt, dEr, dW, dC, n, energy_scales, n_scales, dEdges, n_bins, dH, st))) return rc;
    } else {
        // the copy stream runs ahead of the kernels by whole chunks; a chunk's kernel waits for its four arrays only
        for (int c = 0; c < n_chunks; ++c) {
            const size_t o = (size_t)c * chunk, m = std::min(chunk, n - o);
            CUDA_TRY(cudaMemcpyAsync(dEt + o, E_true_host + o, m * sizeof(double), cudaMemcpyHostToDevice, cs));
            CUDA_TRY(cudaMemcpyAsync(dEr + o, E_reco_host + o, m * sizeof(double), cudaMemcpyHostToDevice, cs));
            CUDA_TRY(cudaMemcpyAsync(dW + o, w0_host + o, m * sizeof(double), cudaMemcpyHostToDevice, cs));
            CUDA_TRY(cudaMemcpyAsync(dC + o, channel_host + o, m, cudaMemcpyHostToDevice, cs));
            CUDA_TRY(cudaEventRecord(g_host.chunk_ready[c], cs));
            CUDA_TRY(cudaStreamWaitEvent(st, g_host.chunk_ready[c], 0));
            if ((rc = osc_reweight_bin_scales(dEt + o, dEr + o, dW + o, dC + o, m, energy_scales, n_scales, dEdges, n_bins,
                                              dH + (size_t)(1 + c) * nout, st)))
                break;
        }
        if (!rc) {
            chunk_sum_kernel<<<(unsigned)((nout + 255) / 256), 256, 0, st>>>(dH + nout, n_chunks, nout, dH);
            rc = post_launch("osc_reweight_bin_scales_host (sum over the chunks)");
        }
        if (rc) {                                       // leave both streams idle before the buffers are used again
            cudaStreamSynchronize(cs);
            cudaStreamSynchronize(st);
            return rc;
        }
    }
    CUDA_TRY(cudaMemcpyAsync(hist_out_host, dH, nout * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return OSC_OK;
}

int osc_reweight_bin_host(const double* E_true_host, const double* E_reco_host, const double* w0_host,
                          const int8_t* channel_host, size_t n, double energy_scale, const double* bin_edges_host,
                          int n_bins, double* hist_out_host)
{
    return osc_reweight_bin_scales_host(E_true_host, E_reco_host, w0_host, channel_host, n, &energy_scale, 1,
                                        bin_edges_host, n_bins, hist_out_host);
}

int osc_set_batch_path(const char* path)
{
    if (!path) return fail(OSC_ERR_INVALID_ARG, "null path");
    int v = -1;
    if (!std::strcmp(path, "auto")) v = 0;
    if (!std::strcmp(path, "k2")) v = 2;
    if (!std::strcmp(path, "k4")) v = 4;
    if (!std::strcmp(path, "k4s")) v = 41;
    if (!std::strcmp(path, "k4c")) v = 42;
    if (!std::strcmp(path, "k5")) v = 5;
    if (v < 0) return fail(OSC_ERR_INVALID_ARG, "osc_set_batch_path: \"%s\" is not auto, k2, k4, k4s, k4c or k5", path);
    g_batch_path.store(v);
    return OSC_OK;
}

int osc_set_k2_tuning(int threads, int slots, int n_sub, int blocks_per_sm)
{
    if (threads != 0 && threads != 768 && threads != 512 && threads != 384 && threads != 256 && threads != 128)
        return fail(OSC_ERR_INVALID_ARG, "osc_set_k2_tuning: k2 is built for 128, 256, 384, 512 and 768 threads, not %d", threads);
    if (slots < 0 || slots > 2) return fail(OSC_ERR_INVALID_ARG, "osc_set_k2_tuning: slots = %d is not 0, 1 or 2", slots);
    if (n_sub != 0 && n_sub != 1 && n_sub != 2 && n_sub != 4)
        return fail(OSC_ERR_INVALID_ARG, "osc_set_k2_tuning: n_sub = %d is not 0, 1, 2 or 4", n_sub);
    if (blocks_per_sm < 0 || blocks_per_sm > 16) return fail(OSC_ERR_INVALID_ARG, "osc_set_k2_tuning: blocks_per_sm = %d", blocks_per_sm);
    g_tune_threads.store(threads);
    g_tune_slots.store(slots);
    g_tune_nsub.store(n_sub);
    g_tune_bps.store(blocks_per_sm);
    return OSC_OK;
}

const char* osc_last_error(void) { return t_err; }

unsigned long long osc_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

const char* osc_version(void) { return "osc_b200 0.2 (sm_100a)"; }

int osc_set_device(int device)
{
    CUDA_TRY(cudaSetDevice(device));
    return OSC_OK;
}

int osc_get_device(int* device)
{
    if (!device) return fail(OSC_ERR_INVALID_ARG, "null device pointer");
    CUDA_TRY(cudaGetDevice(device));
    return OSC_OK;
}

int osc_fp64_peak_probe(int iters, int blocks_per_sm, double* flops_per_launch, void* stream)
{
    if (iters < 1 || blocks_per_sm < 1 || blocks_per_sm > 8) return fail(OSC_ERR_INVALID_ARG, "bad probe arguments");
    int sms = 0;
    int rc = sm_count(&sms);
    if (rc) return rc;
    static double* sink = nullptr;
    if (!sink) CUDA_TRY(cudaMalloc((void**)&sink, 64));
    const int grid = sms * blocks_per_sm;
    dfma_probe_kernel<<<grid, kBlock, 0, static_cast<cudaStream_t>(stream)>>>(sink, iters, 1.0);
    if (flops_per_launch) *flops_per_launch = 2.0 * 8.0 * (double)iters * (double)kBlock * (double)grid;
    return post_launch("osc_fp64_peak_probe");
}

int osc_fp64_issue_probe(int kind, int iters, int blocks_per_sm, double* fp64_inst_per_launch, void* stream)
{
    if (kind < 0 || kind > 6 || iters < 1 || blocks_per_sm < 1 || blocks_per_sm > 8)
        return fail(OSC_ERR_INVALID_ARG, "bad probe arguments");
    int sms = 0;
    int rc = sm_count(&sms);
    if (rc) return rc;
    static double* buf = nullptr;             // in[24] (harmless values near 1), out[1]
    if (!buf) {
        CUDA_TRY(cudaMalloc((void**)&buf, 32 * sizeof(double)));
        double h[32];
        for (int k = 0; k < 32; ++k) h[k] = k < 8 ? 1.0 + 0.01 * k : (k < 16 ? 0.999999 - 1e-7 * k : 1e-9 * (k - 15));
        CUDA_TRY(cudaMemcpy(buf, h, sizeof h, cudaMemcpyHostToDevice));
    }
    const int grid = sms * blocks_per_sm;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    switch (kind) {
    case 0: issue_probe_kernel<0><<<grid, kBlock, 0, st>>>(buf, buf + 24, iters); break;
    case 1: issue_probe_kernel<1><<<grid, kBlock, 0, st>>>(buf, buf + 24, iters); break;
    case 2: issue_probe_kernel<2><<<grid, kBlock, 0, st>>>(buf, buf + 24, iters); break;
    case 3: issue_probe_kernel<3><<<grid, kBlock, 0, st>>>(buf, buf + 24, iters); break;
    case 4: issue_probe_kernel<4><<<grid, kBlock, 0, st>>>(buf, buf + 24, iters); break;
    case 5: issue_probe_kernel<5><<<grid, kBlock, 0, st>>>(buf, buf + 24, iters); break;
    default: issue_probe_kernel<6><<<grid, kBlock, 0, st>>>(buf, buf + 24, iters); break;
    }
    if (fp64_inst_per_launch) *fp64_inst_per_launch = 8.0 * (double)iters * (double)kBlock * (double)grid;
    return post_launch("osc_fp64_issue_probe");
}

} // extern "C"
