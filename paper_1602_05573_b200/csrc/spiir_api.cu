// C ABI of the B200-native SPIIR template-bank filter: see include/spiir.h for the contract.
// Host logic only (validation, bank layout upload, input tape, path choice, launches); every step of the
// hot path runs in the kernels of spiir_kernels.cuh.  No CPU fallback exists.
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/spiir.h"
#include "spiir_kernels.cuh"

using namespace spiir;

namespace {

thread_local char g_err[512] = "";
std::atomic<int64_t> g_launches{0};

int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CU_TRY(expr)                                                                              \
    do {                                                                                          \
        cudaError_t e_ = (expr);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return fail(e_ == cudaErrorMemoryAllocation ? SPIIR_ENOMEM : SPIIR_ECUDA, "%s: %s", #expr, \
                        cudaGetErrorString(e_));                                                  \
    } while (0)

// NVTX range per kernel path ("NVTX ranges per path"); costs one pointer test when no tool is attached.
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
    NvtxRange(const NvtxRange&) = delete;
    NvtxRange& operator=(const NvtxRange&) = delete;
};

// Every entry switches to the bank's device and restores the caller's current device on return (a single-process
// multi-GPU program must not find its current device changed by a library call).
struct DeviceGuard {
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int device)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != device) err = cudaSetDevice(device);
        else prev = -1;                      // nothing to restore
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

template <typename T>
cudaError_t upload(T** dst, const std::vector<T>& v)
{
    *dst = nullptr;
    const size_t bytes = std::max<size_t>(v.size(), 1) * sizeof(T);
    cudaError_t e = cudaMalloc((void**)dst, bytes);
    if (e != cudaSuccess) return e;
    if (!v.empty()) e = cudaMemcpy(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
    return e;
}

}  // namespace

// ---- scratch of the entry point that allocates nothing (spiir_filter_static, see include/spiir.h).
// File-scope device array of a fixed, modest size: every GPU that loads the library holds these 4 MiB until exit.  In host
// code the array's name is only a stand-in, not a device address: the address is looked up once per device with
// cudaGetSymbolAddress (that device current) and handed to the kernels.
constexpr int64_t kStaticStreamTiles = 8192;       // warp tiles (32 * filters_per_thread filter slots each)
static __device__ __align__(256) unsigned long long g_static_stream_scratch[kStaticStreamTiles * spiir::kStreamMax];

namespace {
constexpr int kMaxDevices = 64;
unsigned long long* g_static_scratch_addr[kMaxDevices] = {nullptr};
std::mutex g_static_scratch_mutex;

// The device address of g_static_stream_scratch on `device`, which must be the current device.
int static_scratch_address(int device, unsigned long long** out)
{
    if (device < 0 || device >= kMaxDevices) return fail(SPIIR_EINVAL, "device %d beyond the %d the static scratch serves", device, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_static_scratch_mutex);
    if (!g_static_scratch_addr[device]) {
        unsigned long long* ptr = nullptr;
        CU_TRY(cudaGetSymbolAddress((void**)&ptr, g_static_stream_scratch));
        if (!ptr) return fail(SPIIR_ECUDA, "cudaGetSymbolAddress returned a null address for the static scratch");
        g_static_scratch_addr[device] = ptr;
    }
    *out = g_static_scratch_addr[device];
    return SPIIR_OK;
}
}  // namespace

struct spiir_bank {
    int device = 0;
    int F = 8, W = 16, NC = 1;
    bool uniform_groups = true;
    bool gmem_only = false;          // the history alone exceeds shared memory: x is read through L1/L2
    bool configured[2][2] = {{false, false}, {false, false}};
    int64_t T = 0, K = 0, D = 0, n_slots = 0, n_tiles = 0;
    int32_t n_items = 0;
    double avg_conflict_degree = 0.0;
    spiir_options opt{};
    // device bank
    float *coef = nullptr, *y = nullptr;   // per-tile coefficient records (spiir_layout.hpp), filter state
    int32_t* item_round0 = nullptr;
    int32_t* canon = nullptr;
    int64_t* tile_begin = nullptr;   // [T+1] first warp tile of every template (streaming combine)
    u64* stream_scratch = nullptr;   // [n_tiles][kStreamMax] per-tile partial sums (streaming path)
    unsigned long long* stream_barrier = nullptr;   // arrival counter of the single-launch streaming kernel (monotonic)
    unsigned long long stream_arrivals = 0;
    bool stream_configured = false;
    int stream_occ = 0;
    size_t stream_occ_smem = 0;
    u64* peaks = nullptr;            // [T] packed (power bits << 32 | ~index) of the running call (spiir_filter_peaks)
    float* peak_snr = nullptr;       // internal SNR rows for spiir_filter_peaks without an SNR buffer (multi-round templates)
    int64_t peak_snr_cap = 0;
    bool segmented = false;          // small templates share warp tiles (SEG kernel variant)
    bool multi_round = false;        // some template spans several CTA rounds (its sums accumulate through the SNR rows)
    WarpWork* work = nullptr;
    int64_t* slot_of_filter = nullptr;
    // input tape: tape[cur][0..pos) holds the most recent samples, the next chunk is appended at pos
    float* tape[2] = {nullptr, nullptr};
    int cur = 0;
    int64_t cap = 0, pos = 0;
    // scan scratch
    float *zbuf = nullptr, *cbuf = nullptr;
    int64_t scan_cap_seg = 0;
    unsigned long long* scan_barrier = nullptr;   // arrival counter of the single-launch scan kernel (monotonic)
    unsigned long long scan_arrivals = 0;         // its value once every launch enqueued so far has completed
    bool scan_fused_configured = false;
    int scan_fused_occ = -1;
    size_t scan_fused_occ_smem = 0;
    // host-path scratch
    float* hx = nullptr;
    float* hsnr[2] = {nullptr, nullptr};
    int64_t hx_cap = 0, hsnr_cap = 0;
    cudaStream_t hstream = nullptr, cstream = nullptr;
    cudaEvent_t ev_done[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
    // stream ordering: the bank's state (y, tape) is touched by one call after the other; when a call arrives on another
    // stream than its predecessor's, that stream first waits for an event recorded behind the predecessor's work
    cudaStream_t last_stream = nullptr;
    bool last_stream_valid = false;
    cudaEvent_t ev_order = nullptr;
    bool free_pending[2] = {false, false};
    int64_t host_piece = 0;          // pieces enqueued so far by the host-buffer entry (ping-pong index)
    // device facts
    int n_sm = 0;
    size_t smem_optin = 0;
    int32_t last_path = SPIIR_PATH_AUTO;
    bool poisoned = false;
    // occupancy cache (CTAs per SM for a given dynamic shared memory size)
    size_t occ_smem[8] = {0};
    int occ_val[8] = {0};
    bool occ_gmem[8] = {false};
    int occ_n = 0;
};

namespace {

int64_t round_up(int64_t v, int64_t m) { return (v + m - 1) / m * m; }

void free_bank(spiir_bank* bk)
{
    if (!bk) return;
    cudaFree(bk->coef); cudaFree(bk->y);
    cudaFree(bk->item_round0); cudaFree(bk->canon); cudaFree(bk->tile_begin); cudaFree(bk->stream_scratch); cudaFree(bk->stream_barrier); cudaFree(bk->peaks); cudaFree(bk->peak_snr); cudaFree(bk->work); cudaFree(bk->slot_of_filter);
    cudaFree(bk->tape[0]); cudaFree(bk->tape[1]); cudaFree(bk->zbuf); cudaFree(bk->cbuf); cudaFree(bk->scan_barrier);
    cudaFree(bk->hx); cudaFree(bk->hsnr[0]); cudaFree(bk->hsnr[1]);
    for (int i = 0; i < 2; ++i) {
        if (bk->ev_done[i]) cudaEventDestroy(bk->ev_done[i]);
        if (bk->ev_free[i]) cudaEventDestroy(bk->ev_free[i]);
    }
    if (bk->ev_order) cudaEventDestroy(bk->ev_order);
    if (bk->hstream) cudaStreamDestroy(bk->hstream);
    if (bk->cstream) cudaStreamDestroy(bk->cstream);
    delete bk;
}

// The bank's state is about to be used on stream st: order st behind the stream of the previous call if it differs.
// Calls that stay on one stream (the normal case) cost nothing and put nothing between their kernels.
int order_after_previous(spiir_bank* bk, cudaStream_t st)
{
    if (bk->last_stream_valid && bk->last_stream != st) {
        if (!bk->ev_order) CU_TRY(cudaEventCreateWithFlags(&bk->ev_order, cudaEventDisableTiming));
        CU_TRY(cudaEventRecord(bk->ev_order, bk->last_stream));
        CU_TRY(cudaStreamWaitEvent(st, bk->ev_order, 0));
    }
    bk->last_stream = st;
    bk->last_stream_valid = true;
    return SPIIR_OK;
}

// (re)allocate the tape so that a chunk of n samples fits behind the history; keeps the history
int ensure_tape(spiir_bank* bk, int64_t n, cudaStream_t st)
{
    const int64_t need = round_up(bk->D, 4) + n + 16;
    if (bk->cap >= need && bk->pos + n + 8 <= bk->cap) return SPIIR_OK;
    const int64_t hist0 = round_up(bk->D, 4);
    if (bk->cap < need) {
        const int64_t cap = round_up(bk->D, 4) + std::max<int64_t>(4 * n, 1 << 16) + 16;
        // growing the tape allocates and synchronises the stream (documented in spiir.h: only calls longer than any
        // before, beyond the 65 536 samples the tape is created for)
        float* nt[2] = {nullptr, nullptr};
        cudaError_t e = cudaMalloc((void**)&nt[0], (size_t)cap * sizeof(float));
        if (e == cudaSuccess) e = cudaMalloc((void**)&nt[1], (size_t)cap * sizeof(float));
        if (e == cudaSuccess) e = cudaMemsetAsync(nt[0], 0, (size_t)cap * sizeof(float), st);
        if (e == cudaSuccess) e = cudaMemsetAsync(nt[1], 0, (size_t)cap * sizeof(float), st);
        if (e == cudaSuccess && bk->tape[bk->cur] && bk->D > 0)
            e = cudaMemcpyAsync(nt[0] + hist0 - bk->D, bk->tape[bk->cur] + bk->pos - bk->D,
                                (size_t)bk->D * sizeof(float), cudaMemcpyDeviceToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) {
            cudaFree(nt[0]);
            cudaFree(nt[1]);
            return fail(e == cudaErrorMemoryAllocation ? SPIIR_ENOMEM : SPIIR_ECUDA, "input tape: %s", cudaGetErrorString(e));
        }
        cudaFree(bk->tape[0]);
        cudaFree(bk->tape[1]);
        bk->tape[0] = nt[0];
        bk->tape[1] = nt[1];
        bk->cur = 0;
        bk->cap = cap;
        bk->pos = hist0;
        return SPIIR_OK;
    }
    // compact: move the last D samples to the front of the other buffer
    const int other = bk->cur ^ 1;
    if (bk->D > 0)
        CU_TRY(cudaMemcpyAsync(bk->tape[other] + hist0 - bk->D, bk->tape[bk->cur] + bk->pos - bk->D,
                               (size_t)bk->D * sizeof(float), cudaMemcpyDeviceToDevice, st));
    bk->cur = other;
    bk->pos = hist0;
    return SPIIR_OK;
}

// The compiled (F, W) register/warp blockings of the filter kernel: F filters per thread, W warps per CTA.
// W is chosen so that the register file of an SM is full with one resident CTA (the shared-memory window of
// a 16 384-sample chunk behind a 16 383-sample history allows only one).
const void* select_kernel(int F, int W, int NC, bool g, bool peak = false, bool seg = false)
{
    if (seg) {      // shared tiles of small templates: F = 8 / 16 warps, and F = 4 / 16 and F = 2 / 32 warps for tiny ones
#define SPIIR_SEG(F_, W_, P_)                                                                       \
        if (F == F_ && W == W_) {                                                                   \
            if (g) return (const void*)spiir_filter_kernel<F_, W_, 1, true, 1, P_, true>;           \
            if (NC == 4) return (const void*)spiir_filter_kernel<F_, W_, 4, false, 1, P_, true>;    \
            if (NC == 2) return (const void*)spiir_filter_kernel<F_, W_, 2, false, 1, P_, true>;    \
            return (const void*)spiir_filter_kernel<F_, W_, 1, false, 1, P_, true>;                 \
        }
        if (peak) { SPIIR_SEG(8, 16, true) SPIIR_SEG(4, 16, true) SPIIR_SEG(2, 32, true) }
        else { SPIIR_SEG(8, 16, false) SPIIR_SEG(4, 16, false) SPIIR_SEG(2, 32, false) }
#undef SPIIR_SEG
        return nullptr;
    }
#define SPIIR_VARIANT_P(F_, W_, M_, P_)                                                        \
        if (g) return (const void*)spiir_filter_kernel<F_, W_, 1, true, M_, P_>;               \
        if (NC == 4) return (const void*)spiir_filter_kernel<F_, W_, 4, false, M_, P_>;        \
        if (NC == 2) return (const void*)spiir_filter_kernel<F_, W_, 2, false, M_, P_>;        \
        return (const void*)spiir_filter_kernel<F_, W_, 1, false, M_, P_>;
#define SPIIR_VARIANT(F_, W_, M_)                                                              \
    if (F == F_ && W == W_) {                                                                  \
        if (peak) { SPIIR_VARIANT_P(F_, W_, M_, true) }                                        \
        SPIIR_VARIANT_P(F_, W_, M_, false)                                                     \
    }
    SPIIR_VARIANT(16, 8, 1)
    SPIIR_VARIANT(8, 8, 2)
    SPIIR_VARIANT(8, 16, 1)
    SPIIR_VARIANT(4, 8, 3)
    SPIIR_VARIANT(4, 16, 1)
    SPIIR_VARIANT(4, 32, 1)
    SPIIR_VARIANT(2, 32, 1)
    SPIIR_VARIANT(1, 32, 1)
#undef SPIIR_VARIANT
#undef SPIIR_VARIANT_P
    return nullptr;
}

bool valid_blocking(int F, int W) { return select_kernel(F, W, 1, false) != nullptr; }

// Single-launch time-parallel kernel: the blockings that own an SM (one CTA per SM), shared-memory window, no trigger
// reduction, no shared tiles (those take the three-launch form of the same path).
const void* select_scan_fused_kernel(int F, int W, int NC)
{
#define SPIIR_FUSED(F_, W_)                                                                         \
    if (F == F_ && W == W_) {                                                                        \
        if (NC == 4) return (const void*)spiir_scan_fused_kernel<F_, W_, 4, false, false, false>;    \
        if (NC == 2) return (const void*)spiir_scan_fused_kernel<F_, W_, 2, false, false, false>;    \
        return (const void*)spiir_scan_fused_kernel<F_, W_, 1, false, false, false>;                 \
    }
    SPIIR_FUSED(16, 8)
    SPIIR_FUSED(8, 16)
    SPIIR_FUSED(4, 16)
    SPIIR_FUSED(4, 32)
    SPIIR_FUSED(2, 32)
    SPIIR_FUSED(1, 32)
#undef SPIIR_FUSED
    return nullptr;
}

// F = 4 takes 16 warps: with 32 (64 registers per thread) the body spills and measures 34 % of peak against 41 %
int default_warps(int F) { return F >= 16 ? 8 : (F >= 4 ? 16 : 32); }

// shared memory besides the window copies
// variants compiled for several CTAs per SM keep the CTA-wide barrier and need only 2 partial-sum buffers
int part_buffers(int F, int W) { return (W == 8 && (F == 8 || F == 4)) ? 2 : kPB; }
size_t fixed_smem(int F, int W) { return filter_smem_bytes(W, 1, 0, true, nullptr, part_buffers(F, W)); }

// allow the kernel to use all opt-in shared memory (once per variant and bank)
int configure_kernel(spiir_bank* bk, bool g, const void** fn, bool peak = false)
{
    *fn = select_kernel(bk->F, bk->W, bk->NC, g, peak, bk->segmented);
    if (!*fn) return fail(SPIIR_EINVAL, "unsupported blocking F=%d W=%d%s", bk->F, bk->W, bk->segmented ? " (shared tiles of small templates)" : "");
    if (!bk->configured[g][peak]) {
        CU_TRY(cudaFuncSetAttribute(*fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bk->smem_optin));
        bk->configured[g][peak] = true;
    }
    return SPIIR_OK;
}

int launch_filter(spiir_bank* bk, bool g, const FilterParams& p, dim3 grid, size_t smem, cudaStream_t st)
{
    const void* fn = nullptr;
    int rc = configure_kernel(bk, g, &fn, p.peaks != nullptr);     // the trigger reduction is a variant of its own
    if (rc) return rc;
    void* args[] = {(void*)&p};
    CU_TRY(cudaLaunchKernel(fn, grid, dim3((unsigned)(kWarp * bk->W), 1, 1), args, smem, st));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return SPIIR_OK;
}

int occupancy(spiir_bank* bk, bool g, size_t smem, int* occ)
{
    const void* fn = nullptr;
    int rc = configure_kernel(bk, g, &fn);
    if (rc) return rc;
    CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, fn, kWarp * bk->W, smem));
    return SPIIR_OK;
}

int cached_occupancy(spiir_bank* bk, bool g, size_t smem, int* occ)
{
    for (int i = 0; i < bk->occ_n; ++i)
        if (bk->occ_smem[i] == smem && bk->occ_gmem[i] == g) { *occ = bk->occ_val[i]; return SPIIR_OK; }
    int rc = occupancy(bk, g, smem, occ);
    if (rc) return rc;
    const int i = bk->occ_n < 8 ? bk->occ_n++ : 7;
    bk->occ_smem[i] = smem; bk->occ_gmem[i] = g; bk->occ_val[i] = *occ;
    return SPIIR_OK;
}

FilterParams base_params(const spiir_bank* bk)
{
    FilterParams p{};
    p.coef = bk->coef;
    p.item_round0 = bk->item_round0; p.work = bk->work; p.n_items = bk->n_items;
    p.uniform_groups = bk->uniform_groups ? 1 : 0;
    p.canon = bk->canon;
    return p;
}

// Tiny chunk through the streaming kernels: independent warps + a combine pass.
const void* select_stream_kernel(int F, int NC)
{
#define SPIIR_STREAM(F_)                                                            \
    if (F == F_) {                                                                  \
        if (NC == 4) return (const void*)spiir_stream_kernel<F_, 4>;                \
        if (NC == 2) return (const void*)spiir_stream_kernel<F_, 2>;                \
        return (const void*)spiir_stream_kernel<F_, 1>;                             \
    }
    SPIIR_STREAM(4)
    SPIIR_STREAM(8)
#undef SPIIR_STREAM
    return nullptr;
}

bool stream_applies(const spiir_bank* bk, int w0, int64_t n)
{
    return bk->opt.path == SPIIR_PATH_STREAM && n <= kStreamMax && !bk->gmem_only && select_stream_kernel(bk->F, bk->NC) &&
           stream_smem_bytes(bk->F, bk->NC, w0 + n, nullptr) <= bk->smem_optin;
}

// xnew != nullptr: the chunk is not on the tape yet; the kernel reads it from xnew and CTA 0 appends it at `append`.
int run_stream(spiir_bank* bk, const float* xwin, int w0, int64_t n, float* snr, int64_t ld, cudaStream_t st, u64* peaks,
               const float* xnew = nullptr, float* append = nullptr)
{
    NvtxRange range("spiir_filter: tiny-chunk streaming path");
    const void* fn = select_stream_kernel(bk->F, bk->NC);
    if (!fn) return fail(SPIIR_EINVAL, "no streaming kernel for F=%d NC=%d", bk->F, bk->NC);
    if (!bk->stream_configured) {
        CU_TRY(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bk->smem_optin));
        bk->stream_configured = true;
    }
    if (!bk->stream_scratch)
        CU_TRY(cudaMalloc((void**)&bk->stream_scratch, (size_t)std::max<int64_t>(bk->n_tiles, 1) * kStreamMax * sizeof(u64)));
    u64* scratch = bk->stream_scratch;
    const int kStreamWarps = stream_warps(bk->F);
    const size_t smem = stream_smem_bytes(bk->F, bk->NC, w0 + n, nullptr);
    if (bk->stream_occ_smem != smem) {          // one driver query per window size, not per call
        int occ = 0;
        CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, kWarp * kStreamWarps, smem));
        if (occ < 1) return fail(SPIIR_ECUDA, "streaming kernel does not fit on an SM (smem %zu)", smem);
        bk->stream_occ = occ;
        bk->stream_occ_smem = smem;
    }
    const int occ = bk->stream_occ;
    StreamParams p{};
    p.coef = bk->coef; p.y = bk->y;
    p.xwin = xwin; p.w0 = w0; p.n = (int32_t)n; p.n_tiles = bk->n_tiles; p.scratch = scratch;
    p.xnew = xnew; p.append = append;
    const int64_t ctas = std::min<int64_t>((bk->n_tiles + kStreamWarps - 1) / kStreamWarps, (int64_t)bk->n_sm * occ);
    // scan_launches = 1: one launch per call -- the grid never exceeds what is resident at once, so it can meet at a barrier
    // between the tile phase and the combine phase.  Default: the combine as a kernel of its own, launched programmatically;
    // its small CTAs run beside the first CTAs of the next call's tile kernel, which measures 2 % faster on cfg4
    // (46.9 against 47.8 us per call).
    const bool one_launch = bk->opt.scan_launches == 1;
    if (one_launch) {
        if (!bk->stream_barrier) {
            CU_TRY(cudaMalloc((void**)&bk->stream_barrier, sizeof(unsigned long long)));
            CU_TRY(cudaMemsetAsync(bk->stream_barrier, 0, sizeof(unsigned long long), st));
            bk->stream_arrivals = 0;
        }
        bk->stream_arrivals += (unsigned long long)ctas;
        p.barrier = bk->stream_barrier; p.target = bk->stream_arrivals;
        p.tile_begin = bk->tile_begin; p.n_templates = (int32_t)bk->T; p.snr = snr; p.ld = ld; p.peaks = peaks;
    }
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    {
        // programmatic dependent launch: the grid is set up and the first tile requested while the previous kernel in the
        // stream (normally the previous call's combine pass) drains; the kernel waits for it before it reads anything else
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)ctas, 1, 1);
        cfg.blockDim = dim3(kWarp * kStreamWarps, 1, 1);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        void* args[] = {(void*)&p};
        CU_TRY(cudaLaunchKernelExC(&cfg, fn, args));
    }
    const int64_t total = bk->T * n;
    if (!one_launch) {
        // programmatic dependent launch: the combine grid is set up while the streaming kernel drains and waits
        // (griddepcontrol.wait in the kernel) for its results
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)((total + 255) / 256), 1, 1);
        cfg.blockDim = dim3(256, 1, 1);
        cfg.dynamicSmemBytes = 0;
        cfg.stream = st;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        CU_TRY(cudaLaunchKernelEx(&cfg, spiir_stream_combine_kernel, (const u64*)scratch,
                                  (const int64_t*)bk->tile_begin, (int32_t)bk->T, (int32_t)n, snr, ld, peaks));
    }
    g_launches.fetch_add(one_launch ? 1 : 2, std::memory_order_relaxed);
    CU_TRY(cudaGetLastError());
    bk->last_path = SPIIR_PATH_STREAM;
    return SPIIR_OK;
}

// Run the filter kernels over n samples whose window starts at xwin (aligned), sample 0 at xwin[w0].
// x_dev / append: the chunk is not on the tape yet; every path but the single-launch scan kernel (which reads the caller's
// buffer and appends the chunk itself) first copies it there.
int run_chunk(spiir_bank* bk, const float* xwin, int w0, int64_t n, float* snr, int64_t ld, cudaStream_t st, u64* peaks,
              const float* x_dev, float* append)
{
    bool appended = false;
    auto append_chunk = [&]() -> cudaError_t {
        if (appended) return cudaSuccess;
        appended = true;
        return cudaMemcpyAsync(append, x_dev, (size_t)n * sizeof(float), cudaMemcpyDeviceToDevice, st);
    };
    const size_t smem_cap = bk->smem_optin;
    // window floats per copy that fit beside the reduction buffers (a copy is padded by up to 47 floats)
    const int64_t max_win = ((int64_t)smem_cap - (int64_t)fixed_smem(bk->F, bk->W)) / (4 * bk->NC) - 48;
    const bool gmem = bk->gmem_only;          // history alone does not fit: read x through L1/L2
    int path = bk->opt.path;
    if (stream_applies(bk, w0, n)) { CU_TRY(append_chunk()); return run_stream(bk, xwin, w0, n, snr, ld, st, peaks); }
    // ---- how much time-parallelism is needed to fill the machine?  The scan path does the recurrence twice, so it
    // only pays when the bank leaves at least half of the SMs idle (cfg2: 128 items on 148 SMs run 1.7x faster
    // sequentially).
    int64_t n_seg = 1;
    if (path == SPIIR_PATH_SCAN || (path == SPIIR_PATH_AUTO && 2 * bk->n_items <= bk->n_sm && n >= 4 * kTS)) {
        const int64_t max_seg = std::max<int64_t>(1, n / kTS);
        int64_t want = bk->opt.scan_segments > 0 ? bk->opt.scan_segments
                                                 : ((int64_t)bk->n_sm + bk->n_items - 1) / bk->n_items;   // one wave of CTAs: longer segments amortise the window staging
        n_seg = std::min(std::max<int64_t>(want, 1), max_seg);
        if (n_seg < 2 && path != SPIIR_PATH_SCAN) n_seg = 1;
    }
    if (n_seg <= 1) {
        // ------------------------------------------------ sequential-in-time path
        NvtxRange range("spiir_filter: throughput path");
        CU_TRY(append_chunk());
        bk->last_path = SPIIR_PATH_THROUGHPUT;
        int64_t sub = n;
        if (!gmem) {
            const int64_t sub_max = std::max<int64_t>(kTS, (max_win - w0) / kTS * kTS);
            const int64_t n_launch = (n + sub_max - 1) / sub_max;                 // balanced sub-launches
            sub = std::min(sub_max, round_up((n + n_launch - 1) / n_launch, kTS));
        }
        for (int64_t off = 0; off < n; off += sub) {
            const int64_t ns = std::min(sub, n - off);
            FilterParams p = base_params(bk);
            p.y_in = bk->y; p.y_out = bk->y; p.y_in_stride = 0; p.y_out_stride = 0; p.store_last_only = 1;
            p.xwin = xwin + off; p.w0 = w0; p.n = ns; p.seg_len = ns;
            p.snr = snr ? snr + 2 * off : nullptr; p.ld = ld;
            p.peaks = peaks; p.peak_off = off;
            const size_t smem = filter_smem_bytes(bk->W, bk->NC, w0 + ns, gmem, nullptr, part_buffers(bk->F, bk->W));
            int occ = 1;
            int rc = cached_occupancy(bk, gmem, smem, &occ);
            if (rc) return rc;
            if (occ < 1) return fail(SPIIR_ECUDA, "filter kernel does not fit on an SM (smem %zu)", smem);
            dim3 grid((unsigned)std::min<int64_t>(bk->n_items, (int64_t)bk->n_sm * occ), 1, 1);
            rc = launch_filter(bk, gmem, p, grid, smem, st);
            if (rc) return rc;
        }
        return SPIIR_OK;
    }
    // ---------------------------------------------------- time-parallel scan path (north_star (4))
    NvtxRange range("spiir_filter: time-parallel path");
    bk->last_path = SPIIR_PATH_SCAN;
    // segments of >= 64 samples in steps of 16 (two register tiles; keeps every segment's window 16-byte aligned): cfg1's
    // 4096-sample call over 4 items becomes 37 segments of 112 samples = 148 CTAs instead of 32 of 128 = 128 CTAs
    int64_t seg_len = std::max<int64_t>(kTS, round_up((n + n_seg - 1) / n_seg, 16));
    if (!gmem && w0 + seg_len > max_win) seg_len = std::max<int64_t>(kTS, (max_win - w0) / kTS * kTS);
    n_seg = (n + seg_len - 1) / seg_len;
    if (n_seg > bk->scan_cap_seg) {
        cudaFree(bk->zbuf); cudaFree(bk->cbuf);
        bk->zbuf = bk->cbuf = nullptr;
        bk->scan_cap_seg = 0;
        const size_t bytes = (size_t)n_seg * 2 * bk->n_slots * sizeof(float);
        CU_TRY(cudaMalloc((void**)&bk->zbuf, bytes));
        CU_TRY(cudaMalloc((void**)&bk->cbuf, bytes));
        bk->scan_cap_seg = n_seg;
    }
    const size_t smem = filter_smem_bytes(bk->W, bk->NC, w0 + seg_len, gmem, nullptr, part_buffers(bk->F, bk->W));
    int occ = 1;
    int rc = cached_occupancy(bk, gmem, smem, &occ);
    if (rc) return rc;
    if (occ < 1) return fail(SPIIR_ECUDA, "filter kernel does not fit on an SM (smem %zu)", smem);
    const unsigned gx = (unsigned)bk->n_items;
    // ---- one cooperative launch when every CTA of the (items x segments) grid is resident (cfg0, cfg1)
    const void* fused = (n_seg > 1 && !gmem && !peaks && !bk->segmented && bk->opt.scan_launches != 3)
                            ? select_scan_fused_kernel(bk->F, bk->W, bk->NC) : nullptr;
    if (fused) {
        if (!bk->scan_fused_configured) {
            CU_TRY(cudaFuncSetAttribute(fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bk->smem_optin));
            bk->scan_fused_configured = true;
        }
        if (bk->scan_fused_occ < 0 || bk->scan_fused_occ_smem != smem) {
            int o = 0;
            CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, fused, kWarp * bk->W, smem));
            bk->scan_fused_occ = o;
            bk->scan_fused_occ_smem = smem;
        }
        if ((int64_t)gx * n_seg > (int64_t)bk->n_sm * bk->scan_fused_occ) fused = nullptr;
    }
    if (fused) {
        if (!bk->scan_barrier) {
            CU_TRY(cudaMalloc((void**)&bk->scan_barrier, sizeof(unsigned long long)));
            CU_TRY(cudaMemsetAsync(bk->scan_barrier, 0, sizeof(unsigned long long), st));
            bk->scan_arrivals = 0;
        }
        ScanFusedParams sp{};
        sp.pass1 = base_params(bk);
        sp.pass1.y_in = nullptr; sp.pass1.y_out = bk->zbuf; sp.pass1.y_out_stride = 2 * bk->n_slots; sp.pass1.store_last_only = 0;
        sp.pass1.xwin = xwin; sp.pass1.w0 = w0; sp.pass1.n = (n_seg - 1) * seg_len; sp.pass1.seg_len = seg_len;
        sp.pass1.snr = nullptr; sp.pass1.ld = 0;
        sp.pass2 = base_params(bk);
        sp.pass2.y_in = bk->cbuf; sp.pass2.y_in_stride = 2 * bk->n_slots; sp.pass2.y_out = bk->y; sp.pass2.y_out_stride = 0;
        sp.pass2.store_last_only = 1;
        sp.pass2.xwin = xwin; sp.pass2.w0 = w0; sp.pass2.n = n; sp.pass2.seg_len = seg_len;
        sp.pass2.snr = snr; sp.pass2.ld = ld;
        sp.cbuf = bk->cbuf; sp.z = bk->zbuf; sp.y = bk->y; sp.n_slots = bk->n_slots; sp.n_seg = (int32_t)n_seg;
        sp.xnew = x_dev; sp.append = append;
        sp.barrier = bk->scan_barrier;
        sp.target = bk->scan_arrivals + (unsigned long long)gx * (unsigned long long)n_seg;
        bk->scan_arrivals += 2ull * gx * (unsigned long long)n_seg;      // two grid-wide barriers per launch
        void* args[] = {(void*)&sp};
        // cooperative launch: the driver checks that the whole grid is resident, which the two grid-wide barriers need
        CU_TRY(cudaLaunchCooperativeKernel(fused, dim3(gx, (unsigned)n_seg, 1), dim3((unsigned)(kWarp * bk->W), 1, 1), args, smem, st));
        g_launches.fetch_add(1, std::memory_order_relaxed);
        return SPIIR_OK;
    }
    CU_TRY(append_chunk());
    if (n_seg > 1) {
        // pass 1: zero-state end values of segments 0 .. n_seg-2 (no sums, no output)
        FilterParams p = base_params(bk);
        p.y_in = nullptr; p.y_out = bk->zbuf; p.y_out_stride = 2 * bk->n_slots; p.store_last_only = 0;
        p.xwin = xwin; p.w0 = w0; p.n = (n_seg - 1) * seg_len; p.seg_len = seg_len;
        p.snr = nullptr; p.ld = 0;
        dim3 grid(gx, (unsigned)(n_seg - 1), 1);
        rc = launch_filter(bk, gmem, p, grid, smem, st);
        if (rc) return rc;
    }
    {
        // carry scan: c_0 = y, c_{q+1} = a1^seg_len c_q + z_q   (double precision)
        const int threads = 256;
        const unsigned blocks = (unsigned)((bk->n_slots + threads - 1) / threads);
        spiir_scan_carry_kernel<<<blocks, threads, 0, st>>>(bk->coef, (int32_t)bk->F, bk->y, bk->zbuf, bk->cbuf,
                                                            bk->n_slots, (int32_t)n_seg, seg_len);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        CU_TRY(cudaGetLastError());
    }
    {
        // pass 2: every segment from its true start state, full sums and output; last segment stores y
        FilterParams p = base_params(bk);
        p.y_in = bk->cbuf; p.y_in_stride = 2 * bk->n_slots; p.y_out = bk->y; p.y_out_stride = 0; p.store_last_only = 1;
        p.xwin = xwin; p.w0 = w0; p.n = n; p.seg_len = seg_len;
        p.snr = snr; p.ld = ld;
        p.peaks = peaks; p.peak_off = 0;
        dim3 grid(gx, (unsigned)n_seg, 1);
        rc = launch_filter(bk, gmem, p, grid, smem, st);
        if (rc) return rc;
    }
    return SPIIR_OK;
}

// Relative cost per padded filter slot of the compiled blockings, measured on padding-free banks that fill whole waves of CTA
// items (cfg3 for F = 16; banks of 4- to 256-filter templates below; product build): plain tiles F = 16 / 8 warps 56.2 %,
// F = 8 / 16 warps 53.7 %, F = 4 / 16 warps 47.5 %, F = 2 / 32 warps 36 %, F = 1 (one warp per template) ~ 21 %
// of FP32 peak; shared tiles F = 8: 50.5 % for segments of 8 or 16 lanes, 42.8 % for full 4-lane
// segments (they share a load phase with a neighbour), F = 4: 42.4 / 45.6 / 43.5 % for 4 / 8 / 16 lanes, F = 2: 28 - 34 %.
double slot_cost(int F) { return F == 16 ? 1.0 : (F == 8 ? 1.05 : (F == 4 ? 1.18 : (F == 2 ? 1.56 : 2.6))); }
double shared_tile_cost(int F, int w, double fill)
{
    if (F == 8) return w == 4 ? 1.13 + 0.18 * fill * fill : 1.11;      // padding lanes broadcast: fewer conflicts when not full
    if (F == 4) return w == 4 ? 1.33 : (w == 8 ? 1.23 : 1.29);
    return w == 4 ? 2.0 : (w == 8 ? 1.8 : 1.66);
}

int choose_F(int32_t T, const int64_t* off, int requested, double* cost_out = nullptr)
{
    double best = 0;
    int bestF = 0;
    for (int F : {16, 8, 4, 2, 1}) {
        if (requested && F != requested) continue;
        const int64_t per = 32LL * F;
        double padded = 0;
        for (int32_t t = 0; t < T; ++t) padded += (double)((off[t + 1] - off[t] + per - 1) / per * per);
        padded *= slot_cost(F);
        if (!bestF || padded < best) { best = padded; bestF = F; }
    }
    if (cost_out) *cost_out = best;
    return bestF ? bestF : 8;
}

}  // namespace

extern "C" {

const char* spiir_last_error(void) { return g_err; }
int64_t spiir_kernel_launches(void) { return g_launches.load(); }
int32_t spiir_version(void) { return 100; }

int spiir_layout_probe(int32_t T, const int64_t* off, const int32_t* delays, int32_t F, int32_t W, int32_t NC,
                       int64_t* slot_of_filter, double* stats, int32_t pack_small)
{
    if (!off || !delays) return fail(SPIIR_EINVAL, "null argument");
    if (T <= 0) return fail(SPIIR_EINVAL, "n_templates must be >= 1");
    if (off[0] != 0) return fail(SPIIR_EINVAL, "filter_offsets[0] must be 0");
    for (int32_t t = 0; t < T; ++t)
        if (off[t + 1] <= off[t]) return fail(SPIIR_EINVAL, "template %d has no filters (offsets must increase)", t);
    if (!valid_blocking(F, W)) return fail(SPIIR_EINVAL, "unsupported blocking: filters_per_thread %d with warps_per_cta %d", F, W);
    if (NC != 1 && NC != 2 && NC != 4) return fail(SPIIR_EINVAL, "window_copies must be 1, 2 or 4");
    const int64_t K = off[T];
    for (int64_t k = 0; k < K; ++k)
        if (delays[k] < 0) return fail(SPIIR_EINVAL, "negative delay at filter %lld", (long long)k);
    HostLayout L;
    try {
        std::vector<float> zeros((size_t)2 * K, 0.f);
        L = build_layout(T, off, zeros.data(), zeros.data(), delays, F, W, NC, pack_small != 0);
    } catch (const std::bad_alloc&) {
        return fail(SPIIR_ENOMEM, "out of host memory building the bank layout");
    }
    if (slot_of_filter) memcpy(slot_of_filter, L.slot_of_filter.data(), (size_t)K * sizeof(int64_t));
    if (stats) {
        stats[0] = (double)L.n_slots;
        stats[1] = (double)L.n_tiles;
        stats[2] = (double)(L.item_round0.size() - 1);
        stats[3] = (double)(L.work.size() / (size_t)W);
        stats[4] = L.avg_conflict_degree;
        stats[5] = L.n_slots ? 1.0 - (double)K / (double)L.n_slots : 0.0;
        stats[6] = L.uniform_groups ? 1.0 : 0.0;
        stats[7] = L.segmented ? 1.0 : 0.0;
    }
    return SPIIR_OK;
}

int spiir_bank_create(spiir_bank** out, int32_t T, const int64_t* off, const float* a1, const float* b0,
                      const int32_t* delays, int32_t device, const spiir_options* opt)
{
    if (out) *out = nullptr;
    if (!out || !off || !a1 || !b0 || !delays) return fail(SPIIR_EINVAL, "null argument");
    if (T <= 0) return fail(SPIIR_EINVAL, "n_templates must be >= 1");
    if (off[0] != 0) return fail(SPIIR_EINVAL, "filter_offsets[0] must be 0");
    for (int32_t t = 0; t < T; ++t)
        if (off[t + 1] <= off[t]) return fail(SPIIR_EINVAL, "template %d has no filters (offsets must increase)", t);
    const int64_t K = off[T];
    int64_t D = 0;
    for (int64_t k = 0; k < K; ++k) {
        const float re = a1[2 * k], im = a1[2 * k + 1];
        if (!std::isfinite(re) || !std::isfinite(im) || !std::isfinite(b0[2 * k]) || !std::isfinite(b0[2 * k + 1]))
            return fail(SPIIR_EINVAL, "non-finite coefficient at filter %lld", (long long)k);
        if ((double)re * re + (double)im * im >= 1.0) return fail(SPIIR_EINVAL, "|a1| >= 1 at filter %lld", (long long)k);
        if (delays[k] < 0) return fail(SPIIR_EINVAL, "negative delay at filter %lld", (long long)k);
        D = std::max<int64_t>(D, delays[k]);
    }
    spiir_options o{};
    o.struct_size = (int32_t)sizeof(o);
    if (opt) {
        if (opt->struct_size < (int32_t)(4 * sizeof(int32_t))) return fail(SPIIR_EINVAL, "bad spiir_options.struct_size");
        memcpy(&o, opt, std::min<size_t>((size_t)opt->struct_size, sizeof(o)));
        if (o.path < SPIIR_PATH_AUTO || o.path > SPIIR_PATH_STREAM) return fail(SPIIR_EINVAL, "bad path option");
        if (o.filters_per_thread != 0 && o.filters_per_thread != 1 && o.filters_per_thread != 2 &&
            o.filters_per_thread != 4 && o.filters_per_thread != 8 && o.filters_per_thread != 16)
            return fail(SPIIR_EINVAL, "filters_per_thread must be 0, 1, 2, 4, 8 or 16");
        if (o.scan_segments < 0) return fail(SPIIR_EINVAL, "scan_segments must be >= 0");
        if (o.warps_per_cta != 0 && o.warps_per_cta != 8 && o.warps_per_cta != 16 && o.warps_per_cta != 32)
            return fail(SPIIR_EINVAL, "warps_per_cta must be 0, 8, 16 or 32");
        if (o.window_copies != 0 && o.window_copies != 1 && o.window_copies != 2 && o.window_copies != 4)
            return fail(SPIIR_EINVAL, "window_copies must be 0, 1, 2 or 4");
        if (o.small_templates < 0 || o.small_templates > 2) return fail(SPIIR_EINVAL, "small_templates must be 0, 1 or 2");
        if (o.scan_launches != 0 && o.scan_launches != 1 && o.scan_launches != 3)
            return fail(SPIIR_EINVAL, "scan_launches must be 0, 1 or 3");
    }
    // ---- blocking: F filters per thread, W warps per CTA, shared tiles or not (host logic, no device needed)
    const bool stream = (o.path == SPIIR_PATH_STREAM);     // tiny chunks: small CTAs, several per SM
    double plain_cost = 0;
    int F = stream && !o.filters_per_thread ? 4 : choose_F(T, off, o.filters_per_thread, &plain_cost);
    int W = o.warps_per_cta ? o.warps_per_cta : (stream ? 8 : default_warps(F));
    bool segmented = false;
    // Small templates (<= 128 filters) can share warp tiles (PAPER.md:L333-L335 size-aware mapping):
    // blocking F = 8 / 16 warps.  Taken when asked for, or by itself when its estimated cost is lower.
    // A bank that fits one CTA at one filter per lane (<= 32 warps x 32 lanes) is bound by latency, not by issue slots:
    // one filter per thread (PAPER.md:L335 one warp per small template) spreads it over the most warps.
    bool tiny = false;
    if (!stream && !o.filters_per_thread && o.small_templates != 1 && (o.warps_per_cta == 0 || o.warps_per_cta == 32)) {
        int64_t slots1 = 0;
        for (int32_t t = 0; t < T; ++t) slots1 += round_up(off[t + 1] - off[t], kWarp);
        if (slots1 <= 32 * kWarp) { F = 1; W = 32; tiny = true; }
    }
    if (!stream && !tiny && o.small_templates != 2) {
        double best_packed = 0;
        int best_F = 0;
        bool any_small = false;
        for (int Fs : {8, 4, 2}) {
            const int Ws = default_warps(Fs);
            if ((o.filters_per_thread && o.filters_per_thread != Fs) || (o.warps_per_cta && o.warps_per_cta != Ws)) continue;
            double packed = 0;
            bool small = false;
            const int64_t per = 32LL * Fs;
            for (int32_t t = 0; t < T; ++t) {
                const int64_t Kt = off[t + 1] - off[t];
                const int w = segment_lanes(Kt, Fs, true);
                small |= (w < kWarp);
                packed += w < kWarp ? shared_tile_cost(Fs, w, (double)Kt / (double)(w * Fs)) * (double)(w * Fs)
                                    : slot_cost(Fs) * (double)((Kt + per - 1) / per * per);
            }
            if (small && (!best_F || packed < best_packed)) { best_packed = packed; best_F = Fs; }
            any_small |= small;
        }
        if (any_small && best_F && (o.small_templates == 1 || best_packed < plain_cost)) {
            F = best_F; W = default_warps(best_F); segmented = true;
        }
    }
    // The (filters_per_thread, warps_per_cta) pair must be one a compiled kernel serves: checked here, not at the first
    // spiir_filter.  When only one of the two was requested the other follows it.
    if (!segmented && !valid_blocking(F, W)) {
        if (o.filters_per_thread && o.warps_per_cta)
            return fail(SPIIR_EINVAL, "unsupported blocking: filters_per_thread %d with warps_per_cta %d%s", F, W,
                        stream ? " (SPIIR_PATH_STREAM banks use 8 warps by default: filters_per_thread 4, 8 or 16)" : "");
        if (o.warps_per_cta) {               // W fixed: the largest F that pairs with it
            int f_ok = 0;
            for (int f : {16, 8, 4, 2, 1})
                if (valid_blocking(f, W)) { f_ok = f; break; }
            F = f_ok;
        } else if (stream) {                 // F fixed, W = 8 comes with the streaming path
            return fail(SPIIR_EINVAL, "SPIIR_PATH_STREAM serves filters_per_thread 4, 8 or 16 (got %d)", F);
        } else {
            W = default_warps(F);
        }
        if (!valid_blocking(F, W))
            return fail(SPIIR_EINVAL, "unsupported blocking: filters_per_thread %d with warps_per_cta %d", F, W);
    }
    if (segmented && !select_kernel(F, W, 1, false, false, true))
        return fail(SPIIR_EINVAL, "shared tiles of small templates need the (8, 16), (4, 16) or (2, 32) blocking");

    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev <= 0)
        return fail(SPIIR_ECUDA, "no CUDA device available (this library has no CPU fallback)");
    if (device < 0 || device >= n_dev) return fail(SPIIR_EINVAL, "device %d out of range", device);
    DeviceGuard dg(device);
    CU_TRY(dg.err);

    spiir_bank* bk = new (std::nothrow) spiir_bank();
    if (!bk) return fail(SPIIR_ENOMEM, "out of host memory");
    bk->device = device;
    bk->opt = o;
    bk->T = T; bk->K = K; bk->D = D;
    bk->F = F; bk->W = W; bk->segmented = segmented;
    cudaDeviceProp prop;
    cudaError_t e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) {
        free_bank(bk);
        return fail(SPIIR_ECUDA, "cudaGetDeviceProperties: %s", cudaGetErrorString(e));
    }
    bk->n_sm = prop.multiProcessorCount;
    bk->smem_optin = prop.sharedMemPerBlockOptin;
    // Window copies: as many (4, 2, 1 = LDS.128/.64/.32 per filter) as leave room for >= kMinSub samples per
    // launch behind the history; none at all (global-memory reads) if not even one copy of the history fits.
    {
        const int64_t room = (int64_t)bk->smem_optin - (int64_t)fixed_smem(bk->F, bk->W);
        const int64_t hist = round_up(D, 4) + 4 + 48;
        const int64_t kMinSub = 2048;
        bk->NC = 1;
        for (int nc : {4, 2}) {
            if (stream) {                                   // sized for the streaming kernels (one big CTA per SM)
                if (nc == 4) continue;                      // LDS.128 buys nothing there and costs registers
                if (stream_smem_bytes(bk->F, nc, hist + kStreamMax, nullptr) <= bk->smem_optin &&
                    (hist + 2048) * 4 * nc <= room) { bk->NC = nc; break; }
                continue;
            }

            // F >= 8 keeps 2 copies: the LDS.128 variants are short of registers (F = 16: all 255, 8 % slower on cfg2; F = 8: 128
            // with a spill, 1 - 3 % slower on banks of 64- to 256-filter templates)
            if (nc == 4 && bk->F >= 8) continue;
            if ((hist + kMinSub) * 4 * nc <= room) { bk->NC = nc; break; }
        }
        if (o.window_copies == 1 || o.window_copies == 2 || o.window_copies == 4)
            if ((hist + kTS) * 4 * o.window_copies <= room) bk->NC = o.window_copies;
        bk->gmem_only = (hist + kTS) * 4 > room;
        if (bk->gmem_only) bk->NC = 1;
    }
    HostLayout L;
    try {
        L = build_layout(T, off, a1, b0, delays, bk->F, bk->W, bk->NC, bk->segmented);
        bk->segmented = L.segmented;
    } catch (const std::bad_alloc&) {
        free_bank(bk);
        return fail(SPIIR_ENOMEM, "out of host memory building the bank layout");
    }
    bk->n_slots = L.n_slots;
    bk->n_tiles = L.n_tiles;
    bk->n_items = (int32_t)(L.item_round0.size() - 1);
    bk->avg_conflict_degree = L.avg_conflict_degree;
    bk->uniform_groups = L.uniform_groups;
    bk->multi_round = (L.work.size() / (size_t)bk->W) > (L.item_round0.size() - 1);
    if (e == cudaSuccess) e = upload(&bk->coef, L.coef);
    if (e == cudaSuccess) e = upload(&bk->item_round0, L.item_round0);
    if (e == cudaSuccess) e = upload(&bk->work, L.work);
    if (e == cudaSuccess) e = upload(&bk->canon, L.canon);
    if (e == cudaSuccess) e = upload(&bk->tile_begin, L.tile_begin);
    if (e == cudaSuccess) e = upload(&bk->slot_of_filter, L.slot_of_filter);
    if (e == cudaSuccess) e = cudaMalloc((void**)&bk->y, (size_t)std::max<int64_t>(L.n_slots, 1) * 2 * sizeof(float));
    if (e == cudaSuccess) e = cudaMemset(bk->y, 0, (size_t)std::max<int64_t>(L.n_slots, 1) * 2 * sizeof(float));
    if (e != cudaSuccess) {
        free_bank(bk);
        return fail(e == cudaErrorMemoryAllocation ? SPIIR_ENOMEM : SPIIR_ECUDA, "bank upload: %s", cudaGetErrorString(e));
    }
    int rc = ensure_tape(bk, 1 << 14, nullptr);
    if (rc == SPIIR_OK) {
        e = cudaDeviceSynchronize();
        if (e != cudaSuccess) rc = fail(SPIIR_ECUDA, "bank create: %s", cudaGetErrorString(e));
    }
    if (rc != SPIIR_OK) { free_bank(bk); return rc; }
    *out = bk;
    return SPIIR_OK;
}

namespace {

// spiir_filter and spiir_filter_peaks: append the chunk to the tape, run the kernels, advance the tape.
int filter_impl(spiir_bank* bk, const float* x_dev, int64_t n, float* snr_dev, int64_t ld, cudaStream_t st, u64* peaks)
{
    DeviceGuard dg(bk->device);
    CU_TRY(dg.err);
    int rc = order_after_previous(bk, st);
    if (rc) return rc;
    rc = ensure_tape(bk, n, st);
    if (rc) return rc;
    float* tape = bk->tape[bk->cur];
    const int64_t start_al = (bk->pos - bk->D) / 4 * 4;
    const int w0 = (int)(bk->pos - start_al);
    if (stream_applies(bk, w0, n)) {
        // tiny chunk: no separate copy (it would sit between the kernels and break their launch chain); the kernel stages
        // history + chunk itself and appends the chunk to the tape
        rc = run_stream(bk, tape + start_al, w0, n, snr_dev, ld, st, peaks, x_dev, tape + bk->pos);
    } else {
        rc = run_chunk(bk, tape + start_al, w0, n, snr_dev, ld, st, peaks, x_dev, tape + bk->pos);
    }
    if (rc) { bk->poisoned = true; return rc; }
    bk->pos += n;
    return SPIIR_OK;
}

}  // namespace

int spiir_filter(spiir_bank* bk, const float* x_dev, int64_t n, float* snr_dev, int64_t ld, void* stream)
{
    if (!bk) return fail(SPIIR_EINVAL, "null bank");
    if (bk->poisoned) return fail(SPIIR_ESTATE, "bank unusable after an earlier failure");
    if (n < 0 || ld < n) return fail(SPIIR_EINVAL, "need 0 <= n <= ld");
    if (n == 0) return SPIIR_OK;
    if (!x_dev || !snr_dev) return fail(SPIIR_EINVAL, "null device pointer");
    if (n > (int64_t)1 << 30) return fail(SPIIR_EINVAL, "chunk too long");
    return filter_impl(bk, x_dev, n, snr_dev, ld, (cudaStream_t)stream, nullptr);
}

int spiir_filter_peaks(spiir_bank* bk, const float* x_dev, int64_t n, float* snr_dev, int64_t ld, float* power_dev,
                       int32_t* index_dev, void* stream)
{
    if (!bk) return fail(SPIIR_EINVAL, "null bank");
    if (bk->poisoned) return fail(SPIIR_ESTATE, "bank unusable after an earlier failure");
    if (n < 1) return fail(SPIIR_EINVAL, "need n >= 1 (a peak over no samples is undefined)");
    if (snr_dev && ld < n) return fail(SPIIR_EINVAL, "need n <= ld");
    if (!x_dev || (!power_dev && !index_dev)) return fail(SPIIR_EINVAL, "null device pointer");
    if (n > (int64_t)1 << 30) return fail(SPIIR_EINVAL, "chunk too long");
    cudaStream_t st = (cudaStream_t)stream;
    DeviceGuard dg(bk->device);
    CU_TRY(dg.err);
    {
        int rc0 = order_after_previous(bk, st);
        if (rc0) return rc0;
    }
    if (!bk->peaks) CU_TRY(cudaMalloc((void**)&bk->peaks, (size_t)bk->T * sizeof(u64)));
    if (!snr_dev && bk->multi_round) {
        // templates that span several CTA rounds accumulate their sums through SNR rows: give them private ones
        // (allocates and synchronises the stream the first time and whenever n grows: documented in spiir.h)
        if (bk->peak_snr_cap < bk->T * n) {
            CU_TRY(cudaStreamSynchronize(st));
            cudaFree(bk->peak_snr); bk->peak_snr = nullptr; bk->peak_snr_cap = 0;
            CU_TRY(cudaMalloc((void**)&bk->peak_snr, (size_t)bk->T * n * 2 * sizeof(float)));
            bk->peak_snr_cap = bk->T * n;
        }
        snr_dev = bk->peak_snr;
        ld = n;
    }
    CU_TRY(cudaMemsetAsync(bk->peaks, 0, (size_t)bk->T * sizeof(u64), st));
    int rc = filter_impl(bk, x_dev, n, snr_dev, snr_dev ? ld : n, st, bk->peaks);
    if (rc) return rc;
    spiir_unpack_peaks_kernel<<<(unsigned)((bk->T + 255) / 256), 256, 0, st>>>(bk->peaks, power_dev, index_dev, (int32_t)bk->T);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    CU_TRY(cudaGetLastError());
    return SPIIR_OK;
}

int spiir_filter_host_async(spiir_bank* bk, const float* x_host, int64_t n, float* snr_host, int64_t ld)
{
    if (!bk) return fail(SPIIR_EINVAL, "null bank");
    if (n < 0 || ld < n) return fail(SPIIR_EINVAL, "need 0 <= n <= ld");
    if (n == 0) return SPIIR_OK;
    if (!x_host || !snr_host) return fail(SPIIR_EINVAL, "null host pointer");
    DeviceGuard dg(bk->device);
    CU_TRY(dg.err);
    if (!bk->hstream) {
        CU_TRY(cudaStreamCreateWithFlags(&bk->hstream, cudaStreamNonBlocking));
        CU_TRY(cudaStreamCreateWithFlags(&bk->cstream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CU_TRY(cudaEventCreateWithFlags(&bk->ev_done[i], cudaEventDisableTiming));
            CU_TRY(cudaEventCreateWithFlags(&bk->ev_free[i], cudaEventDisableTiming));
        }
    }
    // The chunk is filtered in pieces; the device-to-host copy of one piece (copy stream) overlaps the kernels of
    // the next ("overlapping technology").  Two device buffers ping-pong.
    int64_t piece = n;
    if (n >= 4 * 2048) piece = round_up((n + 3) / 4, kTS);
    if (bk->hx_cap < n) {
        CU_TRY(cudaStreamSynchronize(bk->hstream));
        cudaFree(bk->hx); bk->hx = nullptr; bk->hx_cap = 0;
        CU_TRY(cudaMalloc((void**)&bk->hx, (size_t)n * sizeof(float)));
        bk->hx_cap = n;
    }
    const int64_t need = bk->T * piece * 2;
    if (bk->hsnr_cap < need) {
        CU_TRY(cudaStreamSynchronize(bk->hstream));
        CU_TRY(cudaStreamSynchronize(bk->cstream));
        for (int i = 0; i < 2; ++i) {
            cudaFree(bk->hsnr[i]); bk->hsnr[i] = nullptr;
        }
        bk->hsnr_cap = 0;
        for (int i = 0; i < 2; ++i) CU_TRY(cudaMalloc((void**)&bk->hsnr[i], (size_t)need * sizeof(float)));
        bk->hsnr_cap = need;
    }
    CU_TRY(cudaMemcpyAsync(bk->hx, x_host, (size_t)n * sizeof(float), cudaMemcpyHostToDevice, bk->hstream));
    int j = 0;
    for (int64_t off = 0; off < n; off += piece, ++j) {
        const int64_t len = std::min(piece, n - off);
        const int b = (int)((bk->host_piece + j) & 1);
        if (bk->free_pending[b]) CU_TRY(cudaStreamWaitEvent(bk->hstream, bk->ev_free[b], 0));   // the last copy out of this buffer is done
        int rc = spiir_filter(bk, bk->hx + off, len, bk->hsnr[b], len, bk->hstream);
        if (rc) return rc;
        CU_TRY(cudaEventRecord(bk->ev_done[b], bk->hstream));
        CU_TRY(cudaStreamWaitEvent(bk->cstream, bk->ev_done[b], 0));
        CU_TRY(cudaMemcpy2DAsync(snr_host + 2 * off, (size_t)ld * 8, bk->hsnr[b], (size_t)len * 8, (size_t)len * 8,
                                 (size_t)bk->T, cudaMemcpyDeviceToHost, bk->cstream));
        CU_TRY(cudaEventRecord(bk->ev_free[b], bk->cstream));
        bk->free_pending[b] = true;
    }
    bk->host_piece += j;
    return SPIIR_OK;
}

int spiir_bank_host_sync(spiir_bank* bk)
{
    if (!bk) return fail(SPIIR_EINVAL, "null bank");
    if (!bk->hstream) return SPIIR_OK;
    DeviceGuard dg(bk->device);
    CU_TRY(dg.err);
    CU_TRY(cudaStreamSynchronize(bk->hstream));
    CU_TRY(cudaStreamSynchronize(bk->cstream));
    bk->free_pending[0] = bk->free_pending[1] = false;
    return SPIIR_OK;
}

int spiir_filter_host(spiir_bank* bk, const float* x_host, int64_t n, float* snr_host, int64_t ld)
{
    int rc = spiir_filter_host_async(bk, x_host, n, snr_host, ld);
    if (rc) return rc;
    return n > 0 ? spiir_bank_host_sync(bk) : SPIIR_OK;
}

int spiir_bank_reset(spiir_bank* bk, void* stream)
{
    if (!bk) return fail(SPIIR_EINVAL, "null bank");
    cudaStream_t st = (cudaStream_t)stream;
    DeviceGuard dg(bk->device);
    CU_TRY(dg.err);
    if (bk->free_pending[0] || bk->free_pending[1]) {      // chunks of the asynchronous host entry may still be in flight
        int rc = spiir_bank_host_sync(bk);
        if (rc) return rc;
    }
    {
        int rc = order_after_previous(bk, st);
        if (rc) return rc;
    }
    CU_TRY(cudaMemsetAsync(bk->y, 0, (size_t)std::max<int64_t>(bk->n_slots, 1) * 2 * sizeof(float), st));
    bk->pos = round_up(bk->D, 4);
    CU_TRY(cudaMemsetAsync(bk->tape[bk->cur], 0, (size_t)(bk->pos + 8) * sizeof(float), st));
    bk->poisoned = false;
    return SPIIR_OK;
}

int64_t spiir_bank_num_templates(const spiir_bank* bk) { return bk ? bk->T : -1; }
int64_t spiir_bank_num_filters(const spiir_bank* bk) { return bk ? bk->K : -1; }
int64_t spiir_bank_max_delay(const spiir_bank* bk) { return bk ? bk->D : -1; }
int32_t spiir_bank_last_path(const spiir_bank* bk) { return bk ? bk->last_path : -1; }

int spiir_bank_get_state(spiir_bank* bk, float* y_dev, float* hist_dev, void* stream)
{
    if (!bk) return fail(SPIIR_EINVAL, "null bank");
    cudaStream_t st = (cudaStream_t)stream;
    DeviceGuard dg(bk->device);
    CU_TRY(dg.err);
    {
        int rc = order_after_previous(bk, st);      // also behind chunks of the host-buffer entry that are still in flight
        if (rc) return rc;
    }
    if (y_dev) {
        const int threads = 256;
        spiir_permute_state_kernel<<<(unsigned)((bk->K + threads - 1) / threads), threads, 0, st>>>(
            bk->y, y_dev, bk->slot_of_filter, bk->K, 0);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        CU_TRY(cudaGetLastError());
    }
    if (hist_dev && bk->D > 0)
        CU_TRY(cudaMemcpyAsync(hist_dev, bk->tape[bk->cur] + bk->pos - bk->D, (size_t)bk->D * sizeof(float),
                               cudaMemcpyDeviceToDevice, st));
    return SPIIR_OK;
}

int spiir_bank_set_state(spiir_bank* bk, const float* y_dev, const float* hist_dev, void* stream)
{
    if (!bk) return fail(SPIIR_EINVAL, "null bank");
    cudaStream_t st = (cudaStream_t)stream;
    DeviceGuard dg(bk->device);
    CU_TRY(dg.err);
    {
        int rc = order_after_previous(bk, st);
        if (rc) return rc;
    }
    if (y_dev) {
        const int threads = 256;
        spiir_permute_state_kernel<<<(unsigned)((bk->K + threads - 1) / threads), threads, 0, st>>>(
            y_dev, bk->y, bk->slot_of_filter, bk->K, 1);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        CU_TRY(cudaGetLastError());
    }
    if (hist_dev && bk->D > 0)
        CU_TRY(cudaMemcpyAsync(bk->tape[bk->cur] + bk->pos - bk->D, hist_dev, (size_t)bk->D * sizeof(float),
                               cudaMemcpyDeviceToDevice, st));
    return SPIIR_OK;
}

// The entry point that allocates nothing (include/spiir.h): a tiny-chunk call of a SPIIR_PATH_STREAM bank whose per-tile
// partial sums go to the file-scope device array g_static_stream_scratch instead of a cudaMalloc'ed buffer.  It never
// reaches cudaMalloc / cudaFree: sizes beyond the array, calls that would grow the tape and stream switches that would
// create an event are rejected.  The kernels are the ones spiir_filter launches for such a call.
int spiir_filter_static(spiir_bank* bk, const float* x_dev, int64_t n, float* snr_dev, int64_t ld, void* stream)
{
    if (!bk) return fail(SPIIR_EINVAL, "null bank");
    if (bk->poisoned) return fail(SPIIR_ESTATE, "bank unusable after an earlier failure");
    if (n < 0 || ld < n) return fail(SPIIR_EINVAL, "need 0 <= n <= ld");
    if (n == 0) return SPIIR_OK;
    if (!x_dev || !snr_dev) return fail(SPIIR_EINVAL, "null device pointer");
    if (bk->opt.path != SPIIR_PATH_STREAM)
        return fail(SPIIR_EINVAL, "spiir_filter_static serves banks created with SPIIR_PATH_STREAM only");
    if (n > kStreamMax)
        return fail(SPIIR_EINVAL, "spiir_filter_static: n = %lld exceeds the %d samples per call of the streaming kernels",
                    (long long)n, kStreamMax);
    if (bk->n_tiles > kStaticStreamTiles)
        return fail(SPIIR_EINVAL, "spiir_filter_static: the bank has %lld warp tiles, the static scratch holds %lld (= %lld filter "
                    "slots at %d filters per thread); use spiir_filter", (long long)bk->n_tiles, (long long)kStaticStreamTiles,
                    (long long)(kStaticStreamTiles * kWarp * bk->F), bk->F);
    cudaStream_t st = (cudaStream_t)stream;
    DeviceGuard dg(bk->device);
    CU_TRY(dg.err);
    if (bk->cap < round_up(bk->D, 4) + n + 16)
        return fail(SPIIR_EINVAL, "spiir_filter_static: the input tape would have to grow (allocation); use spiir_filter");
    if (bk->last_stream_valid && bk->last_stream != st && !bk->ev_order)
        return fail(SPIIR_EINVAL, "spiir_filter_static: the previous call of this bank used another stream and ordering the two "
                    "would create an event; keep the bank on one stream");
    int rc = order_after_previous(bk, st);
    if (rc) return rc;
    rc = ensure_tape(bk, n, st);              // room is there: at most the compaction copy (cudaMemcpyAsync)
    if (rc) return rc;
    float* tape = bk->tape[bk->cur];
    const int64_t start_al = (bk->pos - bk->D) / 4 * 4;
    const int w0 = (int)(bk->pos - start_al);
    if (!stream_applies(bk, w0, n))
        return fail(SPIIR_EINVAL, "spiir_filter_static: the history of this bank does not fit the streaming kernel's shared memory");
    unsigned long long* scratch = nullptr;
    rc = static_scratch_address(bk->device, &scratch);      // cudaGetSymbolAddress, once per device
    if (rc) return rc;
    NvtxRange range("spiir_filter_static: tiny-chunk streaming path, static scratch");
    const void* fn = select_stream_kernel(bk->F, bk->NC);
    if (!bk->stream_configured) {
        CU_TRY(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bk->smem_optin));
        bk->stream_configured = true;
    }
    const int kStreamWarps = stream_warps(bk->F);
    const size_t smem = stream_smem_bytes(bk->F, bk->NC, w0 + n, nullptr);
    if (bk->stream_occ_smem != smem) {
        int occ = 0;
        CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, kWarp * kStreamWarps, smem));
        if (occ < 1) return fail(SPIIR_ECUDA, "streaming kernel does not fit on an SM (smem %zu)", smem);
        bk->stream_occ = occ;
        bk->stream_occ_smem = smem;
    }
    StreamParams p{};
    p.coef = bk->coef; p.y = bk->y;
    p.xwin = tape + start_al; p.w0 = w0; p.n = (int32_t)n; p.n_tiles = bk->n_tiles; p.scratch = scratch;
    p.xnew = x_dev; p.append = tape + bk->pos;
    const int64_t ctas = std::min<int64_t>((bk->n_tiles + kStreamWarps - 1) / kStreamWarps, (int64_t)bk->n_sm * bk->stream_occ);
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)ctas, 1, 1);
        cfg.blockDim = dim3(kWarp * kStreamWarps, 1, 1);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        void* args[] = {(void*)&p};
        CU_TRY(cudaLaunchKernelExC(&cfg, fn, args));
    }
    {
        const int64_t total = bk->T * n;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)((total + 255) / 256), 1, 1);
        cfg.blockDim = dim3(256, 1, 1);
        cfg.dynamicSmemBytes = 0;
        cfg.stream = st;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        CU_TRY(cudaLaunchKernelEx(&cfg, spiir_stream_combine_kernel, (const u64*)scratch, (const int64_t*)bk->tile_begin,
                                  (int32_t)bk->T, (int32_t)n, snr_dev, ld, (u64*)nullptr));
    }
    g_launches.fetch_add(2, std::memory_order_relaxed);
    rc = SPIIR_OK;
    if (cudaGetLastError() != cudaSuccess) { bk->poisoned = true; return fail(SPIIR_ECUDA, "spiir_filter_static: launch failed"); }
    bk->last_path = SPIIR_PATH_STREAM;
    bk->pos += n;
    return SPIIR_OK;
}

int spiir_bank_destroy(spiir_bank* bk)
{
    if (!bk) return SPIIR_OK;
    DeviceGuard dg(bk->device);
    cudaDeviceSynchronize();
    free_bank(bk);
    return SPIIR_OK;
}

}  // extern "C"
