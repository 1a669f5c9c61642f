// Device code of the SPIIR template-bank filter (sm_100a).
//
//   y_k[n] = a1_k y_k[n-1] + b0_k x[n-d_k],   SNR_t[n] = sum_k y_k[n]      (BASELINE.json:north_star;
//   PAPER.md section 3.3: per-filter state in registers, shared input window, warp-shuffle sum)
//
// One thread owns F filters (register slots) of one template; the 32 lanes of a warp own a warp tile of
// 32*F filters; the W warps of a CTA process W warp tiles side by side over the same time range, reading
// the delayed input from one shared-memory window.  Complex numbers are kept as packed (re, im) register
// pairs and advanced with Blackwell's packed FP32 instructions (fma/mul/add .f32x2 -> FFMA2/FMUL2/FADD2):
//     t  = (b_re, b_im) * (x, x)
//     t  = (-a_im, a_im) * (y_im, y_re) + t
//     y' = (a_re, a_re) * (y_re, y_im) + t
//     S += y'
// = 4 packed instructions per filter-sample instead of 8 scalar ones (the register file, not the pipe, then bounds
// the rate: fp32_pipe_probe.cu).  Per-thread partial sums of TT = 8 consecutive samples are
// reduced across the warp through a per-warp shared-memory transpose (fixed order, no atomics -> bitwise
// reproducible), collected per super tile in shared memory, handed over between the warps of a template with
// mbarriers, summed in warp order and written with coalesced 8-byte stores.
//
// Kernels in this file:
//   spiir_filter_kernel<F, W, NC, GMEM_X, MINB, PEAK, SEG>  the blocked kernel (throughput path, both passes of the
//       time-parallel scan path, long calls of streaming banks); PEAK adds the fused trigger reduction, SEG the shared
//       warp tiles of small templates
//   spiir_stream_kernel<F, NC> + spiir_stream_combine_kernel   tiny chunks: independent warps + ordered combine
//   spiir_scan_carry_kernel                                    carry combine of the scan path (powers from double)
//   spiir_scan_fused_kernel<F, W, NC, ...>                     the scan path in one launch (two grid-wide barriers)
//   spiir_unpack_peaks_kernel, spiir_permute_state_kernel      small utilities
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#ifdef SPIIR_SCAN_TIMING
#include <cstdio>
#endif

#include "spiir_layout.hpp"

namespace spiir {

typedef unsigned long long u64;

constexpr int kTT = 8;        // samples per register tile
constexpr int kTS = 64;       // granularity of launches and segments on the host side (multiple of every super tile)
// samples per super tile (cross-warp combine + output granularity): W * super tile = 512 partial sums per buffer
__host__ __device__ constexpr int super_tile(int W) { return W <= 8 ? 64 : 32; }
constexpr int kPB = 3;        // partial-sum buffers per warp (3: a warp may run one super tile ahead of its template's slowest)

__device__ __forceinline__ u64 ffma2(u64 a, u64 b, u64 c) { u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ u64 fmul2(u64 a, u64 b) { u64 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 fadd2(u64 a, u64 b) { u64 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 pack2(float lo, float hi) { u64 d; asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi)); return d; }
__device__ __forceinline__ void unpack2(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 ld_pair(const float* p) { return *reinterpret_cast<const u64*>(p); }

struct FilterParams {
    // bank (slot order)
    const float* coef;      // [n_tiles][5 F x 32] per-tile coefficient records: ar | ai | (b_re, b_im) | delay bits
    // work list
    const int32_t* item_round0;   // [n_items + 1]
    const WarpWork* work;         // [n_rounds * W]
    int32_t n_items;
    int32_t uniform_groups;       // 1: per-template mbarriers, no CTA-wide barrier; 0: CTA-wide barriers (mixed group shapes)
    const int32_t* canon;         // [2W] (first, count) of every warp position (uniform_groups only)
    // state: per segment s (blockIdx.y) read y_in + s*y_in_stride, write y_out + s*y_out_stride
    const float* y_in;      // [2 n_slots] per segment; nullptr = zero state
    float* y_out;           // nullptr = do not store
    int64_t y_in_stride, y_out_stride;   // in floats
    int32_t store_last_only;   // 1: only the last segment stores y_out (at segment index 0)
    // input: xwin[i] = x[g0 - w0 + i] where g0 = global index of this call's first sample
    const float* xwin;      // device, 16-byte aligned
    int32_t w0;             // index of sample g0 inside xwin; max delay <= w0 (< max delay + 4): the
                            // history staged in front of every segment
    // time range of this launch
    int64_t n;              // samples in this launch
    int64_t seg_len;        // samples per segment (multiple of kTS unless single segment)
    // output
    float* snr;             // complex64 rows; nullptr with peaks == nullptr = no sums at all (carry pass)
    int64_t ld;             // row stride in complex elements
    // fused trigger reduction: peaks[t] = max over this call of (bits(|SNR_t[n]|^2) << 32 | ~n),
    // merged with atomicMax (order independent -> deterministic); nullptr = off
    u64* peaks;
    int64_t peak_off;       // index of this launch's first sample within the call
};

// One register tile: advance F filters by NV <= 8 samples, S[j] = sum over the thread's filters.
// The delayed input comes from NC shifted copies of the window (copy c holds win[i + c]), so that every
// filter reads NC consecutive samples with one aligned LDS.32 / LDS.64 / LDS.128 (xo[f] already points
// into the copy that makes its loads aligned).
// SUMS = false: states only (carry pass of the single-launch time-parallel kernel), S is left untouched.
template <int F, int NC, bool FULL, bool SUMS = true>
__device__ __forceinline__ void tile_step(const float* __restrict__ xs, const int (&xo)[F], const float (&ar)[F],
                                          const u64 (&AI)[F], const u64 (&B)[F], u64 (&Y)[F], u64 (&S)[kTT],
                                          int tb, int nv)
{
#pragma unroll
    for (int jb = 0; jb < kTT; jb += NC) {
        float xv[F][NC];
#pragma unroll
        for (int f = 0; f < F; ++f) {
            const float* px = xs + xo[f] + tb + jb;
            if (NC == 4) {
                const float4 v = *reinterpret_cast<const float4*>(px);
                xv[f][0] = v.x; xv[f][1] = v.y; xv[f][NC > 2 ? 2 : 0] = v.z; xv[f][NC > 2 ? 3 : 0] = v.w;
            } else if (NC == 2) {
                const float2 v = *reinterpret_cast<const float2*>(px);
                xv[f][0] = v.x; xv[f][NC > 1 ? 1 : 0] = v.y;
            } else {
                xv[f][0] = *px;
            }
        }
#pragma unroll
        for (int jj = 0; jj < NC; ++jj) {
            const int j = jb + jj;
            if (FULL || j < nv) {
#pragma unroll
                for (int f = 0; f < F; ++f) {
                    const float x = xv[f][jj];
                    u64 t = fmul2(B[f], pack2(x, x));
                    float yr, yi;
                    unpack2(Y[f], yr, yi);
                    t = ffma2(AI[f], pack2(yi, yr), t);
                    Y[f] = ffma2(pack2(ar[f], ar[f]), Y[f], t);
                    // S_j = ((Y_0 + Y_1) + Y_2) + ...: the first two outputs are added directly, no copy of Y_0
                    if (SUMS) {
                        if (F == 1) S[j] = Y[0];
                        else if (f == 1) S[j] = fadd2(Y[0], Y[1]);
                        else if (f > 1) S[j] = fadd2(S[j], Y[f]);
                    }
                }
            } else if (SUMS) {
                S[j] = 0ull;
            }
        }
    }
}

// Cross-lane sum of a register tile through a per-warp shared-memory transpose.  Lane l writes its 8
// partial sums as row l (4 x STS.128, rows padded to 10 u64 = 80 B so that a quarter warp hits all bank
// groups); then lane (g = l >> 3, j = l & 7) adds sample j of the 8 rows of lane group g (8 x LDS.64,
// rows visited in an order that keeps the two groups of a half warp on different banks) and two
// shuffle steps add the 4 groups.  Fixed order, no atomics.  Lanes 0..7 return the warp sum of sample
// `lane`.  Costs ~30 issue slots per tile against ~64 for a shuffle-only transposing butterfly.
constexpr int kTrRow = 10;                      // u64 per scratch row
constexpr int kTrWarp = kWarp * kTrRow;         // u64 per warp

__device__ __forceinline__ u64 warp_reduce_tile(u64 (&S)[kTT], u64* __restrict__ tr, int lane)
{
    const unsigned full = 0xffffffffu;
    ulonglong2* row = reinterpret_cast<ulonglong2*>(tr + lane * kTrRow);
#pragma unroll
    for (int c = 0; c < kTT / 2; ++c) row[c] = make_ulonglong2(S[2 * c], S[2 * c + 1]);
    __syncwarp();
    const int g = lane >> 3, j = lane & 7, b = g & 1;
    const u64* ra = tr + (g * 8 + 4 * b) * kTrRow + j;
    const u64* rb = tr + (g * 8 + 4 * (1 - b)) * kTrRow + j;
    const u64 s0 = fadd2(ra[0], ra[kTrRow]), s1 = fadd2(ra[2 * kTrRow], ra[3 * kTrRow]);
    const u64 s2 = fadd2(rb[0], rb[kTrRow]), s3 = fadd2(rb[2 * kTrRow], rb[3 * kTrRow]);
    // (rows g*8..g*8+3) + (rows g*8+4..g*8+7): IEEE addition commutes, so the half a lane read first is immaterial
    u64 P = fadd2(fadd2(s0, s1), fadd2(s2, s3));
    __syncwarp();                               // rows may be overwritten by the next tile
    P = fadd2(P, __shfl_xor_sync(full, P, 8));
    P = fadd2(P, __shfl_xor_sync(full, P, 16));
    return P;
}

// mbarrier helpers (shared::cta).  The warps of one template hand their partial sums to each other through
// "full" barriers: lane 0 of every warp arrives after the warp has written a super tile, all lanes wait before
// they read it.  Nobody ever waits for the slowest template of the CTA, only for the slowest warp of its own.
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(u64* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(u64* bar)
{
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}" ::"r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(u64* bar, unsigned parity)
{
    asm volatile(
        "{\n .reg .pred p;\n"
        "WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        " @p bra DONE_%=;\n bra WAIT_%=;\n"
        "DONE_%=:\n}" ::"r"(smem_addr(bar)), "r"(parity) : "memory");
}

// Grid-wide barrier of a kernel whose CTAs are all resident: a monotonic arrival counter in global memory, `target` = its value
// once every CTA of this launch has arrived (the host keeps the running total, so the counter is never reset).
__device__ __forceinline__ void grid_barrier(unsigned long long* counter, unsigned long long target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();                                                      // this CTA's end states are visible device-wide
        atomicAdd(counter, 1ull);
        unsigned long long v;
        do {
            asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(counter) : "memory");
        } while (v < target);
    }
    __syncthreads();
}

// Window staging (north_star subsystem (3): "stages the delayed input window into shared
// memory with TMA or cp.async.bulk"; the paper's counterpart is the shared read-only-cache window).
// One thread hands copy 0 of the window to the bulk-copy engine: cp.async.bulk global -> shared, completion counted in
// bytes on an mbarrier (SASS: UBLKCP + SYNCS); the warps meanwhile fetch their coefficients.  Source and destination
// are 16-byte aligned and the size a multiple of 16.  The NC - 1 shifted copies (copy c holds win[i + c]: a 4-byte
// misalignment no bulk copy can produce) are then made shared -> shared by all threads.
__device__ __forceinline__ void mbar_expect_tx(u64* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(void* dst_smem, const void* src_gmem, unsigned bytes, u64* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_addr(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_addr(bar))
                 : "memory");
}
// Called by ONE thread: arm the barrier for `bytes` and issue the copies (pieces of <= 32 KB).
__device__ __forceinline__ void stage_window_issue(float* dst, const float* src, unsigned bytes, u64* bar)
{
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");     // the init is visible to the copy engine
    mbar_expect_tx(bar, bytes);
    constexpr unsigned kPiece = 32768;
    for (unsigned off = 0; off < bytes; off += kPiece)
        bulk_copy_g2s(reinterpret_cast<char*>(dst) + off, reinterpret_cast<const char*>(src) + off,
                      bytes - off < kPiece ? bytes - off : kPiece, bar);
}
// All threads, once copy 0 is complete in shared memory (and visible: a __syncthreads or the copy's mbarrier): build the
// NC - 1 shifted copies from it (float4 i of copy 0 -> 4 scalar stores per further copy).
template <int NC>
__device__ __forceinline__ void make_shifted_copies(float* smem, int64_t cstride, int tid, int n_threads)
{
    if (NC == 1) return;
    const int n4 = (int)(cstride / 4);
    for (int i = tid; i < n4; i += n_threads) {
        const float4 v = reinterpret_cast<const float4*>(smem)[i];
        const float e[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int c = 1; c < NC; ++c) {
            float* dst = smem + (int64_t)c * cstride + 4 * i - c;
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (4 * i + q - c >= 0) dst[q] = e[q];
        }
    }
}

// Sum the partial rows of the warps of one template for ns samples and store them (fixed order over warps).
// The ns samples are shared out over the lanes of the template's warps.
// |z|^2 and the sample index packed so that an unsigned max picks the largest power and, among equals, the earliest
// sample (powers are non-negative floats: their bit patterns order like unsigned integers).
__device__ __forceinline__ u64 peak_key(u64 z, int64_t idx)
{
    float re, im;
    unpack2(z, re, im);
    const float m = fmaf(re, re, im * im);
    return ((u64)__float_as_uint(m) << 32) | (u64)(0xffffffffu - (unsigned)idx);
}

__device__ __forceinline__ void peak_commit(u64 best, u64* __restrict__ slot)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        const u64 o = __shfl_xor_sync(0xffffffffu, best, d);
        best = o > best ? o : best;
    }
    if ((threadIdx.x & 31) == 0 && best) atomicMax(slot, best);
}

// Sum the partial rows of the warps of one template for ns samples and store them (fixed order over warps).
// The ns samples are shared out over the lanes of the template's warps.  out == nullptr: no SNR output;
// peak != nullptr: fold |SNR|^2 of these samples (call indices idx0 ..) into the template's peak.
template <int TS, bool PEAK>
__device__ __forceinline__ void cross_warp_store(const u64* __restrict__ pb, const WarpWork& ww, int warp, int lane, int ns,
                                                 u64* __restrict__ out, bool accumulate, u64* __restrict__ peak = nullptr,
                                                 int64_t idx0 = 0)
{
    if constexpr (!PEAK) {
        for (int s = lane + kWarp * (warp - ww.first); s < ns; s += kWarp * ww.count) {
            u64 acc = pb[(size_t)ww.first * TS + s];
            for (int w = 1; w < ww.count; ++w) acc = fadd2(acc, pb[(size_t)(ww.first + w) * TS + s]);
            if (accumulate) acc = fadd2(out[s], acc);
            out[s] = acc;
        }
    } else {
        u64 best = 0ull;
        for (int s = lane + kWarp * (warp - ww.first); s < ns; s += kWarp * ww.count) {
            u64 acc = pb[(size_t)ww.first * TS + s];
            for (int w = 1; w < ww.count; ++w) acc = fadd2(acc, pb[(size_t)(ww.first + w) * TS + s]);
            if (out) {
                if (accumulate) acc = fadd2(out[s], acc);
                out[s] = acc;
            }
            if (peak) {
                const u64 k = peak_key(acc, idx0 + s);
                best = k > best ? k : best;
            }
        }
        if (peak) peak_commit(best, peak);
    }
}

// Shared ("segmented") warp tiles: the 32 lanes hold 32/w small templates of w = 4, 8 or 16 lanes each (x F register
// slots).  Same transpose as warp_reduce_tile; the lane group sums are already per template for w = 8, split in two
// for w = 4 and joined by one shuffle step for w = 16.  The sums go straight to the templates' SNR rows (8 samples
// = 64 contiguous bytes per template), no partial buffer and no cross-warp pass.  Every template is summed by the
// same tree wherever its segment sits in the tile.
// Largest key among the 8 lanes of a lane group (the 8 samples of one template segment); lane j = 0 commits it.
__device__ __forceinline__ void seg_peak_commit(u64 key, bool valid, int j, u64* __restrict__ slot)
{
    if (!valid) key = 0ull;
#pragma unroll
    for (int d = 1; d < 8; d <<= 1) {
        const u64 o = __shfl_xor_sync(0xffffffffu, key, d);
        key = o > key ? o : key;
    }
    if (j == 0 && key) atomicMax(slot, key);
}

template <bool PEAK>
__device__ __forceinline__ void seg_reduce_store(u64 (&S)[kTT], u64* __restrict__ tr, int lane, int w, int n_seg, int nv,
                                                 u64* __restrict__ out_row0, int64_t ld, u64* __restrict__ peak0 = nullptr,
                                                 int64_t idx0 = 0)
{
    ulonglong2* row = reinterpret_cast<ulonglong2*>(tr + lane * kTrRow);
#pragma unroll
    for (int c = 0; c < kTT / 2; ++c) row[c] = make_ulonglong2(S[2 * c], S[2 * c + 1]);
    __syncwarp();
    const int g = lane >> 3, j = lane & 7, b = g & 1;
    const u64* ra = tr + (g * 8 + 4 * b) * kTrRow + j;
    const u64* rb = tr + (g * 8 + 4 * (1 - b)) * kTrRow + j;
    const u64 sa = fadd2(fadd2(ra[0], ra[kTrRow]), fadd2(ra[2 * kTrRow], ra[3 * kTrRow]));   // lanes g*8 + 4b .. +3
    const u64 sb = fadd2(fadd2(rb[0], rb[kTrRow]), fadd2(rb[2 * kTrRow], rb[3 * kTrRow]));   // the other half of the group
    __syncwarp();
    if (w == 4) {
        const int seg_a = 2 * g + b, seg_b = 2 * g + 1 - b;
        const bool va = j < nv && seg_a < n_seg, vb = j < nv && seg_b < n_seg;
        if (out_row0) {
            if (va) out_row0[(int64_t)seg_a * ld + j] = sa;
            if (vb) out_row0[(int64_t)seg_b * ld + j] = sb;
        }
        if (PEAK && peak0) {
            seg_peak_commit(peak_key(sa, idx0 + j), va, j, peak0 + seg_a);
            seg_peak_commit(peak_key(sb, idx0 + j), vb, j, peak0 + seg_b);
        }
    } else {
        u64 P = fadd2(sa, sb);                                         // 8 lanes
        int seg = g;
        if (w == 16) {
            P = fadd2(P, __shfl_xor_sync(0xffffffffu, P, 8));
            seg = g >> 1;
        }
        const bool v = j < nv && seg < n_seg && (w == 8 || b == 0);
        if (out_row0 && v) out_row0[(int64_t)seg * ld + j] = P;
        if (PEAK && peak0) seg_peak_commit(peak_key(P, idx0 + j), v, j, peak0 + seg);
    }
}

// Shared memory of the filter kernel, in this order:
//   NC window copies of `cstride` floats each (absent when GMEM_X), W transpose scratches, kPB x W x kTS partial sums,
//   W x kPB mbarriers of the template hand-over + 1 mbarrier of the window's bulk copy
__host__ __device__ inline size_t filter_smem_bytes(int W, int NC, int64_t win_len, bool gmem_x, int64_t* cstride_out,
                                                     int part_buffers = kPB)
{
    // copy stride = 0 mod 32 floats: every copy starts on bank 0, as the lane dealing assumes
    const int64_t cstride = gmem_x ? 0 : ((win_len + 16 + 31) / 32 * 32);
    if (cstride_out) *cstride_out = cstride;
    return (size_t)(gmem_x ? 0 : NC * cstride) * sizeof(float) + (size_t)W * kTrWarp * sizeof(u64) +
           (size_t)part_buffers * W * super_tile(W) * sizeof(u64) + (size_t)(W * kPB + 1) * sizeof(u64);
}

// MINB = CTAs the register allocation must leave room for on one SM (tiny-chunk streaming: several small CTAs
// per SM overlap one CTA's coefficient loads with another's arithmetic).
// PEAK compiles the fused trigger reduction in (spiir_filter_peaks); the plain kernel is untouched by it.
// SEG compiles the shared-tile path for banks of small templates in.
// The body of the blocked kernel for time segment `seg`, items item0, item0 + item_stride, ...; `staged` = the window of this
// segment is already in shared memory (second pass of the fused time-parallel kernel).
// SUMS = false compiles the sums, the reduction and the output out (carry pass).
template <int F, int W, int NC, bool GMEM_X, int MINB, bool PEAK, bool SEG, bool SUMS = true>
__device__ __forceinline__ void filter_body(const FilterParams& p, const int seg, const int item0, const int item_stride,
                                            const bool staged)
{
    static_assert(!GMEM_X || NC == 1, "the global-memory window variant reads scalars");
    constexpr int kThreads = kWarp * W;
    constexpr bool kAsync = (MINB == 1);
    constexpr int TS = super_tile(W);
    extern __shared__ __align__(16) float smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t t0 = (int64_t)seg * p.seg_len;             // first sample of this segment in the launch
    const int64_t nseg = min(p.seg_len, p.n - t0);
    if (nseg <= 0) return;

    // ---- stage the input window [t0 - w0, t0 + nseg) into shared memory, NC times (copy c shifted by c): copy 0 by
    // one bulk copy (cp.async.bulk + mbarrier complete_tx), the shifted copies shared -> shared
    const int win_len = p.w0 + (int)nseg;
    int64_t cstride;
    filter_smem_bytes(W, NC, win_len, GMEM_X, &cstride);
    u64* trbuf = reinterpret_cast<u64*>(smem + (GMEM_X ? 0 : NC * cstride));   // [W][kTrWarp]
    u64* part64 = trbuf + (size_t)W * kTrWarp;                                 // [kPB][W][TS]
    u64* bars = part64 + (size_t)(kAsync ? kPB : 2) * W * TS;                  // [W][kPB], indexed by a group's first warp
    u64* stage_bar = bars + (size_t)W * kPB;
    u64* mytr = trbuf + (size_t)warp * kTrWarp;
    const float* xs = GMEM_X ? p.xwin + t0 : smem;
    const int staged_floats = (win_len + 3) / 4 * 4;                           // floats the bulk copy brings (16-byte units)
    if (!GMEM_X && !staged && tid == 0) stage_window_issue(smem, p.xwin + t0, (unsigned)staged_floats * 4u, stage_bar);   // t0, xwin: 16-byte aligned
    // per-template hand-over without any CTA-wide barrier: only where one CTA owns the SM and all rounds have one shape
    const bool sums = SUMS && (PEAK ? (p.snr || p.peaks) : (p.snr != nullptr));                              // false: carry pass, states only
    const bool async = kAsync && p.uniform_groups && sums;
    if (async && tid < W) {
        const int first = p.canon[2 * tid], count = p.canon[2 * tid + 1];
        if (first == tid && count > 0)
            for (int b = 0; b < kPB; ++b) mbar_init(bars + tid * kPB + b, count);
    }
    unsigned use = 0;                                                          // super tiles this warp has produced
    __syncthreads();                                                           // barrier inits visible to every thread
    if (!GMEM_X && !staged) {
        mbar_wait(stage_bar, 0);                                               // copy 0 has landed
        // zero what lies behind the valid samples (partial register tiles read a few floats beyond them)
        for (int k = win_len + tid; k < (int)cstride; k += kThreads) smem[k] = 0.f;
        if (NC > 1) __syncthreads();
        make_shifted_copies<NC>(smem, cstride, tid, kThreads);
        __syncthreads();
    }

    const bool last_seg = (t0 + nseg >= p.n);
    for (int item = item0; item < p.n_items; item += item_stride) {
        const int r0 = p.item_round0[item], r1 = p.item_round0[item + 1];
        for (int r = r0; r < r1; ++r) {
            WarpWork ww = p.work[r * W + warp];
            const bool active = ww.tile >= 0;
            int seg_w = 0, seg_n = 0;                  // > 0: this warp's tile is shared by seg_n templates of seg_w lanes
            if (SEG) { seg_w = (ww.first >> 8) & 0xff; seg_n = ww.first >> 16; ww.first &= 0xff; }
            float ar[F];
            u64 AI[F], B[F], Y[F];
            int xo[F];
#pragma unroll
            for (int f = 0; f < F; ++f) {
                if (active) {
                    const int64_t s = ((int64_t)ww.tile * F + f) * kWarp + lane;
                    const float* rec = p.coef + (int64_t)ww.tile * (5 * F * kWarp) + f * kWarp + lane;
                    ar[f] = rec[0];
                    { const float a_im = rec[F * kWarp]; AI[f] = pack2(-a_im, a_im); }
                    B[f] = ld_pair(rec + 2 * F * kWarp + f * kWarp + lane);
                    Y[f] = p.y_in ? ld_pair(p.y_in + (int64_t)seg * p.y_in_stride + 2 * s) : 0ull;
                    const int p0 = p.w0 - __float_as_int(rec[4 * F * kWarp]);   // window index of this filter's first input
                    const int c = p0 & (NC - 1);               // the copy in which p0 is aligned
                    xo[f] = (int)(c * cstride) + p0 - c;
                } else {
                    ar[f] = 0.f; AI[f] = 0ull; B[f] = 0ull; Y[f] = 0ull; xo[f] = 0;
                }
            }
            const bool accumulate = (r > r0);
            u64* const out_row = (!PEAK || p.snr) ? reinterpret_cast<u64*>(p.snr) + (int64_t)ww.row * p.ld + t0 : nullptr;
            // multi-round templates: only the last round sees the complete sums
            u64* const peak = (PEAK && p.peaks && active && r == r1 - 1) ? p.peaks + ww.row : nullptr;
            const int64_t idx_row = p.peak_off + t0;
            if (async) {
                if (active) {
                    int prev_ns = 0;
                    int64_t prev_st = 0;
                    unsigned prev_use = 0;
                    u64* mybars = bars + ww.first * kPB;
                    for (int64_t st = 0; st < nseg; st += TS) {
                        const int ns = (int)min((int64_t)TS, nseg - st);
                        const unsigned i = use++;
                        u64* mypart = part64 + ((size_t)(i % kPB) * W + warp) * TS;
#pragma unroll 1
                        for (int tt = 0; tt < ns; tt += kTT) {
                            u64 S[kTT];
                            const int nv = ns - tt;
                            if (nv >= kTT) tile_step<F, NC, true>(xs, xo, ar, AI, B, Y, S, (int)st + tt, kTT);
                            else tile_step<F, NC, false>(xs, xo, ar, AI, B, Y, S, (int)st + tt, nv);
                            const u64 P = warp_reduce_tile(S, mytr, lane);
                            if (lane < kTT) mypart[tt + lane] = P;
                        }
                        // finish the previous super tile before announcing this one (keeps 3 buffers sufficient)
                        if (prev_ns) {
                            mbar_wait(mybars + prev_use % kPB, (prev_use / kPB) & 1);
                            cross_warp_store<TS, PEAK>(part64 + (size_t)(prev_use % kPB) * W * TS, ww, warp, lane, prev_ns, (!PEAK || out_row) ? out_row + prev_st : nullptr, accumulate, peak, idx_row + prev_st);
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(mybars + i % kPB);
                        prev_ns = ns; prev_st = st; prev_use = i;
                    }
                    if (prev_ns) {
                        mbar_wait(mybars + prev_use % kPB, (prev_use / kPB) & 1);
                        cross_warp_store<TS, PEAK>(part64 + (size_t)(prev_use % kPB) * W * TS, ww, warp, lane, prev_ns, (!PEAK || out_row) ? out_row + prev_st : nullptr, accumulate, peak, idx_row + prev_st);
                    }
                }
            } else {
                // a round made of shared tiles only has nothing to hand over between warps: no CTA-wide barrier in its loop
                const bool round_bar = !SEG || __syncthreads_or(active && seg_w == 0);
                int buf = 0;
                for (int64_t st = 0; st < nseg; st += TS, buf ^= 1) {
                    const int ns = (int)min((int64_t)TS, nseg - st);
                    if (active) {
                        u64* mypart = part64 + ((size_t)buf * W + warp) * TS;
#pragma unroll 1
                        for (int tt = 0; tt < ns; tt += kTT) {
                            u64 S[kTT];
                            const int nv = ns - tt;
                            if (nv >= kTT) tile_step<F, NC, true, SUMS>(xs, xo, ar, AI, B, Y, S, (int)st + tt, kTT);
                            else tile_step<F, NC, false, SUMS>(xs, xo, ar, AI, B, Y, S, (int)st + tt, nv);
                            if (sums) {
                                if (SEG && seg_w) {
                                    seg_reduce_store<PEAK>(S, mytr, lane, seg_w, seg_n, nv, (!PEAK || out_row) ? out_row + st + tt : nullptr, p.ld,
                                                           peak, idx_row + st + tt);
                                } else {
                                    const u64 P = warp_reduce_tile(S, mytr, lane);
                                    if (lane < kTT) mypart[tt + lane] = P;
                                }
                            }
                        }
                    }
                    if (sums && round_bar) {
                        __syncthreads();
                        if (active && !(SEG && seg_w))
                            cross_warp_store<TS, PEAK>(part64 + (size_t)buf * W * TS, ww, warp, lane, ns, (!PEAK || out_row) ? out_row + st : nullptr, accumulate, peak, idx_row + st);
                    }
                }
            }
            if (active && p.y_out && (!p.store_last_only || last_seg)) {
                float* yo = p.y_out + (p.store_last_only ? 0 : (int64_t)seg * p.y_out_stride);
#pragma unroll
                for (int f = 0; f < F; ++f) {
                    const int64_t s = ((int64_t)ww.tile * F + f) * kWarp + lane;
                    *reinterpret_cast<u64*>(yo + 2 * s) = Y[f];
                }
            }
            if (sums && !async) __syncthreads();      // part rows are rewritten in the next round (kept for shared tiles too:
                                                      // once per round, and the next round's __syncthreads_or needs all warps)
        }
    }
}

// Main kernel.  grid.x strides over items, grid.y = time segments (1 for the sequential path).
template <int F, int W, int NC, bool GMEM_X, int MINB = 1, bool PEAK = false, bool SEG = false>
__global__ void __launch_bounds__(kWarp * W, MINB) spiir_filter_kernel(const FilterParams p)
{
    filter_body<F, W, NC, GMEM_X, MINB, PEAK, SEG>(p, (int)blockIdx.y, (int)blockIdx.x, (int)gridDim.x, false);
}

// ---- time-parallel path in ONE launch (north_star subsystem (4)).  Grid = items x segments,
// every CTA resident (cooperative launch).  Phase 1: the segment from zero state, end states z_seg to global memory
// (no sums); grid-wide barrier; the grid's threads then derive the true start states of all segments, one filter
// slot per thread, c_{q+1} = a1^L c_q + z_q from c_0 = carried state (a1^L from double, SURVEY.md section 8(c) finding F2), with
// the same arithmetic and rounding as spiir_scan_carry_kernel; a second barrier; every CTA runs its segment again with sums and
// output.  The window stays
// in shared memory between the phases.
// c <- A c + z in FP32 (A = a1^L rounded from double); one fixed order of fused multiply-adds, shared by the standalone carry
// kernel and the single-launch kernel so that both forms of the path produce the same bits
__device__ __forceinline__ void scan_carry_step(float Ar, float Ai, float zr, float zi, float& cr, float& ci)
{
    const float nr = fmaf(Ar, cr, fmaf(-Ai, ci, zr));
    const float ni = fmaf(Ar, ci, fmaf(Ai, cr, zi));
    cr = nr; ci = ni;
}

struct ScanFusedParams {
    FilterParams pass1, pass2;
    float* cbuf;                     // [n_seg][2 n_slots] start states
    const float* z;                  // = pass1.y_out
    const float* y;                  // carried state (slot order)
    int64_t n_slots;
    int32_t n_seg;
    const float* xnew;               // the call's chunk in the caller's buffer (not on the tape yet) ...
    float* append;                   // ... and where it goes on the tape: every CTA appends its own segment
    unsigned long long* barrier;     // monotonic arrival counter
    unsigned long long target;       // its value when every CTA of this launch has arrived at the first barrier
};

// -DSPIIR_SCAN_TIMING: the first and the last segment's CTA of item 0 print the duration of every phase (%globaltimer, ns)
// for the first launches of a bank -- the launch-gap / phase instrument of profiles/r02_scan_phases.md (no nsys in the image).
#ifdef SPIIR_SCAN_TIMING
#define SPIIR_STAMP(k) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(stamp[k]))
#else
#define SPIIR_STAMP(k)
#endif

template <int F, int W, int NC, bool GMEM_X, bool PEAK, bool SEG>
__global__ void __launch_bounds__(kWarp * W, 1) spiir_scan_fused_kernel(const ScanFusedParams sp)
{
#ifdef SPIIR_SCAN_TIMING
    unsigned long long stamp[6];
#endif
    SPIIR_STAMP(0);
    const int seg = blockIdx.y, item = blockIdx.x;
    const bool has_pass1 = seg + 1 < sp.n_seg;                    // the last segment's zero-state end values are never used
    {
        // The window [t0 - w0, t0 + nseg) of this segment: history from the bank's tape, the call's own samples straight from
        // the caller's buffer (the kernel appends them to the tape itself, so a call is this one launch and nothing else).
        const FilterParams& p = sp.pass2;
        const int64_t t0 = (int64_t)seg * p.seg_len;
        const int nseg = (int)min(p.seg_len, p.n - t0);
        const int win_len = p.w0 + nseg;
        int64_t cstride;
        filter_smem_bytes(W, NC, win_len, GMEM_X, &cstride);
        extern __shared__ __align__(16) float smem[];
        const int64_t first = t0 - p.w0;                         // call-relative sample index of window element 0
        for (int k = threadIdx.x; k < (int)cstride; k += kWarp * W) {
            const int64_t i = first + k;
            smem[k] = k < win_len ? (i < 0 ? p.xwin[t0 + k] : sp.xnew[i]) : 0.f;
        }
        if (item == 0)
            for (int k = threadIdx.x; k < nseg; k += kWarp * W) sp.append[t0 + k] = sp.xnew[t0 + k];
        __syncthreads();
        make_shifted_copies<NC>(smem, cstride, threadIdx.x, kWarp * W);
        __syncthreads();
    }
    SPIIR_STAMP(1);
    if (has_pass1) filter_body<F, W, NC, GMEM_X, 1, PEAK, SEG, false>(sp.pass1, seg, item, sp.pass1.n_items, true);
    SPIIR_STAMP(2);
    grid_barrier(sp.barrier, sp.target);
    SPIIR_STAMP(3);
    {
        // true start states of every segment, one slot per thread over the whole grid (the chain over the segments of a
        // slot is sequential, the slots are independent): c_0 = carried state, c_{q+1} = a1^L c_q + z_q in double
        const FilterParams& p = sp.pass1;
        const int64_t L = p.seg_len;
        const int64_t n_threads = (int64_t)gridDim.x * gridDim.y * blockDim.x;
        const int64_t per_tile = (int64_t)F * kWarp;
        for (int64_t s = ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * blockDim.x + threadIdx.x; s < sp.n_slots; s += n_threads) {
            const float* rec = p.coef + (s / per_tile) * 5 * per_tile + s % per_tile;
            // the chain over the segments is dependent, the loads of the end states are not: two batches of kB in flight,
            // the first one requested before the power is worked out
            constexpr int kB = 8;
            float2 za[kB], zb[kB];
            const float* zs = sp.z + 2 * s;
            const int64_t zstride = 2 * sp.n_slots;
            const int n_z = sp.n_seg - 1;
            auto fetch = [&](float2 (&zz)[kB], int q0) {
#pragma unroll
                for (int i = 0; i < kB; ++i)
                    zz[i] = __ldcg(reinterpret_cast<const float2*>(zs + (int64_t)min(q0 + i, n_z - 1) * zstride));
            };
            if (n_z > 0) fetch(za, 0);
            float cr = sp.y[2 * s], ci = sp.y[2 * s + 1];
            double pr = 1.0, pi = 0.0, br = (double)rec[0], bi = (double)rec[per_tile];
            for (int64_t e = L; e > 0; e >>= 1) {                              // a1^L by binary powering in double
                if (e & 1) { const double tr = pr * br - pi * bi, ti = pr * bi + pi * br; pr = tr; pi = ti; }
                const double tr = br * br - bi * bi, ti = 2.0 * br * bi; br = tr; bi = ti;
            }
            const float Ar = (float)pr, Ai = (float)pi;                        // a1^L: from double, rounded once
            *reinterpret_cast<float2*>(sp.cbuf + 2 * s) = make_float2(cr, ci);
            auto chain = [&](const float2 (&zz)[kB], int q0) {
#pragma unroll
                for (int i = 0; i < kB; ++i) {
                    if (q0 + i < n_z) {
                        scan_carry_step(Ar, Ai, zz[i].x, zz[i].y, cr, ci);
                        *reinterpret_cast<float2*>(sp.cbuf + (int64_t)(q0 + i + 1) * zstride + 2 * s) = make_float2(cr, ci);
                    }
                }
            };
            for (int q0 = 0; q0 < n_z; q0 += 2 * kB) {
                if (q0 + kB < n_z) fetch(zb, q0 + kB);
                chain(za, q0);
                if (q0 + 2 * kB < n_z) fetch(za, q0 + 2 * kB);
                if (q0 + kB < n_z) chain(zb, q0 + kB);
            }
        }
    }
    grid_barrier(sp.barrier, sp.target + (unsigned long long)gridDim.x * gridDim.y);
    SPIIR_STAMP(4);
    filter_body<F, W, NC, GMEM_X, 1, PEAK, SEG>(sp.pass2, seg, item, sp.pass2.n_items, true);
    SPIIR_STAMP(5);
#ifdef SPIIR_SCAN_TIMING
    if (threadIdx.x == 0 && item == 0 && (seg == 0 || seg == sp.n_seg - 1) && sp.target < 40ull * gridDim.x * gridDim.y)
        printf("scan launch, segment %d of %d: window %llu  carry pass %llu  barrier %llu  carries + barrier %llu  output pass %llu ns\n",
               seg, sp.n_seg, stamp[1] - stamp[0], stamp[2] - stamp[1], stamp[3] - stamp[2], stamp[4] - stamp[3], stamp[5] - stamp[4]);
#endif
}

// ---- tiny-chunk streaming (SPIIR_PATH_STREAM, n <= kStreamMax samples per call).
// Every call streams the whole bank through the SMs once, so the path is bound by HBM and by per-round
// overhead, not by arithmetic.  Warps are independent: a warp takes warp tiles round-robin, loads their
// coefficients and state, advances the n samples, reduces over its 32 lanes and writes the tile's partial sums
// to a scratch row; no barrier, no shared partial buffers.  spiir_stream_combine_kernel then adds the tiles of
// every template in tile order (fixed order -> bitwise reproducible).
constexpr int kStreamMax = 64;          // samples per call served by the streaming kernels
// warps per CTA (one CTA per SM; the warps never synchronise, a big CTA only shares the staged window): what the
// register file allows
__host__ __device__ constexpr int stream_warps(int F) { return F <= 4 ? 24 : 16; }

struct StreamParams {
    const float* coef;            // per-tile coefficient records (see FilterParams)
    float* y;                     // state, updated in place
    const float* xwin; int32_t w0; int32_t n;   // history: xwin[0 .. w0) (16-byte aligned); the n new samples follow it ...
    const float* xnew;            // ... unless xnew != nullptr: then they are read from the caller's chunk xnew[0 .. n)
    float* append;                // where CTA 0 stores the chunk for later calls (the bank's tape); nullptr: already there
    int64_t n_tiles;
    u64* scratch;                 // [n_tiles][kStreamMax] partial sums of every warp tile
    // combine phase of the same launch (barrier == nullptr: a separate spiir_stream_combine_kernel follows instead)
    const int64_t* tile_begin;    // [n_templates + 1] first warp tile of every template
    int32_t n_templates;
    float* snr; int64_t ld;       // complex64 rows
    u64* peaks;                   // fused trigger reduction or nullptr
    unsigned long long* barrier;  // grid-wide barrier between the two phases
    unsigned long long target;
};

// SNR[t][j] = sum over the warp tiles of template t, in tile order, of scratch[tile][j] (fixed order -> bitwise reproducible,
// independent of a template's position in the bank).
__device__ __forceinline__ void stream_combine_one(const u64* __restrict__ scratch, const int64_t* __restrict__ tile_begin, int64_t i,
                                                   int32_t n, float* __restrict__ snr, int64_t ld, u64* __restrict__ peaks, bool cg)
{
    const int32_t t = (int32_t)(i / n), j = (int32_t)(i % n);
    const int64_t t0 = tile_begin[t], t1 = tile_begin[t + 1];
    u64 acc = cg ? __ldcg(scratch + t0 * kStreamMax + j) : scratch[t0 * kStreamMax + j];
    // loads 16 tiles ahead of the (ordered) additions: the chain of adds is short, the chain of L2 latencies is not
    for (int64_t tile = t0 + 1; tile < t1; tile += 16) {
        u64 v[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const u64* src = scratch + (tile + q) * kStreamMax + j;
            v[q] = (tile + q < t1) ? (cg ? __ldcg(src) : *src) : 0ull;
        }
#pragma unroll
        for (int q = 0; q < 16; ++q)
            if (tile + q < t1) acc = fadd2(acc, v[q]);
    }
    if (snr) reinterpret_cast<u64*>(snr)[(int64_t)t * ld + j] = acc;
    if (peaks) atomicMax(peaks + t, peak_key(acc, j));
}

__host__ __device__ inline size_t stream_smem_bytes(int F, int NC, int64_t win_len, int64_t* cstride_out)
{
    const int64_t cstride = (win_len + 16 + 31) / 32 * 32;
    if (cstride_out) *cstride_out = cstride;
    // window copies, one transpose scratch per warp, the mbarrier of the window's bulk copy
    return (size_t)(NC * cstride) * sizeof(float) + (size_t)stream_warps(F) * kTrWarp * sizeof(u64) + 2 * sizeof(u64);
}

// The 7F cache lines of a warp tile's coefficients and state, one or two per lane, requested into L1.
template <int F>
__device__ __forceinline__ void stream_prefetch_tile(const StreamParams& p, int64_t tile, int lane)
{
    const float* rec = p.coef + tile * (5 * F * kWarp);    // 5F consecutive lines of coefficients
    const float* st = p.y + 2 * tile * F * kWarp;          // 2F consecutive lines of state
#pragma unroll
    for (int q = 0; q < (7 * F + kWarp - 1) / kWarp; ++q) {
        const int idx = lane + q * kWarp;
        const float* line = idx < 5 * F ? rec + idx * kWarp : st + (idx - 5 * F) * kWarp;
        if (idx < 7 * F) asm volatile("prefetch.global.L1 [%0];" ::"l"(line));
    }
}

template <int F, int NC>
__global__ void __launch_bounds__(kWarp * stream_warps(F), 1) spiir_stream_kernel(const StreamParams p)
{
    constexpr int kStreamWarps = stream_warps(F);
    constexpr int kThreads = kWarp * kStreamWarps;
    extern __shared__ __align__(16) float smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int win_len = p.w0 + p.n;
    int64_t cstride;
    stream_smem_bytes(F, NC, win_len, &cstride);
    u64* const stage_bar = reinterpret_cast<u64*>(smem + NC * cstride) + (size_t)kStreamWarps * kTrWarp;   // completion of the window's bulk copy
    // the first tile's coefficients travel while the window is staged
    if ((int64_t)blockIdx.x * kStreamWarps + warp < p.n_tiles) stream_prefetch_tile<F>(p, (int64_t)blockIdx.x * kStreamWarps + warp, lane);
    // Launched with programmatic dependent launch: the grid is set up and the first coefficients are requested while the
    // previous kernel in the stream (normally the previous call) is still running.  Everything read from here on may
    // have been written by that kernel or by the caller's own kernels: wait for them.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    {
        // copy 0 of the window: the part that is whole 16-byte units of the tape by one bulk copy (cp.async.bulk +
        // mbarrier complete_tx); the few floats behind it (and the chunk itself while it is
        // still in the caller's buffer) by ordinary loads; then the shifted copies shared -> shared
        const int bulk_floats = p.xnew ? p.w0 / 4 * 4 : (win_len + 3) / 4 * 4;
        if (tid == 0 && bulk_floats > 0) stage_window_issue(smem, p.xwin, (unsigned)bulk_floats * 4u, stage_bar);
        for (int k = bulk_floats + tid; k < (int)cstride; k += kThreads)
            smem[k] = k < p.w0 ? p.xwin[k] : (k < win_len ? p.xnew[k - p.w0] : 0.f);
        __syncthreads();                               // the barrier's init and the stores above are visible
        if (bulk_floats > 0) mbar_wait(stage_bar, 0);
        if (bulk_floats > win_len) {                   // the copy brought up to 3 floats from beyond the window
            if (win_len + tid < bulk_floats) smem[win_len + tid] = 0.f;
            __syncthreads();
        }
        make_shifted_copies<NC>(smem, cstride, tid, kThreads);
    }
    const float* xs = smem;
    u64* mytr = reinterpret_cast<u64*>(smem + NC * cstride) + (size_t)warp * kTrWarp;
    __syncthreads();
    // the chunk joins the history for later calls (every CTA has staged its window: nobody reads the tape beyond w0)
    if (p.append && p.xnew && blockIdx.x == 0)
        for (int i = tid; i < p.n; i += kThreads) p.append[i] = p.xnew[i];

    const int64_t n_warps = (int64_t)gridDim.x * kStreamWarps;
    for (int64_t tile = (int64_t)blockIdx.x * kStreamWarps + warp; tile < p.n_tiles; tile += n_warps) {
        float ar[F];
        u64 AI[F], B[F], Y[F];
        int xo[F];
        const int64_t s0 = tile * F * kWarp + lane;
#pragma unroll
        for (int f = 0; f < F; ++f) {
            const int64_t s = s0 + f * kWarp;
            const float* rec = p.coef + tile * (5 * F * kWarp) + f * kWarp + lane;
            ar[f] = rec[0];
            { const float a_im = rec[F * kWarp]; AI[f] = pack2(-a_im, a_im); }
            B[f] = ld_pair(rec + 2 * F * kWarp + f * kWarp + lane);
            Y[f] = ld_pair(p.y + 2 * s);
            const int p0 = p.w0 - __float_as_int(rec[4 * F * kWarp]);
            const int c = p0 & (NC - 1);
            xo[f] = (int)(c * cstride) + p0 - c;
        }
        // Ask for the next tile of this warp now (its 7F cache lines, one or two per lane), so that its loads hit L1
        // after this tile's arithmetic instead of waiting for HBM: the warps never have nothing in flight.
        if (tile + n_warps < p.n_tiles) stream_prefetch_tile<F>(p, tile + n_warps, lane);
        u64* row = p.scratch + tile * kStreamMax;
#pragma unroll 1
        for (int tt = 0; tt < p.n; tt += kTT) {
            u64 S[kTT];
            const int nv = p.n - tt;
            if (nv >= kTT) tile_step<F, NC, true>(xs, xo, ar, AI, B, Y, S, tt, kTT);
            else tile_step<F, NC, false>(xs, xo, ar, AI, B, Y, S, tt, nv);
            const u64 P = warp_reduce_tile(S, mytr, lane);
            if (lane < kTT) row[tt + lane] = P;
        }
#pragma unroll
        for (int f = 0; f < F; ++f) *reinterpret_cast<u64*>(p.y + 2 * (s0 + f * kWarp)) = Y[f];
    }
    if (p.barrier) {
        // second phase of the same launch: every CTA is resident (grid <= SMs x occupancy), so the grid can meet at a
        // barrier; the partial rows are then summed per (template, sample) by all threads of the grid
        asm volatile("griddepcontrol.launch_dependents;");     // the next call's kernel may be set up (it waits itself)
        grid_barrier(p.barrier, p.target);
        const int64_t total = (int64_t)p.n_templates * p.n;
        for (int64_t i = (int64_t)blockIdx.x * kThreads + tid; i < total; i += (int64_t)gridDim.x * kThreads)
            stream_combine_one(p.scratch, p.tile_begin, i, p.n, p.snr, p.ld, p.peaks, true);
    }
}

// The combine as a kernel of its own (one thread per (t, j)): used when the streaming kernel's grid cannot meet at a barrier.
__global__ void spiir_stream_combine_kernel(const u64* __restrict__ scratch, const int64_t* __restrict__ tile_begin,
                                            int32_t n_templates, int32_t n, float* __restrict__ snr, int64_t ld,
                                            u64* __restrict__ peaks)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (int64_t)n_templates * n) return;
    asm volatile("griddepcontrol.wait;" ::: "memory");     // launched early (PDL): the streaming kernel's rows from here on
    asm volatile("griddepcontrol.launch_dependents;");     // the next call's streaming kernel may be set up (it waits itself)
    stream_combine_one(scratch, tile_begin, i, n, snr, ld, peaks, false);
}

// ---- time-parallel scan: carry combine.  For every slot, given the carried state c_0 = y and the
// zero-state end values z_p of segments p = 0..P-2 (all of length seg_len), produce the true start
// states c_{p+1} = a1^seg_len * c_p + z_p.  The power is evaluated in double from the float32 a1 by binary powering and
// rounded once to float32 (SURVEY.md section 8(c) finding F2: 2.7e-6 of max|SNR| with multipliers from double against
// 3.3e-5 with FP32 repeated squaring); the combine itself is the same FP32 complex multiply-add a filter step is.
__global__ void spiir_scan_carry_kernel(const float* __restrict__ coef, int32_t F,
                                        const float* __restrict__ y, const float* __restrict__ z,
                                        float* __restrict__ c, int64_t n_slots, int32_t n_seg, int64_t seg_len)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_slots) return;
    const int64_t per_tile = (int64_t)F * kWarp;
    const float* rec = coef + (s / per_tile) * 5 * per_tile + s % per_tile;
    double pr = 1.0, pi = 0.0, br = (double)rec[0], bi = (double)rec[per_tile];
    for (int64_t e = seg_len; e > 0; e >>= 1) {
        if (e & 1) { const double tr = pr * br - pi * bi, ti = pr * bi + pi * br; pr = tr; pi = ti; }
        const double tr = br * br - bi * bi, ti = 2.0 * br * bi; br = tr; bi = ti;
    }
    const float Ar = (float)pr, Ai = (float)pi;
    float cr = y[2 * s], ci = y[2 * s + 1];
    // c[0] is the carried state itself (segment 0 starts from it)
    c[2 * s] = cr;
    c[2 * s + 1] = ci;
    // the carries are a dependent chain, the loads of z are not: fetch them kB at a time ahead of the chain
    constexpr int kB = 8;
    for (int32_t q0 = 0; q0 + 1 < n_seg; q0 += kB) {
        float2 zz[kB];
#pragma unroll
        for (int i = 0; i < kB; ++i) {
            const int32_t q = min(q0 + i, n_seg - 2);
            zz[i] = *reinterpret_cast<const float2*>(z + (int64_t)q * 2 * n_slots + 2 * s);
        }
#pragma unroll
        for (int i = 0; i < kB; ++i) {
            const int32_t q = q0 + i;
            if (q + 1 < n_seg) {
                scan_carry_step(Ar, Ai, zz[i].x, zz[i].y, cr, ci);
                *reinterpret_cast<float2*>(c + (int64_t)(q + 1) * 2 * n_slots + 2 * s) = make_float2(cr, ci);
            }
        }
    }
}

// ---- small utilities
__global__ void spiir_unpack_peaks_kernel(const u64* __restrict__ peaks, float* __restrict__ power, int32_t* __restrict__ arg,
                                          int32_t n_templates)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_templates) return;
    const u64 k = peaks[t];
    if (power) power[t] = __uint_as_float((unsigned)(k >> 32));
    if (arg) arg[t] = (int32_t)(0xffffffffu - (unsigned)(k & 0xffffffffu));
}

__global__ void spiir_permute_state_kernel(const float* __restrict__ src, float* __restrict__ dst,
                                           const int64_t* __restrict__ slot_of_filter, int64_t K, int to_slots)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= K) return;
    const int64_t s = slot_of_filter[k];
    if (to_slots) { dst[2 * s] = src[2 * k]; dst[2 * s + 1] = src[2 * k + 1]; }
    else { dst[2 * k] = src[2 * s]; dst[2 * k + 1] = src[2 * s + 1]; }
}

}  // namespace spiir
