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
// = 4 issue slots per filter-sample instead of 8 scalar ones.  Per-thread partial sums of TT = 8
// consecutive samples are reduced across the warp with a transposing shuffle butterfly (fixed order, no
// atomics -> bitwise reproducible), staged in shared memory per 64-sample super tile, summed across the
// warps of a template and written with coalesced 8-byte stores.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "spiir_layout.hpp"

namespace spiir {

typedef unsigned long long u64;

constexpr int kTT = 8;        // samples per register tile
constexpr int kTS = 64;       // samples per super tile (cross-warp combine + output granularity)

__device__ __forceinline__ u64 ffma2(u64 a, u64 b, u64 c) { u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ u64 fmul2(u64 a, u64 b) { u64 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 fadd2(u64 a, u64 b) { u64 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 pack2(float lo, float hi) { u64 d; asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi)); return d; }
__device__ __forceinline__ void unpack2(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 ld_pair(const float* p) { return *reinterpret_cast<const u64*>(p); }

struct FilterParams {
    // bank (slot order)
    const float* ar;        // [n_slots]
    const float* ai2;       // [2 n_slots] (-a_im, a_im)
    const float* b;         // [2 n_slots] (b_re, b_im)
    const int32_t* dly;     // [n_slots]
    // work list
    const int32_t* item_round0;   // [n_items + 1]
    const WarpWork* work;         // [n_rounds * W]
    int32_t n_items;
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
    float* snr;             // complex64 rows, nullptr = no output (carry pass)
    int64_t ld;             // row stride in complex elements
};

// One register tile: advance F filters by NV <= 8 samples, S[j] = sum over the thread's filters.
template <int F, bool FULL>
__device__ __forceinline__ void tile_step(const float* __restrict__ xs, const int (&xo)[F], const float (&ar)[F],
                                          const u64 (&AI)[F], const u64 (&B)[F], u64 (&Y)[F], u64 (&S)[kTT],
                                          int tb, int nv)
{
#pragma unroll
    for (int j = 0; j < kTT; ++j) {
        if (FULL || j < nv) {
#pragma unroll
            for (int f = 0; f < F; ++f) {
                const float x = xs[xo[f] + tb + j];
                u64 t = fmul2(B[f], pack2(x, x));
                float yr, yi;
                unpack2(Y[f], yr, yi);
                t = ffma2(AI[f], pack2(yi, yr), t);
                Y[f] = ffma2(pack2(ar[f], ar[f]), Y[f], t);
                S[j] = (f == 0) ? Y[f] : fadd2(S[j], Y[f]);
            }
        } else {
            S[j] = 0ull;
        }
    }
}

// Transposing butterfly: on return every lane holds the warp-wide sum of sample bitrev3(lane & 7).
__device__ __forceinline__ u64 warp_reduce_tile(u64 (&S)[kTT], int lane)
{
    const unsigned full = 0xffffffffu;
    u64 R[4], Q[2];
    const bool b0 = lane & 1, b1 = lane & 2, b2 = lane & 4;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const u64 send = b0 ? S[i] : S[i + 4];
        const u64 keep = b0 ? S[i + 4] : S[i];
        R[i] = fadd2(keep, __shfl_xor_sync(full, send, 1));
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const u64 send = b1 ? R[i] : R[i + 2];
        const u64 keep = b1 ? R[i + 2] : R[i];
        Q[i] = fadd2(keep, __shfl_xor_sync(full, send, 2));
    }
    const u64 send = b2 ? Q[0] : Q[1];
    const u64 keep = b2 ? Q[1] : Q[0];
    u64 P = fadd2(keep, __shfl_xor_sync(full, send, 4));
    P = fadd2(P, __shfl_xor_sync(full, P, 8));
    P = fadd2(P, __shfl_xor_sync(full, P, 16));
    return P;
}

// Main kernel.  grid.x strides over items, grid.y = time segments (1 for the sequential path).
// Dynamic shared memory: [xwin window floats][2 * W * kTS complex partial sums].
template <int F, int W, bool GMEM_X>
__global__ void __launch_bounds__(kWarp * W) spiir_filter_kernel(const FilterParams p)
{
    constexpr int kThreads = kWarp * W;
    extern __shared__ __align__(16) float smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int seg = blockIdx.y;
    const int64_t t0 = (int64_t)seg * p.seg_len;             // first sample of this segment in the launch
    const int64_t nseg = min(p.seg_len, p.n - t0);
    if (nseg <= 0) return;

    // ---- stage the input window [t0 - w0, t0 + nseg) into shared memory
    const int64_t win0 = t0;                                  // index in xwin of the window start (mult of 4)
    const int win_len = p.w0 + (int)nseg;
    const int win_pad = (win_len + 3) & ~3;
    const float* xs;
    float* part;
    if (GMEM_X) {
        xs = p.xwin + win0;
        part = smem;
    } else {
        const float4* src = reinterpret_cast<const float4*>(p.xwin + win0);
        float4* dst = reinterpret_cast<float4*>(smem);
        for (int i = tid; i < win_pad / 4; i += kThreads) dst[i] = src[i];
        xs = smem;
        part = smem + win_pad;
    }
    u64* part64 = reinterpret_cast<u64*>(part);               // [2][W][kTS]
    __syncthreads();

    const bool last_seg = (t0 + nseg >= p.n);
    for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
        const int r0 = p.item_round0[item], r1 = p.item_round0[item + 1];
        for (int r = r0; r < r1; ++r) {
            const WarpWork ww = p.work[r * W + warp];
            const bool active = ww.tile >= 0;
            float ar[F];
            u64 AI[F], B[F], Y[F];
            int xo[F];
#pragma unroll
            for (int f = 0; f < F; ++f) {
                if (active) {
                    const int64_t s = ((int64_t)ww.tile * F + f) * kWarp + lane;
                    ar[f] = p.ar[s];
                    AI[f] = ld_pair(p.ai2 + 2 * s);
                    B[f] = ld_pair(p.b + 2 * s);
                    Y[f] = p.y_in ? ld_pair(p.y_in + (int64_t)seg * p.y_in_stride + 2 * s) : 0ull;
                    xo[f] = p.w0 - p.dly[s];
                } else {
                    ar[f] = 0.f; AI[f] = 0ull; B[f] = 0ull; Y[f] = 0ull; xo[f] = 0;
                }
            }
            const bool accumulate = (r > r0);
            int buf = 0;
            for (int64_t st = 0; st < nseg; st += kTS, buf ^= 1) {
                const int ns = (int)min((int64_t)kTS, nseg - st);
                if (active) {
                    u64* mypart = part64 + ((size_t)buf * W + warp) * kTS;
#pragma unroll 1
                    for (int tt = 0; tt < ns; tt += kTT) {
                        u64 S[kTT];
                        const int nv = ns - tt;
                        if (nv >= kTT) tile_step<F, true>(xs, xo, ar, AI, B, Y, S, (int)st + tt, kTT);
                        else tile_step<F, false>(xs, xo, ar, AI, B, Y, S, (int)st + tt, nv);
                        if (p.snr) {
                            const u64 P = warp_reduce_tile(S, lane);
                            if (lane < kTT) {
                                const int sidx = ((lane & 1) << 2) | (lane & 2) | ((lane & 4) >> 2);
                                mypart[tt + sidx] = P;
                            }
                        }
                    }
                }
                if (p.snr) {
                    __syncthreads();
                    if (active) {
                        // warps of one template share its ns samples; fixed summation order over warps
                        const u64* pb = part64 + (size_t)buf * W * kTS;
                        for (int s = lane + kWarp * (warp - ww.first); s < ns; s += kWarp * ww.count) {
                            u64 acc = pb[(size_t)ww.first * kTS + s];
                            for (int w = 1; w < ww.count; ++w) acc = fadd2(acc, pb[(size_t)(ww.first + w) * kTS + s]);
                            u64* out = reinterpret_cast<u64*>(p.snr) + (int64_t)ww.row * p.ld + t0 + st + s;
                            if (accumulate) acc = fadd2(*out, acc);
                            *out = acc;
                        }
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
            if (p.snr) __syncthreads();   // part buffers are reused by the next round
        }
    }
}

// ---- time-parallel scan: carry combine.  For every slot, given the carried state c_0 = y and the
// zero-state end values z_p of segments p = 0..P-2 (all of length seg_len), produce the true start
// states c_{p+1} = a1^seg_len * c_p + z_p.  Powers and the combine are evaluated in double from the
// float32 a1 (SURVEY.md section 8(c) finding F2), then rounded once to float32.
__global__ void spiir_scan_carry_kernel(const float* __restrict__ ar, const float* __restrict__ ai2,
                                        const float* __restrict__ y, const float* __restrict__ z,
                                        float* __restrict__ c, int64_t n_slots, int32_t n_seg, int64_t seg_len)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_slots) return;
    // a^L by binary exponentiation in double
    double pr = 1.0, pi = 0.0, br = (double)ar[s], bi = (double)ai2[2 * s + 1];
    for (int64_t e = seg_len; e > 0; e >>= 1) {
        if (e & 1) { const double tr = pr * br - pi * bi, ti = pr * bi + pi * br; pr = tr; pi = ti; }
        const double tr = br * br - bi * bi, ti = 2.0 * br * bi; br = tr; bi = ti;
    }
    double cr = (double)y[2 * s], ci = (double)y[2 * s + 1];
    // c[0] is the carried state itself (segment 0 starts from it)
    c[2 * s] = (float)cr;
    c[2 * s + 1] = (float)ci;
    for (int32_t q = 0; q + 1 < n_seg; ++q) {
        const double zr = (double)z[(int64_t)q * 2 * n_slots + 2 * s], zi = (double)z[(int64_t)q * 2 * n_slots + 2 * s + 1];
        const double nr = pr * cr - pi * ci + zr, ni = pr * ci + pi * cr + zi;
        // continue from the float32-rounded carry: that is the state segment q+1 really starts from
        cr = (double)(float)nr;
        ci = (double)(float)ni;
        c[(int64_t)(q + 1) * 2 * n_slots + 2 * s] = (float)nr;
        c[(int64_t)(q + 1) * 2 * n_slots + 2 * s + 1] = (float)ni;
    }
}

// ---- small utilities
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
