// fp32_pipe_probe -- what FP32 rate can the SPIIR filter body reach on this GPU?
//
// The roofline of the filter kernel is the FP32 FMA pipe.  Its nominal peak
// (SMs x 128 lanes x 2 flop x clock) assumes one FMA per lane per clock, but a packed FFMA2 whose three
// operands are all per-lane register pairs needs more register-file read bandwidth than the register
// file delivers in the two cycles the pipe needs.  This probe times, on every SM, loops of
//   (a) single packed instructions by operand mix, and
//   (b) the filter body  t = B*x; t = AI*swap(Y) + t; Y = ar*Y + t; S += Y  (4 packed instructions),
// with all operands in per-lane registers as in the kernel, and prints cycles per packed instruction per
// SM sub-partition (2.0 = pipe peak) and the resulting ceiling for the kernel in % of nominal peak.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fp32_pipe_probe fp32_pipe_probe.cu
// It shares no code with the library; it only measures the machine.
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
typedef unsigned long long u64;
__device__ __forceinline__ u64 ffma2(u64 a, u64 b, u64 c) { u64 d; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ u64 fmul2(u64 a, u64 b) { u64 d; asm volatile("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 fadd2(u64 a, u64 b) { u64 d; asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 pack2(float lo, float hi) { u64 d; asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi)); return d; }
__device__ __forceinline__ void unpack2(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }

constexpr int C = 8;      // independent chains (filters) per thread, as in the kernel
constexpr int TT = 4;     // samples per unrolled step

enum { FFMA2_3PAIRS, FFMA2_3PAIRS_SWAP, FFMA2_SCALAR_2PAIRS, FMUL2_PAIR_SCALAR, FADD2_2PAIRS, FFMA_SCALAR, BODY, BODY_AI_SCALAR };

template <int MODE>
__global__ void __launch_bounds__(512) probe(float* out, const float* in, int iters)
{
    const int lane = threadIdx.x & 31;
    float ar[C], ai[C], yr[C], yi[C];
    u64 AI[C], B[C], Y[C], S[TT];
#pragma unroll
    for (int c = 0; c < C; ++c) {
        ar[c] = in[c + lane] * 0.5f;
        ai[c] = in[c + 9 + lane] * 0.5f;
        AI[c] = pack2(-in[c + 8 + lane] * 0.5f, in[c + 9 + lane] * 0.5f);
        B[c] = pack2(in[c + 16 + lane], in[c + 24 + lane]);
        Y[c] = pack2(in[c + 32 + lane], in[c + 64 + lane]);
        yr[c] = in[c + 40 + lane]; yi[c] = in[c + 50 + lane];
    }
#pragma unroll
    for (int j = 0; j < TT; ++j) S[j] = pack2(in[lane + j], in[lane + j + 1]);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < TT; ++j) {
#pragma unroll
            for (int c = 0; c < C; ++c) {
                if (MODE == FFMA2_3PAIRS) Y[c] = ffma2(AI[c], Y[c], B[c]);
                if (MODE == FFMA2_3PAIRS_SWAP) { float a, b; unpack2(Y[c], a, b); Y[c] = ffma2(AI[c], pack2(b, a), B[c]); }
                if (MODE == FFMA2_SCALAR_2PAIRS) Y[c] = ffma2(pack2(ar[c], ar[c]), Y[c], B[c]);
                if (MODE == FMUL2_PAIR_SCALAR) { float a, b; unpack2(Y[(c + 1) % C], a, b); Y[c] = fmul2(B[c], pack2(a, a)); }
                if (MODE == FADD2_2PAIRS) Y[c] = fadd2(Y[c], B[c]);
                if (MODE == FFMA_SCALAR) { yr[c] = fmaf(ar[c], yr[c], yi[(c + 1) % C]); yi[c] = fmaf(ai[c], yi[c], yr[(c + 3) % C]); }
                if (MODE == BODY || MODE == BODY_AI_SCALAR) {
                    float xa, xb; unpack2(Y[(c + 3) % C], xa, xb);        // stands in for x[n-d]: a per-lane scalar register
                    u64 t = fmul2(B[c], pack2(xa, xa));
                    float a, b; unpack2(Y[c], a, b);
                    t = ffma2(MODE == BODY ? AI[c] : pack2(-ai[c], ai[c]), pack2(b, a), t);
                    Y[c] = ffma2(pack2(ar[c], ar[c]), Y[c], t);
                    S[j] = fadd2(S[j], Y[c]);
                }
            }
        }
    }
    float acc = 0.f;
#pragma unroll
    for (int c = 0; c < C; ++c) { float a, b; unpack2(Y[c], a, b); acc += a + b + yr[c] + yi[c]; }
#pragma unroll
    for (int j = 0; j < TT; ++j) { float a, b; unpack2(S[j], a, b); acc += a + b; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

static int g_nsm = 0;
static double g_clock_hz = 0;

template <int MODE>
double run(const char* name, int threads, double instr_per_step, float* out, const float* in)
{
    const int iters = 4000;
    probe<MODE><<<g_nsm, threads>>>(out, in, 100);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0);
    probe<MODE><<<g_nsm, threads>>>(out, in, iters);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    const double warp_instr = (double)g_nsm * (threads / 32) * C * TT * iters * instr_per_step;
    const double cyc = ms * 1e-3 * g_clock_hz * g_nsm * 4;     // SM sub-partition cycles
    const double cpi = cyc / warp_instr;
    printf("| %-44s | %4d | %8.3f | %5.2f |\n", name, threads, ms, cpi);
    return cpi;
}

int main(int argc, char** argv)
{
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, 0) != cudaSuccess) { fprintf(stderr, "no CUDA device\n"); return 1; }
    g_nsm = prop.multiProcessorCount;
    int khz = 0; cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
    g_clock_hz = (argc > 1 ? atof(argv[1]) * 1e6 : khz * 1e3);
    printf("device %s, %d SMs, clock used for cycle counts %.0f MHz\n\n", prop.name, g_nsm, g_clock_hz / 1e6);
    float *out, *in;
    cudaMalloc(&out, (size_t)g_nsm * 1024 * 4); cudaMalloc(&in, 4096 * 4);
    float h[4096]; for (int i = 0; i < 4096; ++i) h[i] = 0.001f * (i % 97) + 0.1f;
    cudaMemcpy(in, h, sizeof(h), cudaMemcpyHostToDevice);
    printf("| loop of | threads/SM | ms | cycles per instruction per sub-partition |\n|---|---|---|---|\n");
    double body = 0;
    for (int thr : {256, 512}) {
        run<FFMA_SCALAR>("FFMA   d = a*b + c, 3 scalar registers", thr, 2, out, in);
        run<FFMA2_3PAIRS>("FFMA2  3 register pairs", thr, 1, out, in);
        run<FFMA2_3PAIRS_SWAP>("FFMA2  3 register pairs, one swapped (LO_HI)", thr, 1, out, in);
        run<FFMA2_SCALAR_2PAIRS>("FFMA2  broadcast scalar + 2 pairs", thr, 1, out, in);
        run<FMUL2_PAIR_SCALAR>("FMUL2  pair * broadcast scalar", thr, 1, out, in);
        run<FADD2_2PAIRS>("FADD2  2 pairs", thr, 1, out, in);
        body = run<BODY>("filter body, 4 packed instructions", thr, 4, out, in);
        run<BODY_AI_SCALAR>("filter body, (-ai, ai) built from one scalar", thr, 4, out, in);
    }
    // 12 algorithmic flops per filter-sample in 4 packed instructions; the nominal peak is 2 flop per lane-cycle
    printf("\nfilter body: %.2f cycles per filter-sample per sub-partition (pipe floor 8.00)\n", 4 * body);
    printf("ceiling of the kernel by 12-flop accounting: %.1f %% of nominal FP32 FMA peak (pipe floor: 75.0 %%)\n", 100.0 * 12.0 / (2.0 * 4 * body));
    return 0;
}
