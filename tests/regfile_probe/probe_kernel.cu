// Kernel of the register-file probe (test infrastructure): the timed loop body is NBODY independent FFMA2 placeholders that
// tests/regfile_probe/sass_patch.py overwrites in the compiled cubin; registers R4..R203 hold the 100 value pairs.
#include <cuda_runtime.h>
#include <stdint.h>
typedef unsigned long long u64;
#define NV 100
#ifndef NBODY
#define NBODY 1024
#endif
__device__ __forceinline__ u64 ffma2(u64 a, u64 b, u64 c) { u64 d; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
extern "C" __global__ void __launch_bounds__(256,1) kprobe(u64* out, const u64* in, int iters, long long* cyc)
{
    u64 v[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) v[i] = in[threadIdx.x + 256*i];
    long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < NBODY; ++i) v[i % NV] = ffma2(v[(i + 1) % NV], v[(i + 2) % NV], v[i % NV]);
    }
    long long t1 = clock64();
    u64 s = 0;
#pragma unroll
    for (int i = 0; i < NV; ++i) s ^= v[i];
    out[blockIdx.x*256+threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}
