// Runner of the register-file probe (test infrastructure): loads patched cubins with the driver API, launches kprobe on every SM and
// prints the cycles one warp needs per loop iteration (clock64 inside the kernel) and a checksum of the results.
// usage: run_probe <warps_per_cta> <iters> cubin...
#include <cuda.h>
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <string>
#include <fstream>
#include <iterator>
#define CK(x) do { CUresult r_ = (x); if (r_ != CUDA_SUCCESS) { const char* s; cuGetErrorString(r_, &s); fprintf(stderr, "%s: %s\n", #x, s); exit(1);} } while (0)
int main(int argc, char** argv)
{
    int warps = atoi(argv[1]); int iters = atoi(argv[2]);
    CK(cuInit(0)); CUdevice dev; CK(cuDeviceGet(&dev, 0)); CUcontext ctx; CK(cuCtxCreate(&ctx, 0, dev));
    int nsm; CK(cuDeviceGetAttribute(&nsm, CU_DEVICE_ATTRIBUTE_MULTIPROCESSOR_COUNT, dev));
    CUdeviceptr in, out, cyc;
    CK(cuMemAlloc(&in, 256 * 128 * 8)); CK(cuMemAlloc(&out, (size_t)nsm * 1024 * 8)); CK(cuMemAlloc(&cyc, nsm * 8));
    std::vector<float> h(256 * 128 * 2);
    for (size_t i = 0; i < h.size(); ++i) h[i] = 0.5f + 0.001f * (float)(i % 97);
    { unsigned* u = (unsigned*)h.data(); for (int vi = 72; vi <= 73; ++vi) for (int t = 0; t < 256; ++t) { unsigned ad = (unsigned)((t * 8) & 0xfff); u[2 * (t + 256 * vi)] = ad; u[2 * (t + 256 * vi) + 1] = ad; } }
    CK(cuMemcpyHtoD(in, h.data(), h.size() * 4));
    for (int f = 3; f < argc; ++f) {
        std::ifstream s(argv[f], std::ios::binary);
        std::vector<char> img((std::istreambuf_iterator<char>(s)), std::istreambuf_iterator<char>());
        CUmodule mod; CUresult r = cuModuleLoadData(&mod, img.data());
        if (r != CUDA_SUCCESS) { const char* e; cuGetErrorString(r, &e); printf("%s LOADFAIL %s\n", argv[f], e); continue; }
        CUfunction fn; CK(cuModuleGetFunction(&fn, mod, "kprobe"));
        void* args[] = {&out, &in, &iters, &cyc};
        double best = 1e30;
        for (int rep = 0; rep < 3; ++rep) {
            CK(cuLaunchKernel(fn, nsm, 1, 1, 32 * warps, 1, 1, 32768, 0, args, 0));
            CUresult rr = cuCtxSynchronize();
            if (rr != CUDA_SUCCESS) { const char* e; cuGetErrorString(rr, &e); printf("%s RUNFAIL %s\n", argv[f], e); return 1; }
            std::vector<long long> c(nsm); CK(cuMemcpyDtoH(c.data(), cyc, nsm * 8));
            double avg = 0; for (auto v : c) avg += (double)v; avg /= nsm;
            if (avg < best) best = avg;
        }
        std::vector<unsigned long long> ho((size_t)256); CK(cuMemcpyDtoH(ho.data(), out, 256 * 8));
        unsigned long long cs = 0; for (int q = 0; q < 32 * warps && q < 256; ++q) cs = cs * 1000003ull + ho[q];
        double wps = warps / 4.0;   // warps per sub-partition
        fflush(stdout); printf("%s warps/SMSP %.2f cycles/iter %.1f checksum %016llx out0 %016llx out1 %016llx\n", argv[f], wps, best / iters, cs, ho[0], ho[1]);
        cuModuleUnload(mod); fflush(stdout);
    }
    return 0;
}
