// qmc_probe.cu -- instruction-rate microbenchmarks of the B200 pipes the pair loops lean on.
// MEASUREMENT TOOL, not part of the product library: built as its own libqmc_probe_b200.so (include/qmc_probe.h),
// used by bench.py to report the live denominators beside the derived ALU peak.
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

#include "../../include/qmc_probe.h"

namespace qmc {

// ------------------------------------------------------------------------------------------
// FP pipe peak: 8 independent FMA chains per thread, 2048 threads per SM, no memory traffic.
// ------------------------------------------------------------------------------------------
template <typename Real>
__global__ void __launch_bounds__(256) fma_peak_kernel(Real *sink, int iters, Real a, Real b)
{
    Real v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = (Real)(threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 8; ++rep)
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = fma(v[k], a, b);
    }
    Real s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += v[k];
    if (s == (Real)123456789) sink[0] = s;      // never true; keeps the chains alive
}

}  // namespace qmc

// Instruction-rate probes behind qmc_probe_rate kinds 2..5: 8 independent chains per thread of one
// instruction kind (inline PTX, so that the kind in SASS is the one named), no memory traffic.
namespace qmc {
template <int KIND>
__global__ void __launch_bounds__(256) rate_probe_kernel(float *sink, int iters, float a, float b)
{
    float v[8];
    unsigned long long p[8], pa, pb;
    double d[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        v[k] = a + (float)(threadIdx.x + k);
        asm("mov.b64 %0, {%1, %2};" : "=l"(p[k]) : "f"(v[k]), "f"(v[k] + 0.5f));
        d[k] = (double)v[k];
    }
    asm("mov.b64 %0, {%1, %1};" : "=l"(pa) : "f"(a));
    asm("mov.b64 %0, {%1, %1};" : "=l"(pb) : "f"(b));
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 8; ++rep)
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (KIND == 2) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[k]) : "l"(pa), "l"(pb));
                if (KIND == 3) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(v[k]));
                if (KIND == 4) asm volatile("{.reg .s32 t; mov.b32 t, %0; cvt.rn.f32.s32 %0, t;}" : "+f"(v[k]));
                if (KIND == 5) asm volatile("{.reg .f32 t; cvt.rn.f32.f64 t, %0; cvt.f64.f32 %0, t;}" : "+d"(d[k]));
            }
    }
    float s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        float lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p[k]));
        s += v[k] + lo + hi + (float)d[k];
    }
    if (s == 123456789.0f) sink[0] = s;         // never true; keeps the chains alive
}
}  // namespace qmc

using namespace qmc;

extern "C" int qmc_probe_rate(int32_t which, void *cuda_stream, double *h_fma_per_s)
{
    if (!h_fma_per_s || which < 0 || which > 5) return -1;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        return -3;
    }
    void *sink = nullptr;
    if (cudaMalloc(&sink, 64) != cudaSuccess) return -3;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = which == 1 ? 8000 : (which == 0 || which == 2 || which == 4 ? 4000 : 1000);
    const int grid = sms * 8, block = 256;
    float best_ms = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        switch (which) {
        case 0: fma_peak_kernel<double><<<grid, block, 0, st>>>((double *)sink, iters, 0.999999, 1e-7); break;
        case 1: fma_peak_kernel<float><<<grid, block, 0, st>>>((float *)sink, iters, 0.999999f, 1e-7f); break;
        case 2: rate_probe_kernel<2><<<grid, block, 0, st>>>((float *)sink, iters, 0.999999f, 1e-7f); break;
        case 3: rate_probe_kernel<3><<<grid, block, 0, st>>>((float *)sink, iters, 0.999999f, 1e-7f); break;
        case 4: rate_probe_kernel<4><<<grid, block, 0, st>>>((float *)sink, iters, 0.999999f, 1e-7f); break;
        default: rate_probe_kernel<5><<<grid, block, 0, st>>>((float *)sink, iters, 0.999999f, 1e-7f); break;
        }
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    cudaError_t e = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    if (e != cudaSuccess) { fprintf(stderr, "qmc_probe_rate: %s\n", cudaGetErrorString(e)); return -3; }
    const double per_iter = which == 5 ? 128.0 : 64.0;          // kind 5 issues two conversions per chain step
    *h_fma_per_s = (double)grid * block * (double)iters * per_iter / (best_ms * 1e-3);
    return 0;
}
