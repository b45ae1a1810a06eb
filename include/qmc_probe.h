/*
 * qmc_probe.h -- instruction-rate microbenchmark of the B200 pipes (measurement tool, separate library
 * libqmc_probe_b200.so; not part of the product ABI of qmc.h).  DESIGN.md "Roofline".
 */
#ifndef QMC_PROBE_B200_H
#define QMC_PROBE_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Runs a dependent-chain-free kernel of ONE instruction kind on every SM of the current device (8 CTAs of 256
 * threads per SM, 8 independent chains per thread, no memory traffic) on `cuda_stream` (a cudaStream_t as void*)
 * and writes thread-level instructions per second to the HOST double *h_rate; synchronous.
 * which: 0 = fp64 DFMA, 1 = fp32 FFMA, 2 = packed FFMA2 (fma.rn.f32x2; two FMAs per instruction),
 * 3 = MUFU.RSQ (fp32 rsqrt.approx), 4 = I2FP (s32 -> f32), 5 = F2F (f64 -> f32 -> f64, both counted).
 * Returns 0, -1 (bad argument) or -3 (CUDA error, e.g. no device). */
int qmc_probe_rate(int32_t which, void *cuda_stream, double *h_rate);

#ifdef __cplusplus
}
#endif
#endif /* QMC_PROBE_B200_H */
