// qmc_f32c.cuh -- building blocks of the FP32C mode (R20): fixed-point coordinate codec and the packed
// fp32 (f32x2) arithmetic of Blackwell (FFMA2 / FMUL2 / FADD2: two fp32 lanes per 64-bit register pair and
// ONE issue slot; the FMA pipe still spends two cycles on it -- measured, profiles/r01_pipes.md).
//
// A coordinate x in [0, L) is stored in global memory as the fp32 number s = 1 + x/L in [1,2): every such
// fp32 is a multiple of 2^-23.  On chip it is held as the 32-bit fixed-point number k << 9 (k = the 23-bit
// mantissa of s), so that a - b in WRAPPING 32-bit integer arithmetic is the signed minimum image
// times 2^32, exactly; one I2FP turns it into fp32.
#pragma once
#include <cstdint>

namespace qmc {

__device__ __forceinline__ int32_t enc_coord(float s) { return (int32_t)((__float_as_uint(s) & 0x7FFFFFu) << 9); }
__device__ __forceinline__ float dec_coord(int32_t k) { return __uint_as_float(0x3F800000u | ((uint32_t)k >> 9)); }
__device__ __forceinline__ int32_t wadd(int32_t a, int32_t b) { return (int32_t)((uint32_t)a + (uint32_t)b); }
// a - b, forced onto the integer-add unit: written as the three-input sum a - b + zero, which the
// multiply-add unit cannot take over (ptxas otherwise turns half of the subtractions of a pair loop into
// IMAD.IADD, which runs at half rate on the pipe the FFMA2s need).  `zero` must be an opaque register
// holding 0 (opaque_zero()).
__device__ __forceinline__ int32_t wsub3(int32_t a, int32_t b, int32_t zero)
{
    int32_t d;
    asm("{.reg .b32 t; sub.s32 t, %1, %2; add.s32 %0, t, %3;}" : "=r"(d) : "r"(a), "r"(b), "r"(zero));
    return d;
}
__device__ __forceinline__ int32_t wsub(int32_t a, int32_t b) { return (int32_t)((uint32_t)a - (uint32_t)b); }
// 0 that neither nvcc nor ptxas can prove to be 0, and that has to live in a register: read back from a
// shared-memory word the caller has zeroed (and synchronised) before.
__device__ __forceinline__ int32_t opaque_zero(const volatile int32_t *zeroed_shared_word) { return *zeroed_shared_word; }

typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ f32x2 pk1(float a) { return pk2(a, a); }
__device__ __forceinline__ void upk2(f32x2 r, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(r)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ float hsum2(f32x2 a) { float x, y; upk2(a, x, y); return x + y; }

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

}  // namespace qmc
