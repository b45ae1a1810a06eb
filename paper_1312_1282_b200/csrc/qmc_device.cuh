// qmc_device.cuh -- device-side building blocks of the He-4 VMC hot path (sm_100a).
//
// Independent implementation of the definitions in DESIGN.md ("Definitions", "Randomness");
// shares nothing with oracle/.  PAPER.md = arXiv:1312.1282.
//
//   pair correlation   u(r) = f(r) + f(L-r) - 2 f(L/2),  f(r) = -1/2 (b/r)^5     Eq.(8)/(9), R1
//   written here as    u = c1 * (y^5 + z^5) + c0,  y = 1/r, z = 1/(L-r),
//                      c1 = -b^5/2,  c0 = b^5 / h^5  (= -2 f(h)),  h = L/2
//   minimum image      per component m = h - | h - |a-b| |   ( = min(|d|, L-|d|) for |d| <= L,
//                      and squares to the right value for L < |d| < 3L/2 )                 l.325, R5
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace qmc {

// ---------------------------------------------------------------------------------------------
// Per-parameter-point constants (device copy, doubles; kernels narrow them for FP32C).
// ---------------------------------------------------------------------------------------------
// Lengths are expressed in the mode's COORDINATE UNIT: 1 Angstrom in FP64; the box edge in FP32C,
// where a coordinate is stored as s = 1 + x/L in [1,2) -- every fp32 in [1,2) is a multiple of 2^-23,
// so coordinate differences and the minimum-image fold are EXACT in fp32.
struct AzizDev {            // HFD-B(HE), l.131, R3; inv_rm, rm2, Drm in coordinate units
    double eps, inv_rm, rm2, A, alpha, beta, c6, c8, c10, D, Drm;
    double f32_scale;       // FP32C: the potential is summed in units of this number of kelvin (qmc_energy_f32_pair.cuh)
};

struct GroupDev {
    double L, h, h2;        // box edge, cutoff L/2, cutoff squared            [coordinate units]
    double c1, c0;          // u = c1*(y^5+z^5) + c0 = c1*t,  t = y^5 + z^5 - sh  [coordinate units]
    double sh;              // 2/h^5: t(h) = 0 (exactly 64 in FP32C box units)
    double b5;              // b^5 (for u', u'')                                 [coordinate units]
    double unit, inv_unit;  // Angstrom per coordinate unit and its inverse (1 in FP64, L and 1/L in FP32C)
    double origin;          // stored coordinate of x = 0 (0 in FP64, 1 in FP32C)
    double L_A;             // box edge in Angstrom
    double step;            // proposal half-width of the current qmc_sweep call [Angstrom]
    double a_lat;           // FCC lattice constant L/k (R13)                    [Angstrom]
    int32_t k_lat;          // cells per edge
    int32_t pad;
    AzizDev az;
};

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11): 10 rounds of
//   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),  key += (W0,W1).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k)
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}

// Exact maps of a 32-bit word to (-1,1) and (0,1) (R7, R8): (2x+1)/2^32 - 1 and (2x+1)/2^33.
__device__ __forceinline__ double word_to_pm1(uint32_t x)
{
    return __dadd_rn(__dmul_rn(__dadd_rn(__uint2double_rn(x), 0.5), 4.656612873077392578125e-10), -1.0);
}
__device__ __forceinline__ double word_to_unit(uint32_t x)
{
    return __dmul_rn(__dadd_rn(__uint2double_rn(x), 0.5), 2.3283064365386962890625e-10);
}

// ---------------------------------------------------------------------------------------------
// Proposal 1 (PAPER.md l.144 random particle, l.325 Gaussian displacement by Box-Muller): standard normals
// from 32-bit words with IEEE +, -, *, /, sqrt only, every operation rounded once in the order DESIGN.md
// "Proposal 1" fixes, so that the CPU oracle's independent implementation agrees bit for bit.
//   ln u, u = (2w+1) 2^-33:  n = 2w+1 = m 2^e, m in [1,2); m > sqrt2 -> m/2, e+1; s = (m-1)/(m+1);
//                            ln m = 2 s sum_{k<=10} s^2k/(2k+1) (Horner), ln u = ln m + (e-33) ln2
//   cos/sin 2 pi (w+1/2) 2^-32: quadrant w>>30, f from the low 30 bits; f > 1/2: use 1-f and swap;
//                            x = f pi/2, Taylor in x^2 to x^15 (sin) and x^16 (cos) by Horner
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double ln_unit33(uint32_t w)
{
    const unsigned long long n = 2ull * (unsigned long long)w + 1ull;
    int e = 63 - __clzll((long long)n);
    double m = __ddiv_rn(__ull2double_rn(n), __ull2double_rn(1ull << e));
    if (m > 1.4142135623730951) { m = __dmul_rn(0.5, m); e += 1; }
    const double s = __ddiv_rn(__dadd_rn(m, -1.0), __dadd_rn(m, 1.0));
    const double s2 = __dmul_rn(s, s);
    double P = 1.0 / 21.0;
#pragma unroll
    for (int k = 9; k >= 0; --k) P = __dadd_rn(__dmul_rn(P, s2), 1.0 / (double)(2 * k + 1));
    const double lnm = __dmul_rn(__dmul_rn(2.0, s), P);
    return __dadd_rn(lnm, __dmul_rn((double)(e - 33), 0.6931471805599453));
}
__device__ __forceinline__ void cos_sin_2pi32(uint32_t w, double &c, double &s)
{
    const uint32_t q = w >> 30;
    double f = __dmul_rn(__dadd_rn(__uint2double_rn(w & 0x3FFFFFFFu), 0.5), 1.0 / 1073741824.0);
    const bool swap = f > 0.5;
    if (swap) f = __dadd_rn(1.0, -f);
    const double x = __dmul_rn(f, 1.5707963267948966);
    const double x2 = __dmul_rn(x, x);
    double ps = -1.0 / 1307674368000.0;
    ps = __dadd_rn(__dmul_rn(ps, x2), 1.0 / 6227020800.0);
    ps = __dadd_rn(__dmul_rn(ps, x2), -1.0 / 39916800.0);
    ps = __dadd_rn(__dmul_rn(ps, x2), 1.0 / 362880.0);
    ps = __dadd_rn(__dmul_rn(ps, x2), -1.0 / 5040.0);
    ps = __dadd_rn(__dmul_rn(ps, x2), 1.0 / 120.0);
    ps = __dadd_rn(__dmul_rn(ps, x2), -1.0 / 6.0);
    ps = __dadd_rn(__dmul_rn(ps, x2), 1.0);
    const double sn = __dmul_rn(x, ps);
    double pc = 1.0 / 20922789888000.0;
    pc = __dadd_rn(__dmul_rn(pc, x2), -1.0 / 87178291200.0);
    pc = __dadd_rn(__dmul_rn(pc, x2), 1.0 / 479001600.0);
    pc = __dadd_rn(__dmul_rn(pc, x2), -1.0 / 3628800.0);
    pc = __dadd_rn(__dmul_rn(pc, x2), 1.0 / 40320.0);
    pc = __dadd_rn(__dmul_rn(pc, x2), -1.0 / 720.0);
    pc = __dadd_rn(__dmul_rn(pc, x2), 1.0 / 24.0);
    pc = __dadd_rn(__dmul_rn(pc, x2), -0.5);
    pc = __dadd_rn(__dmul_rn(pc, x2), 1.0);
    const double c1 = swap ? sn : pc, s1 = swap ? pc : sn;
    c = (q == 0) ? c1 : (q == 1) ? -s1 : (q == 2) ? -c1 : s1;
    s = (q == 0) ? s1 : (q == 1) ? c1 : (q == 2) ? -s1 : -c1;
}
__device__ __forceinline__ void normal_pair(uint32_t w1, uint32_t w2, double &z0, double &z1)
{
    const double R = __dsqrt_rn(__dmul_rn(-2.0, ln_unit33(w1)));
    double c, s;
    cos_sin_2pi32(w2, c, s);
    z0 = __dmul_rn(R, c);
    z1 = __dmul_rn(R, s);
}

// ---------------------------------------------------------------------------------------------
// Fast reciprocal square root / reciprocal in fp64: hardware seed (MUFU.RSQ64H / MUFU.RCP64H,
// relative error <= ~2^-20) followed by ONE third-order correction, error ~ seed^3 < 2^-58.
// Arguments here are always normal, positive and far from the exponent limits.
// ---------------------------------------------------------------------------------------------
// 1/sqrt(x), x > 0.  The hardware seed looks at the upper 32 bits of x only: relative error e up to ~2^-20; third
// order, error ~e^3 (below rounding).  (A second-order step, one instruction less, leaves 4e-13 on y and 2e-12 on
// y^5: measured 6.8 % faster fp64 sweeps, but E = V + T to 3e-11 only and the margins of overlapping trials beyond
// the 1e-12 the trajectory tests hold them to -- not taken.)
__device__ __forceinline__ double rsqrt_pos(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = x * y;
    const double e = fma(-t, y, 1.0);          // e = 1 - x y^2
    const double p = fma(e, 0.375, 0.5);       // 1/2 + 3/8 e
    const double q = y * e;
    return fma(q, p, y);                       // y (1 + e/2 + 3 e^2/8)
}
// a < b for a >= 0 or NaN, b > 0: the same answer as the fp64 comparison (the bit patterns of non-negative doubles
// order like integers, NaN -- the poison of the sweep kernel -- lies above every number), taken on the integer
// pipe, which idles in fp64 mode, instead of a DSETP on the fp64 pipe that bounds it
__device__ __forceinline__ bool less_pos(double a, double b)
{
    return (unsigned long long)__double_as_longlong(a) < (unsigned long long)__double_as_longlong(b);      // unsigned: a NaN of either sign is large
}
// 1/x for the z = 1/(L - r) terms: second order, relative error e^2 < 1e-12 on terms that make up 1e-3 of the pair
// sums and vanish against y^5 where a trial overlaps a neighbour
__device__ __forceinline__ double rcp_pos(double x)
{
    double z;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(z) : "d"(x));
    const double e = fma(-x, z, 1.0);          // e = 1 - x z, |e| up to ~2^-20
    return fma(z, e, z);                       // z (1 + e): relative error e^2 < 1e-12 on a term that is 1e-3 of the sums
}
__device__ __forceinline__ float rsqrt_pos(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_pos(float x)
{
    float z;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(z) : "f"(x));
    return z;
}

template <typename Real> __device__ __forceinline__ Real rabs(Real x);
template <> __device__ __forceinline__ double rabs<double>(double x) { return fabs(x); }
template <> __device__ __forceinline__ float rabs<float>(float x) { return fabsf(x); }

// Constants of one parameter point narrowed to the arithmetic type of the mode.
template <typename Real>
struct PairConst {
    Real L, h, h2, c1, c0;
    __device__ __forceinline__ void load(const GroupDev &g)
    {
        L = (Real)g.L;
        h = (Real)0.5 * L;            // exactly half of the box edge AS REPRESENTED in Real
        h2 = h * h;
        c1 = (Real)g.c1;
        c0 = (Real)g.c0;
    }
};

// ---------------------------------------------------------------------------------------------
// Warp / block sums.  The xor butterfly leaves the bitwise-identical total in every lane
// (IEEE addition commutes), so every thread can take the same decision without a broadcast.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    return v;
}

}  // namespace qmc
