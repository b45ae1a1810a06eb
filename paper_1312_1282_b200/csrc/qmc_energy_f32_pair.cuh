// qmc_energy_f32_pair.cuh -- packed fp32 pair arithmetic shared by the two FP32C local-energy kernels
// (qmc_energy_f32.cu: ordered pairs, any N; qmc_energy_f32s.cu: every unordered pair once).
// Box units (L = 1, h = 1/2); coordinates are 32-bit fixed point (qmc_f32c.cuh).
#pragma once
#include "qmc_internal.h"
#include "qmc_f32c.cuh"

namespace qmc {
namespace e32 {

// Units.  r^2 arrives as d^2 2^64 (integer differences); ONE integer instruction (VIADDMNMX: add to the exponent
// field, then min) rescales it by 2^-62 and clamps it: a4 = min(4 r^2, 1).  Everything after that is in HALF units:
// yh = rsqrt(a4) = y/2, q = a4 yh = 2r, zh = 1/(2 - q) = z/2; at the clamp yh = zh = q = 1.  The sums the kernels
// keep are therefore scaled by exact powers of two, undone in fp64 at the end:
//   pair-sum term  t/32   = yh^5 + zh^5 - 2                       (kSUnit)
//   gradient       gm/128 = yh^7 - zh^6 yh                        (kGUnit)
//   Laplacian      lt/128 = 2 yh^7 + 3 zh^7 + zh^6 yh = 6 at the clamp   (kGUnit, kLamClamp)
constexpr int    kClampBits = 0x3F800000;      // bit pattern of 1.0f = the clamped a4; inside the cutoff iff bits(a4) < this
constexpr double kSUnit = 32.0, kGUnit = 128.0, kLamClamp = 6.0;

// The four amplitudes (eps A and the three dispersion coefficients) are single fp32 numbers; their rounding errors
// (up to 6e-8 each) are systematic, and the repulsive and the dispersion sums are each several times |V|, so they showed
// as +0.5 ... 2e-6 on V.  The potential is therefore summed in units of s kelvin, with s in [1, 2) searched on the host
// (aziz_f32_scale, once per qmc_create) such that all four amplitudes divided by s round to fp32 with a relative
// error below ~5e-9; the total is multiplied by s in fp64 at the end.
inline double aziz_f32_scale(const AzizDev &a)
{
    const double r2 = a.rm2, r6 = r2 * r2 * r2;
    const double c[4] = {a.eps * a.A, a.eps * a.c6 * r6 * 64.0, a.eps * a.c8 * r6 * r2 * 256.0, a.eps * a.c10 * r6 * r2 * r2 * 1024.0};
    double best = 1.0, best_err = 1e300;
    for (int i = 0; i < 400000; ++i) {
        const double s = 1.0 + (double)i * 2.5e-6;
        double err = 0.0;
        for (int k = 0; k < 4; ++k) {
            const double v = c[k] / s;
            const double e = fabs((double)(float)v / v - 1.0);
            err = e > err ? e : err;
        }
        if (err < best_err) { best_err = err; best = s; }
    }
    return best;
}

// HFD-B(HE) constants for packed fp32 evaluation.  Every constant that multiplies into the steep
// repulsive exponential or the dispersion sum is folded (in fp64, on load) into ONE rounded coefficient
// or carried as hi + lo, so that no fp32 rounding of a CONSTANT puts a systematic relative error on
// every pair (the box-unit value of r_m is an arbitrary real number).  With R = 2r and Y = y/2 (half units):
//   rep  = eps A 2^(a1 R + a2 R^2),  a1 = -alpha log2(e) / (2 r_m),  a2 = beta log2(e) / (4 r_m^2)   (hi + lo)
//   disp = v^3 (k6 + v (k8 + v k10)),  v = Y^2,  k_n = eps c_n r_m^n 2^n
//   F    = 2^(-(sqrt(log2 e) max(2 D r_m Y - 1, 0))^2)                              (2 D r_m hi + lo)
struct AzizF32 {
    f32x2 a1h, a1l, a2h, a2l, epsA, epsAln2, nk6, nk8, nk10, Dh, Dl, nDc;
    __device__ __forceinline__ void load(const AzizDev &a)
    {
        const double log2e = 1.4426950408889634, ln2 = 0.6931471805599453, sl = 1.2011224087864498;   // sqrt(log2 e)
        auto split = [](double v, f32x2 &hi, f32x2 &lo) {
            const float h = __double2float_rn(v);
            hi = pk1(h);
            lo = pk1(__double2float_rn(v - (double)h));
        };
        split(-0.5 * a.alpha * a.inv_rm * log2e, a1h, a1l);
        split(0.25 * a.beta * a.inv_rm * a.inv_rm * log2e, a2h, a2l);
        const double is = 1.0 / a.f32_scale;                         // see aziz_f32_scale()
        const float eA = (float)(a.eps * a.A * is);
        epsA = pk1(eA);
        epsAln2 = pk1((float)((double)eA * ln2));
        const double r2 = a.rm2, r6 = r2 * r2 * r2;
        nk6 = pk1((float)(-a.eps * a.c6 * r6 * 64.0 * is));
        nk8 = pk1((float)(-a.eps * a.c8 * r6 * r2 * 256.0 * is));
        nk10 = pk1((float)(-a.eps * a.c10 * r6 * r2 * r2 * 1024.0 * is));
        split(2.0 * a.Drm * sl, Dh, Dl);
        nDc = pk1((float)(-sl));
    }
};

// Everything the pair arithmetic of two j produces (half units, see above).
struct Pair2 {
    f32x2 mx, my, mz;      // signed minimum image, 2^32 box units
    f32x2 q;               // 2r
    f32x2 y, z;            // y/2 = 1/(2r), z/2 = 1/(2(1-r))
    f32x2 y2, z2, y4, z4;
    float a, b;            // the two lanes of a4 = min(4 r^2, 1)
};

__device__ __forceinline__ float scale_clamp_r2(float a)
{
    return __int_as_float(__viaddmin_s32(__float_as_int(a), -(62 << 23), kClampBits));
}

__device__ __forceinline__ Pair2 pair_geom(int32_t xi, int32_t yi, int32_t zi, int32_t X0, int32_t X1, int32_t Y0, int32_t Y1,
                                           int32_t Z0, int32_t Z1, f32x2 bias2, int32_t zero)
{
    Pair2 p;
    p.mx = pk2(__int2float_rn(wsub3(xi, X0, zero)), __int2float_rn(wsub3(xi, X1, zero)));
    p.my = pk2(__int2float_rn(wsub3(yi, Y0, zero)), __int2float_rn(wsub3(yi, Y1, zero)));
    p.mz = pk2(__int2float_rn(wsub3(zi, Z0, zero)), __int2float_rn(wsub3(zi, Z1, zero)));
    const f32x2 r2p = fma2(p.mx, p.mx, fma2(p.my, p.my, fma2(p.mz, p.mz, bias2)));
    upk2(r2p, p.a, p.b);
    p.a = scale_clamp_r2(p.a);
    p.b = scale_clamp_r2(p.b);
    p.y = pk2(rsqrt_pos(p.a), rsqrt_pos(p.b));
    p.q = mul2(pk2(p.a, p.b), p.y);
    const f32x2 w = fma2(p.q, pk1(-1.0f), pk1(2.0f));
    float wa, wb;
    upk2(w, wa, wb);
    p.z = pk2(rcp_pos(wa), rcp_pos(wb));
    p.y2 = mul2(p.y, p.y);
    p.z2 = mul2(p.z, p.z);
    p.y4 = mul2(p.y2, p.y2);
    p.z4 = mul2(p.z2, p.z2);
    return p;
}

// t/32 = yh^5 + zh^5 - 2 (raw pair-sum term t = y^5 + z^5 - 64, u = c1 t); exactly 0 at the clamp
__device__ __forceinline__ f32x2 pair_t(const Pair2 &p) { return fma2(p.z4, p.z, fma2(p.y4, p.y, pk1(-2.0f))); }

// HFD-B(HE) of the two pairs in K (in units of f32_scale K).  The hardware rsqrt is first refined by one Newton step
// (the seed is good to ~2^-22 and the repulsive exponential amplifies a relative error of r ~11x), written as
//   c = 1/2 - q yh / 2 (one FMA: the small correction keeps its full relative precision),  Y = yh + yh c,  R = q + q c.
// The form Y = yh f with f = 3/2 - q yh / 2 costs the same four instructions but rounds f on the fp32 grid around 1
// (spacing 6e-8 below, 1.2e-7 above): measured mean errors -1.5e-8 on Y and -1.0e-8 on R, i.e. -9e-8 on Y^6 and
// +1.4e-7 on the repulsive term -- the +0.5 ... 2e-6 systematic error V used to carry, since the two sums are each
// several times |V|.  With c the means are < 4e-10.
__device__ __forceinline__ f32x2 aziz2(const Pair2 &p, const AzizF32 &E)
{
    const f32x2 c = fma2(p.q, mul2(p.y, pk1(-0.5f)), pk1(0.5f));
    const f32x2 y = fma2(p.y, c, p.y);
    const f32x2 r = fma2(p.q, c, p.q);
    const f32x2 v = mul2(y, y);
    const f32x2 v3 = mul2(mul2(v, v), v);
    const f32x2 ndisp = mul2(v3, fma2(v, fma2(v, E.nk10, E.nk8), E.nk6));   // -disp
    const f32x2 t = fma2(E.Dl, y, fma2(E.Dh, y, E.nDc));                    // sqrt(log2 e) (D/x - 1)
    float ta, tb;
    upk2(t, ta, tb);
    const f32x2 tc = pk2(fmaxf(ta, 0.0f), fmaxf(tb, 0.0f));                 // F = 1 for x >= D
    float f0, f1;
    upk2(mul2(tc, tc), f0, f1);
    const f32x2 F = pk2(ex2_approx(-f0), ex2_approx(-f1));
    const f32x2 t1 = fma2(E.a2h, r, E.a1h);
    const f32x2 ah = mul2(r, t1);
    float r0, r1, t10, t11, h0, h1;
    upk2(r, r0, r1);
    upk2(t1, t10, t11);
    upk2(ah, h0, h1);
    f32x2 al = pk2(fmaf(r0, t10, -h0), fmaf(r1, t11, -h1));                 // exact residual of the product
    al = fma2(r, fma2(E.a2l, r, E.a1l), al);
    const f32x2 e2 = pk2(ex2_approx(h0), ex2_approx(h1));
    const f32x2 rep = mul2(e2, fma2(al, E.epsAln2, E.epsA));                // eps A 2^ah (1 + ln2 al)
    return fma2(F, ndisp, rep);
}

}  // namespace e32
}  // namespace qmc
