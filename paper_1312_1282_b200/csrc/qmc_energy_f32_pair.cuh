// qmc_energy_f32_pair.cuh -- packed fp32 pair arithmetic shared by the two FP32C local-energy kernels
// (qmc_energy_f32.cu: ordered pairs, any N; qmc_energy_f32s.cu: every unordered pair once).
// Box units (L = 1, h = 1/2); coordinates are 32-bit fixed point (qmc_f32c.cuh).
#pragma once
#include "qmc_internal.h"
#include "qmc_f32c.cuh"

namespace qmc {
namespace e32 {

constexpr float kClamp = 0x1p62f;              // h^2 2^64
constexpr int   kClampBits = 0x5E800000;       // bit pattern of 2^62

// HFD-B(HE) constants for packed fp32 evaluation.  Every constant that multiplies into the steep
// repulsive exponential or the dispersion sum is folded (in fp64, on load) into ONE rounded coefficient
// or carried as hi + lo, so that no fp32 rounding of a CONSTANT puts a systematic relative error on
// every pair (the box-unit value of r_m is an arbitrary real number):
//   rep  = eps A 2^(a1 r + a2 r^2),  a1 = -alpha log2(e) / r_m,  a2 = beta log2(e) / r_m^2   (hi + lo)
//   disp = v^3 (k6 + v (k8 + v k10)),  v = y^2,  k_n = eps c_n r_m^n
//   F    = 2^(-(sqrt(log2 e) max(D r_m y - 1, 0))^2)                              (D r_m hi + lo)
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
        split(-a.alpha * a.inv_rm * log2e, a1h, a1l);
        split(a.beta * a.inv_rm * a.inv_rm * log2e, a2h, a2l);
        const float eA = (float)(a.eps * a.A);
        epsA = pk1(eA);
        epsAln2 = pk1((float)((double)eA * ln2));
        const double r2 = a.rm2, r6 = r2 * r2 * r2;
        nk6 = pk1((float)(-a.eps * a.c6 * r6));
        nk8 = pk1((float)(-a.eps * a.c8 * r6 * r2));
        nk10 = pk1((float)(-a.eps * a.c10 * r6 * r2 * r2));
        split(a.Drm * sl, Dh, Dl);
        nDc = pk1((float)(-sl));
    }
};

// Everything the pair arithmetic of two j produces.
struct Pair2 {
    f32x2 mx, my, mz;      // signed minimum image, 2^32 box units
    f32x2 yp, q;           // y 2^-32 (hardware rsqrt), r 2^32
    f32x2 y, z;            // 1/r, 1/(1-r)
    f32x2 y2, z2, y4, z4;
    float a, b;            // the two lanes of min(r^2, h^2) 2^64
};

__device__ __forceinline__ Pair2 pair_geom(int32_t xi, int32_t yi, int32_t zi, int32_t X0, int32_t X1, int32_t Y0, int32_t Y1,
                                           int32_t Z0, int32_t Z1, f32x2 bias2, int32_t zero)
{
    Pair2 p;
    p.mx = pk2(__int2float_rn(wsub3(xi, X0, zero)), __int2float_rn(wsub3(xi, X1, zero)));
    p.my = pk2(__int2float_rn(wsub3(yi, Y0, zero)), __int2float_rn(wsub3(yi, Y1, zero)));
    p.mz = pk2(__int2float_rn(wsub3(zi, Z0, zero)), __int2float_rn(wsub3(zi, Z1, zero)));
    const f32x2 r2p = fma2(p.mx, p.mx, fma2(p.my, p.my, fma2(p.mz, p.mz, bias2)));
    upk2(r2p, p.a, p.b);
    p.a = fminf(p.a, kClamp);
    p.b = fminf(p.b, kClamp);
    p.yp = pk2(rsqrt_pos(p.a), rsqrt_pos(p.b));
    p.q = mul2(pk2(p.a, p.b), p.yp);
    const f32x2 omr = fma2(p.q, pk1(-0x1p-32f), pk1(1.0f));
    float oa, ob;
    upk2(omr, oa, ob);
    p.z = pk2(rcp_pos(oa), rcp_pos(ob));
    p.y = mul2(p.yp, pk1(0x1p32f));
    p.y2 = mul2(p.y, p.y);
    p.z2 = mul2(p.z, p.z);
    p.y4 = mul2(p.y2, p.y2);
    p.z4 = mul2(p.z2, p.z2);
    return p;
}

// t = y^5 + z^5 - 64 (raw pair-sum term, u = c1 t); exactly 0 at the clamp
__device__ __forceinline__ f32x2 pair_t(const Pair2 &p) { return fma2(p.z4, p.z, fma2(p.y4, p.y, pk1(-64.0f))); }

// HFD-B(HE) of the two pairs in K.  The hardware rsqrt is first refined by one Newton step,
// y = y0 f with f = 3/2 - r^2 y0^2 / 2 (the seed is good to ~2^-22 and the repulsive exponential
// amplifies a relative error of r ~11x); r = r^2 y0 f.
__device__ __forceinline__ f32x2 aziz2(const Pair2 &p, const AzizF32 &E)
{
    const f32x2 f = fma2(p.q, mul2(p.yp, pk1(-0.5f)), pk1(1.5f));
    const f32x2 y = mul2(p.y, f);
    const f32x2 r = mul2(mul2(p.q, pk1(0x1p-32f)), f);
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
