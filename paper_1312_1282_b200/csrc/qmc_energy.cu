// qmc_energy.cu -- local-energy estimator over all pairs and the
// from-scratch rebuild of the running pair sums S_i.
//
// One CTA per walker, coordinates in shared memory; thread t owns particles i = t, t+T, ... and
// streams every j from shared memory (all lanes read the same j: a broadcast, no bank conflicts),
// keeping grad_i log psi, lap_i log psi, V and S_i in registers -- the scatter-free n-body layout
// ("extra memory to store wavefunction derivatives": here they never leave registers).
//
//   G_i      = sum_{j != i} u'(r_ij) d_ij / r_ij          u'/r  =  5/2 b^5 y (y^6 - z^6)
//   Lambda_i = sum_{j != i} [u'' + 2 u'/r]                     =  -b^5 (10 y^7 + 15 z^7 + 5 z^6 y)
//   V        = sum_{i<j, r<h} V_Aziz(r_ij)                 (HFD-B(HE), truncated at h, R3)
//   T_PB = -Dk sum_i (Lambda_i + |G_i|^2),  T_JF = -Dk/2 sum_i Lambda_i,  E_PB = V + T_PB   (R14)
// with y = 1/r, z = 1/(L-r).  This ordered-pair kernel is the FP64 fallback for N whose per-particle accumulators do
// not fit the unordered-pair kernel of qmc_energy_f64.cu (N > ~4100) and the dispatcher of all energy kernels.
#include "qmc_internal.h"

namespace qmc {

constexpr int kFlush = 16;

// Constants of the potential as DESIGN.md §2 writes it (this file serves FP64 only; the FP32C kernels are
// qmc_energy_f32.cu and qmc_energy_f32s.cu).
template <typename Real> struct EnergyConst;

template <> struct EnergyConst<double> {
    double b5, eps, inv_rm, rm2, A, alpha, beta, c6, c8, c10, D, Drm;
    __device__ __forceinline__ void load(const GroupDev &g, const AzizDev &a)
    {
        b5 = g.b5; eps = a.eps; inv_rm = a.inv_rm; rm2 = a.rm2; A = a.A;
        alpha = a.alpha; beta = a.beta; c6 = a.c6; c8 = a.c8; c10 = a.c10;
        D = a.D; Drm = a.Drm;
    }
};

// Signed minimum-image component for |d| <= L.
template <typename Real>
__device__ __forceinline__ Real min_image_signed(Real d, const PairConst<Real> &P)
{
    const Real shift = d > P.h ? P.L : (d < -P.h ? -P.L : (Real)0);
    return d - shift;
}

// HFD-B(HE) in K from r^2, r and y = 1/r.
__device__ __forceinline__ double aziz_pair(double, double r, double y, const EnergyConst<double> &E)
{
    const double x = r * E.inv_rm;
    const double w = E.rm2 * y * y;                             // 1/x^2
    const double disp = w * w * w * fma(w, fma(w, E.c10, E.c8), E.c6);
    double F = 1.0;
    if (x < E.D) {
        const double t = E.Drm * y - 1.0;                       // D/x - 1
        F = exp(-t * t);
    }
    const double rep = E.A * exp(x * fma(E.beta, x, -E.alpha));
    return E.eps * (rep - F * disp);
}

template <typename Real, int T, bool kEnergy>
__global__ void __launch_bounds__(T)
energy_kernel(StateView sv, double Dk, double *__restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = sv.N, ld = sv.ld;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int nwarps = T >> 5;
    const int w = blockIdx.x;

    double *red = reinterpret_cast<double *>(smem_raw);            // [3][32]
    Real *X = reinterpret_cast<Real *>(red + 96);                  // [3][ld]
    Real *x = X, *y = X + ld, *z = X + 2 * ld;

    const GroupDev g = sv.groups[sv.group_of[w]];
    PairConst<Real> P;
    P.load(g);
    EnergyConst<Real> E;
    E.load(g, g.az);
    const Real sh = (Real)g.sh;

    const Real *gpos = reinterpret_cast<const Real *>(sv.pos) + (size_t)w * 3 * ld;
    {
        uint4 *d = reinterpret_cast<uint4 *>(X);
        const uint4 *s = reinterpret_cast<const uint4 *>(gpos);
        for (int i = tid; i < 3 * ld * (int)sizeof(Real) / 16; i += T) d[i] = s[i];
    }
    __syncthreads();

    double tLam = 0.0, tG2 = 0.0, tV = 0.0;
    const int n_iter = (N + T - 1) / T;                            // same trip count for every thread (votes)
    for (int it = 0; it < n_iter; ++it) {
        const int i = tid + it * T;
        const bool live = i < N;
        const int ic = live ? i : N - 1;
        const Real xi = x[ic], yi = y[ic], zi = z[ic];
        double gx = 0.0, gy = 0.0, gz = 0.0, lam = 0.0, v = 0.0, s = 0.0;
        for (int j0 = 0; j0 < N; j0 += kFlush) {
            Real pgx = 0, pgy = 0, pgz = 0, plam = 0, pv = 0, ps = 0;
            const int j1 = min(j0 + kFlush, N);
            for (int j = j0; j < j1; ++j) {
                const Real dx = min_image_signed<Real>(xi - x[j], P);
                const Real dy = min_image_signed<Real>(yi - y[j], P);
                const Real dz = min_image_signed<Real>(zi - z[j], P);
                Real r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                const bool in = (r2 < P.h2) && (j != ic) && live;
                if (!in) r2 = P.h2;
                const Real yy = rsqrt_pos(r2);
                const Real r = r2 * yy;
                const Real zz = rcp_pos(P.L - r);
                const Real y2 = yy * yy, z2 = zz * zz;
                const Real y4 = y2 * y2, z4 = z2 * z2;
                const Real t = fma(z4, zz, fma(y4, yy, -sh));      // raw pair sum term, u = c1 t
                ps += in ? t : (Real)0;
                if (kEnergy) {
                    const Real y6 = y4 * y2, z6 = z4 * z2;
                    const Real y7 = y6 * yy, z7 = z6 * zz;
                    const Real gr = (Real)2.5 * E.b5 * yy * (y6 - z6);               // u'/r
                    const Real lt = -E.b5 * fma((Real)10, y7, fma((Real)15, z7, (Real)5 * z6 * yy));
                    const Real gm = in ? gr : (Real)0;
                    pgx = fma(gm, dx, pgx);
                    pgy = fma(gm, dy, pgy);
                    pgz = fma(gm, dz, pgz);
                    plam += in ? lt : (Real)0;
                    const bool needV = in && (j > ic);
                    if (__any_sync(0xffffffffu, needV)) {
                        const Real vp = aziz_pair(r2, r, yy, E);
                        pv += needV ? vp : (Real)0;
                    }
                }
            }
            s += (double)ps;
            if (kEnergy) {
                gx += (double)pgx; gy += (double)pgy; gz += (double)pgz;
                lam += (double)plam; v += (double)pv;
            }
        }
        if (live) {
            sv.S[(size_t)w * ld + i] = s;                          // R17: rebuild the running sum
            tLam += lam;
            tG2 += gx * gx + gy * gy + gz * gz;
            tV += v;
        }
    }

    if (kEnergy) {
        tLam = warp_sum(tLam); tG2 = warp_sum(tG2); tV = warp_sum(tV);
        if (lane == 0) { red[warp] = tLam; red[32 + warp] = tG2; red[64 + warp] = tV; }
        __syncthreads();
        if (warp == 0) {
            double a = lane < nwarps ? red[lane] : 0.0;
            double b = lane < nwarps ? red[32 + lane] : 0.0;
            double c = lane < nwarps ? red[64 + lane] : 0.0;
            a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
            if (lane == 0) {
                const double Dku = Dk * g.inv_unit * g.inv_unit;       // gradients are per coordinate unit
                const double T_PB = -Dku * (a + b);
                const double T_JF = -0.5 * Dku * a;
                double *o = out + (size_t)w * 4;
                o[0] = c + T_PB; o[1] = c; o[2] = T_PB; o[3] = T_JF;
            }
        }
    }
}

static int energy_smem_bytes(int ld, int mode)
{
    return 96 * 8 + 3 * ld * ((mode == QMC_FP64) ? 8 : 4);
}

#define QMC_ENERGY_THREADS(X) X(32) X(64) X(128) X(256) X(512) X(1024)

template <typename Real, int T>
static cudaError_t launch_e(qmc_ctx *c, double *d_out, bool energy)
{
    const int smem = c->energy_plan.smem_bytes;
    cudaError_t e;
    if (energy) {
        auto k = energy_kernel<Real, T, true>;
        if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
        k<<<c->W, T, smem, c->stream>>>(c->sv, c->p.hbar2_over_2m, d_out);
    } else {
        auto k = energy_kernel<Real, T, false>;
        if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
        k<<<c->W, T, smem, c->stream>>>(c->sv, c->p.hbar2_over_2m, d_out);
    }
    return cudaGetLastError();
}

cudaError_t launch_energy(qmc_ctx *c, double *d_out, bool energy)
{
    c->launches += 1;
    if (c->p.mode != QMC_FP64) {
        if (c->energy_plan.variant == 3) { c->launches -= 1; return launch_energy_f32g(c, d_out, energy); }   // counts its own launches
        return c->energy_plan.variant == 2 ? launch_energy_f32s(c, d_out, energy)    // qmc_energy_f32s.cu
                                           : launch_energy_f32(c, d_out, energy);    // qmc_energy_f32.cu
    }
    if (c->energy_plan.variant == 1) return launch_energy_f64(c, d_out, energy);  // qmc_energy_f64.cu
    const int T = c->energy_plan.threads;
#define X(TT) if (T == TT) return launch_e<double, TT>(c, d_out, energy);
    QMC_ENERGY_THREADS(X)
#undef X
    return cudaErrorInvalidValue;
}

bool plan_energy(qmc_ctx *c, EnergyPlan *out)
{
    out->variant = 0;
    out->parts = 1;
    if (c->p.mode != QMC_FP64) {
        // one walker per block while that fills the GPU; the gridded kernel for few walkers of many atoms (a block
        // per walker would leave SMs idle) and for N beyond one block's shared memory.
        // qmc_set_tuning("energy_ordered"): 0 heuristic, 1 ordered pairs, 2 unordered pairs, 3 gridded.
        const int want = c->tuning.energy_ordered;
        const bool few = (long long)c->W * 2 < c->sm_count && c->p.N >= 1024;
        if (want == 3 || (want == 0 && few)) return plan_energy_f32g(c, out);
        if (want != 1 && plan_energy_f32s(c, out)) return true;
        out->variant = 0;
        if (plan_energy_f32(c, out)) return true;
        return plan_energy_f32g(c, out);
    }
    if (c->tuning.energy_ordered != 1 && plan_energy_f64(c, out)) return true;
    out->variant = 0;
    const int N = c->p.N;
    int T = 32;
    while (T < N && T < 256) T *= 2;
    if (c->tuning.energy_threads > 0) {
        const int v = c->tuning.energy_threads;
        if (v >= 32 && v <= 1024 && (v & (v - 1)) == 0) T = v;
    }
    out->threads = T;
    out->smem_bytes = energy_smem_bytes(c->ld, c->p.mode);
    if (out->smem_bytes > 227 * 1024) return false;
    int occ = 0;
#define X(TT) if (T == TT) { auto k = energy_kernel<double, TT, true>; \
            cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, out->smem_bytes); \
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, TT, out->smem_bytes); }
    QMC_ENERGY_THREADS(X)
#undef X
    out->ctas_per_sm = occ;
    return true;
}

}  // namespace qmc
