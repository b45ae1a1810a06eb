// qmc_energy_f32s.cu -- FP32C local-energy estimator, every UNORDERED pair evaluated once.
//
// Same pair arithmetic as qmc_energy_f32.cu (packed f32x2, fixed-point minimum image, clamp-and-count cutoff),
// same schedule as the fp64 kernel of qmc_energy_f64.cu: particles in blocks of 32, a warp takes a pair of
// blocks (A, B) along a ring (B = A + k mod n, k = 0 .. n/2), lane l holds particle i = 32A + l and the
// accumulators of particle j = 32B + l, and in steps s, s+1 (one packed instruction) it evaluates the pairs
// (i_l, j_{(l+s) mod 32}) and (i_l, j_{(l+s+1) mod 32}).  G_i, S_i sums stay in the lane's registers; the terms
// of j travel by indexed shuffles to the lanes that hold them.  Halves the special-function, integer and
// FMA work of the ordered-pair kernel for the price of 8 shuffles per two pairs; it needs 32 more bytes of
// shared memory per particle (fp64 per-particle accumulators), so large N keeps the ordered-pair kernel.
//
// Cutoff as in qmc_energy_f32.cu: r^2 clamped to h^2, where a pair adds exactly 0 to S and G and exactly the
// constants K_L = 768 and K_V = V(h) to the Laplacian and potential sums; clamped slots (beyond the cutoff,
// padding particles, the inactive half of the last diagonal step: forced by a bias on r^2) are counted and
// their constants removed in fp64.
//
// R20: per-pair terms are fp32; at most 16 of them are summed in fp32 (two packed lanes of 8) before they are
// added to an fp64 accumulator (per-lane accumulators for i, shared memory for j; fixed order, reproducible to the bit).
#include "qmc_energy_f32_pair.cuh"

namespace qmc {

namespace {

using namespace e32;

constexpr int kMaxOwn32 = 20;                        // i-blocks one warp can own (planner: ceil(nblk / nwarps) <= kMaxOwn32)

__device__ __forceinline__ float shfl_f(float v, int src) { return __shfl_sync(0xffffffffu, v, src); }

struct SymAcc {            // fp32 partial sums of up to 8 packed steps
    f32x2 gxi, gyi, gzi, si;       // this lane's particle i
    f32x2 gxj, gyj, gzj, sj;       // the particle j this lane holds
    f32x2 lam, v;                  // totals
};

// Eight packed steps (16 pairs) of one block pair, starting at step s0 (step s pairs lane l with j-lane (l+s) & 31).
//   kBias: some slots must be forced beyond the cutoff (padding particles, second half of diagonal step 16)
template <bool kEnergy, bool kBias>
__device__ __forceinline__ void sym_steps16(const int32_t *__restrict__ x, const int32_t *__restrict__ y, const int32_t *__restrict__ z,
                                            int jb, int s0, int lane, bool vi, int N, bool diag,
                                            int32_t xi, int32_t yi, int32_t zi, const AzizF32 &E, int32_t zero,
                                            SymAcc &P, int &n_in)
{
#pragma unroll 2
    for (int p = 0; p < 8; ++p) {
        const int sa = s0 + 2 * p, sb = sa + 1;
        const int ja = (lane + sa) & 31, jl = (lane + sb) & 31;
        f32x2 bias2 = pk1(0.0f);
        if (kBias) {
            const bool oka = vi && (jb + ja < N);
            const bool okb = vi && (jb + jl < N) && !(diag && sb == 16 && lane >= 16);
            bias2 = pk2(oka ? 0.0f : 0x1p63f, okb ? 0.0f : 0x1p63f);
        }
        const Pair2 q = pair_geom(xi, yi, zi, x[jb + ja], x[jb + jl], y[jb + ja], y[jb + jl], z[jb + ja], z[jb + jl], bias2, zero);
        n_in += (__float_as_int(q.a) < kClampBits ? 1 : 0) + (__float_as_int(q.b) < kClampBits ? 1 : 0);
        const f32x2 t = pair_t(q);
        P.si = add2(P.si, t);
        float t0, t1;
        upk2(t, t0, t1);
        // lane m holds j = m: it receives the first pair's terms from lane m - sa, the second's from m - sb
        const int fa = (lane - sa) & 31, fb = (lane - sb) & 31;
        P.sj = add2(P.sj, pk2(shfl_f(t0, fa), shfl_f(t1, fb)));
        if (kEnergy) {
            const f32x2 y6 = mul2(q.y4, q.y2), z6 = mul2(q.z4, q.z2);
            const f32x2 y7 = mul2(y6, q.y), z6y = mul2(z6, q.y), z7 = mul2(z6, q.z);
            const f32x2 gm = sub2(y7, z6y);
            const f32x2 cx = mul2(gm, q.mx), cy = mul2(gm, q.my), cz = mul2(gm, q.mz);
            P.gxi = add2(P.gxi, cx);
            P.gyi = add2(P.gyi, cy);
            P.gzi = add2(P.gzi, cz);
            float a0, a1, b0, b1, c0, c1;
            upk2(cx, a0, a1);
            upk2(cy, b0, b1);
            upk2(cz, c0, c1);
            P.gxj = add2(P.gxj, pk2(shfl_f(a0, fa), shfl_f(a1, fb)));      // subtracted when flushed (d_ji = -d_ij)
            P.gyj = add2(P.gyj, pk2(shfl_f(b0, fa), shfl_f(b1, fb)));
            P.gzj = add2(P.gzj, pk2(shfl_f(c0, fa), shfl_f(c1, fb)));
            P.lam = add2(P.lam, fma2(y7, pk1(2.0f), fma2(z7, pk1(3.0f), z6y)));
            P.v = add2(P.v, aziz2(q, E));
        }
    }
}

template <int T, bool kEnergy>
__global__ void __launch_bounds__(T, (T <= 128 ? 4 : (T <= 256 ? 2 : 1)))
energy32s_kernel(StateView sv, double Dk, double *__restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = sv.N, ld = sv.ld;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int nwarps = T >> 5;
    const int w = blockIdx.x;
    const int nblk = (N + 31) >> 5, NP = nblk << 5;

    double  *red = reinterpret_cast<double *>(smem_raw);              // [3][32]
                                                                      // red[97]: opaque zero
    double  *ag  = red + 98;                                          // [4][NP]: G_x, G_y, G_z (2^32 box units), S
    int32_t *x   = reinterpret_cast<int32_t *>(ag + 4 * NP);          // [3][NP]
    int32_t *y = x + NP, *z = x + 2 * NP;

    const GroupDev g = sv.groups[sv.group_of[w]];
    AzizF32 E;
    E.load(g.az);

    const float *gpos = reinterpret_cast<const float *>(sv.pos) + (size_t)w * 3 * ld;
    for (int j = tid; j < NP; j += T) {
        const bool in = j < N;
        x[j] = in ? enc_coord(gpos[j]) : 0;
        y[j] = in ? enc_coord(gpos[ld + j]) : 0;
        z[j] = in ? enc_coord(gpos[2 * ld + j]) : 0;
        ag[j] = 0.0; ag[NP + j] = 0.0; ag[2 * NP + j] = 0.0; ag[3 * NP + j] = 0.0;
    }
    if (tid == 0) *reinterpret_cast<int32_t *>(red + 97) = 0;
    __syncthreads();
    const int32_t zero = opaque_zero(reinterpret_cast<int32_t *>(red + 97));

    float KV = 0.0f;                                                  // V of a clamped slot, by the same instructions
    if (kEnergy) {
        const Pair2 pc = pair_geom(0, 0, 0, 0, 0, 0, 0, 0, 0, pk1(0x1p63f), zero);
        float va, vb;
        upk2(aziz2(pc, E), va, vb);
        KV = va;
    }

    // Schedule as in qmc_energy_f64.cu (deterministic): warp v owns the i-blocks A = v, v + nwarps, ...;
    // all warps step through the ring offsets k together (one barrier per offset), so within one offset the j-blocks
    // B = A + k of different warps are different and the j-side sums are added to shared memory by plain
    // read-modify-writes in the order of k; the i-side sums wait in local accumulators until the last offset.
    const int K = (nblk - 1) >> 1;
    const bool even = (nblk & 1) == 0, ragged = (N & 31) != 0;
    double tLam = 0.0, tV = 0.0;
    long long slots = 0, inside = 0;
    double own[kMaxOwn32][4];                                         // G_x, G_y, G_z, S of this lane's particle in each own block
#pragma unroll 1
    for (int a = 0; a < kMaxOwn32; ++a) { own[a][0] = 0.0; own[a][1] = 0.0; own[a][2] = 0.0; own[a][3] = 0.0; }
    const int kend = K + (even ? 1 : 0);
#pragma unroll 1
    for (int k = 0; k <= kend; ++k) {
        int a = 0;
#pragma unroll 1
        for (int A = warp; A < nblk; A += nwarps, ++a) {
            if (k > K && A >= (nblk >> 1)) break;                    // even n: the offset n/2 once per block pair
            const int i = (A << 5) + lane;
            const bool vi = i < N;
            const int32_t xi = x[i], yi = y[i], zi = z[i];
            double gxi = 0.0, gyi = 0.0, gzi = 0.0, si = 0.0;
            int B = A + k;
            if (B >= nblk) B -= nblk;
            const int jb = B << 5;
            const bool diag = (k == 0);
            const bool bias = diag || (ragged && (A == nblk - 1 || B == nblk - 1));
            double gxj = 0.0, gyj = 0.0, gzj = 0.0, sj = 0.0;
            const int nhalf = diag ? 1 : 2;
            for (int hlf = 0; hlf < nhalf; ++hlf) {
                SymAcc P;
                P.gxi = P.gyi = P.gzi = P.si = P.gxj = P.gyj = P.gzj = P.sj = P.lam = P.v = pk1(0.0f);
                int n_in = 0;
                const int s0 = diag ? 1 : 16 * hlf;
                if (bias) sym_steps16<kEnergy, true>(x, y, z, jb, s0, lane, vi, N, diag, xi, yi, zi, E, zero, P, n_in);
                else      sym_steps16<kEnergy, false>(x, y, z, jb, s0, lane, vi, N, diag, xi, yi, zi, E, zero, P, n_in);
                slots += 16; inside += n_in;
                si += (double)hsum2(P.si);
                sj += (double)hsum2(P.sj);
                if (kEnergy) {
                    gxi += (double)hsum2(P.gxi); gyi += (double)hsum2(P.gyi); gzi += (double)hsum2(P.gzi);
                    gxj += (double)hsum2(P.gxj); gyj += (double)hsum2(P.gyj); gzj += (double)hsum2(P.gzj);
                    tLam += (double)hsum2(P.lam);
                    tV += (double)hsum2(P.v);
                }
            }
            if (jb + lane < N) {
                ag[3 * NP + jb + lane] += sj;
                if (kEnergy) {
                    ag[jb + lane] -= gxj;
                    ag[NP + jb + lane] -= gyj;
                    ag[2 * NP + jb + lane] -= gzj;
                }
            }
            own[a][3] += si;
            if (kEnergy) { own[a][0] += gxi; own[a][1] += gyi; own[a][2] += gzi; }
        }
        __syncthreads();
    }
    {
        int a = 0;
#pragma unroll 1
        for (int A = warp; A < nblk; A += nwarps, ++a) {
            const int i = (A << 5) + lane;
            if (i < N) {
                ag[3 * NP + i] += own[a][3];
                if (kEnergy) { ag[i] += own[a][0]; ag[NP + i] += own[a][1]; ag[2 * NP + i] += own[a][2]; }
            }
        }
    }
    __syncthreads();

    double tG2 = 0.0;
    for (int i = tid; i < N; i += T) {
        sv.S[(size_t)w * ld + i] = ag[3 * NP + i];                    // R17: rebuild the running sum
        if (kEnergy) {
            const double a = ag[i], b = ag[NP + i], c = ag[2 * NP + i];
            tG2 += a * a + b * b + c * c;
        }
    }
    if (kEnergy) {
        const double n_out = (double)(slots - inside);
        tLam = 2.0 * (tLam - 768.0 * n_out);                          // each unordered pair seen once
        tV -= (double)KV * n_out;
        tLam = warp_sum(tLam); tG2 = warp_sum(tG2); tV = warp_sum(tV);
        if (lane == 0) { red[warp] = tLam; red[32 + warp] = tG2; red[64 + warp] = tV; }
        __syncthreads();
        if (warp == 0) {
            double a = lane < nwarps ? red[lane] : 0.0;
            double b = lane < nwarps ? red[32 + lane] : 0.0;
            double c = lane < nwarps ? red[64 + lane] : 0.0;
            a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
            if (lane == 0) {
                const double Dku = Dk * g.inv_unit * g.inv_unit;
                const double lam = -5.0 * g.b5 * a;                                     // sum_i Lambda_i
                const double g2 = (2.5 * g.b5 * 0x1p-32) * (2.5 * g.b5 * 0x1p-32) * b;   // sum_i |G_i|^2
                const double T_PB = -Dku * (lam + g2);
                const double T_JF = -0.5 * Dku * lam;
                double *o = out + (size_t)w * 4;
                o[0] = c + T_PB; o[1] = c; o[2] = T_PB; o[3] = T_JF;
            }
        }
    }
}

int smem_bytes32s(int N) { const int NP = ((N + 31) >> 5) << 5; return 98 * 8 + 4 * NP * 8 + 3 * NP * 4; }

template <int T>
cudaError_t launch32s(qmc_ctx *c, double *d_out, bool energy)
{
    const int smem = smem_bytes32s(c->p.N);
    cudaError_t e;
    if (energy) {
        auto k = energy32s_kernel<T, true>;
        if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
        k<<<c->W, T, smem, c->stream>>>(c->sv, c->p.hbar2_over_2m, d_out);
    } else {
        auto k = energy32s_kernel<T, false>;
        if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
        k<<<c->W, T, smem, c->stream>>>(c->sv, c->p.hbar2_over_2m, d_out);
    }
    return cudaGetLastError();
}

template <int T>
int occupancy32s(int smem)
{
    int occ = 0;
    auto k = energy32s_kernel<T, true>;
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, T, smem);
    return occ;
}

}  // namespace

#define QMC_E32S_THREADS(X) X(32) X(64) X(128) X(256) X(512)

cudaError_t launch_energy_f32s(qmc_ctx *c, double *d_out, bool energy)
{
    const int T = c->energy_plan.threads;
#define X(TT) if (T == TT) return launch32s<TT>(c, d_out, energy);
    QMC_E32S_THREADS(X)
#undef X
    return cudaErrorInvalidValue;
}

// false: the per-particle fp64 accumulators do not leave room for two CTAs per SM (N > ~2500) -- the caller
// keeps the ordered-pair kernel.  qmc_set_tuning("energy_threads") overrides the thread count (tuning experiments).
bool plan_energy_f32s(qmc_ctx *c, EnergyPlan *out)
{
    const int N = c->p.N;
    const int smem = smem_bytes32s(N);
    if (smem > 113 * 1024) return false;
    int T = 32;
    while (2 * T < N && T < 256) T *= 2;
    if (g_tuning.energy_threads > 0) {
        const int v = g_tuning.energy_threads;
        if (v >= 32 && v <= 512 && (v & (v - 1)) == 0) T = v;
    }
    const int nblk = (N + 31) >> 5;
    while ((nblk + (T >> 5) - 1) / (T >> 5) > kMaxOwn32 && T < 512) T *= 2;     // own-block accumulators per warp
    if ((nblk + (T >> 5) - 1) / (T >> 5) > kMaxOwn32) return false;
    out->threads = T;
    out->smem_bytes = smem;
    out->variant = 2;
    out->ctas_per_sm = 0;
#define X(TT) if (T == TT) out->ctas_per_sm = occupancy32s<TT>(smem);
    QMC_E32S_THREADS(X)
#undef X
    return true;
}

}  // namespace qmc
