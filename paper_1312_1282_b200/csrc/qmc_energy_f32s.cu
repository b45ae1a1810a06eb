// qmc_energy_f32s.cu -- FP32C local-energy estimator, every UNORDERED pair evaluated once.
//
// Same pair arithmetic as qmc_energy_f32.cu (packed f32x2, fixed-point minimum image, clamp-and-count cutoff),
// same schedule as the fp64 kernel of qmc_energy_f64.cu: particles in blocks of 32, a warp takes a pair of
// blocks (A, B) along a ring (B = A + k mod n, k = 0 .. n/2), lane l holds particle i = 32A + l and the
// accumulators of particle j = 32B + l, and in steps s, s+1 (one packed instruction) it evaluates the pairs
// (i_l, j_{(l+s) mod 32}) and (i_l, j_{(l+s+1) mod 32}).  G_i, S_i sums stay in the lane's registers; the terms
// of j travel by indexed shuffles to the lanes that hold them.  Halves the special-function, integer and
// FMA work of the ordered-pair kernel for the price of 8 shuffles per two pairs; it needs 32 more bytes of
// shared memory per particle (64-bit per-particle accumulators), so large N keeps the ordered-pair kernel.
//
// Cutoff as in qmc_energy_f32.cu: r^2 clamped to h^2, where a pair adds exactly 0 to S and G and exactly the
// constants K_L = 768 (6 in the kernel's units, qmc_energy_f32_pair.cuh) and K_V = V(h) to the Laplacian and
// potential sums; clamped slots (beyond the cutoff, padding particles, the inactive half of the last diagonal
// step: forced by a bias on r^2) are counted and their constants removed in fp64.
//
// R20: per-pair terms are fp32; a packed lane sums at most 16 of them in fp32, the two lanes are added (32 terms, one
// block pair) and the result goes to a wide accumulator: 64-bit fixed point for the per-particle sums (integer
// atomic adds in shared memory: exact, hence independent of the order of arrival and reproducible to the bit), fp64
// for the per-thread totals.
#include "qmc_energy_f32_pair.cuh"

namespace qmc {

namespace {

using namespace e32;

// fixed-point grids of the per-particle accumulators: 2^-24 of a pair-sum term (t/32) and of a gradient term
// (gm/128 times the minimum image in box units; the terms arrive times 2^32)
constexpr double kFixS = 0x1p24, kFixG = 0x1p-8;
// bad: a partial sum the fixed-point accumulator cannot carry -- not finite (two particles on one grid point), or so
// large that a few of them would wrap the 56-bit hi:lo sum of a particle (|sum| < 2^55 units): anything
// from 2^52 units up, i.e. |v| >= 2^28 for a pair-sum partial and 2^60 for a gradient partial.  A pair-sum partial
// reaches 2^28 only with a pair closer than ~0.01 L (a liquid's nearest pairs, r > 0.04 L, give ~2^18), where the fp32
// pair term has lost the rest of the sum anyway.  Eight such partials on ONE particle stay inside the range; more
// would need nine partners of one particle within 0.01 L of it, in nine different blocks of 32.
__device__ __forceinline__ long long fix_s(float v, bool &bad) { bad |= !(fabsf(v) < 0x1p28f); return __float2ll_rn(v * 0x1p24f); }
__device__ __forceinline__ long long fix_g(float v, bool &bad) { bad |= !(fabsf(v) < 0x1p60f); return __float2ll_rn(v * 0x1p-8f); }
// A 64-bit fixed-point accumulator is two 32-bit words, hi (signed, units of 2^24) and lo (unsigned): v = hi 2^24 +
// lo with 0 <= lo < 2^24 is added by TWO native 32-bit shared-memory atomics (a 64-bit atomic add on shared memory is
// a compare-and-swap loop).  A particle receives at most nblk + 1 <= 81 additions, so lo stays below 2^31 and no
// carry is ever lost; fix_get() puts the words together.
__device__ __forceinline__ void fix_add(int32_t *ag, int idx, long long v)
{
    atomicAdd(ag + 2 * idx, (int32_t)(v >> 24));
    atomicAdd(reinterpret_cast<uint32_t *>(ag) + 2 * idx + 1, (uint32_t)v & 0xFFFFFFu);
}
__device__ __forceinline__ double fix_get(const int32_t *ag, int idx)
{
    return (double)(((long long)ag[2 * idx] << 24) + (long long)reinterpret_cast<const uint32_t *>(ag)[2 * idx + 1]);
}

__device__ __forceinline__ float shfl_f(float v, int src) { return __shfl_sync(0xffffffffu, v, src); }

struct SymAcc {            // fp32 partial sums of up to 16 packed steps
    f32x2 gxi, gyi, gzi, si;       // this lane's particle i
    f32x2 gxj, gyj, gzj, sj;       // the particle j this lane holds
    f32x2 lam, lg, v;              // totals: y^7 + z^7, gm, V
};

// npk packed steps (2 npk pairs) of one block pair, starting at step s0 (step s pairs lane l with j-lane (l+s) & 31):
// npk = 16, s0 = 0 for a full block pair, npk = 8, s0 = 1 for the diagonal block.
//   kBias: some slots must be forced beyond the cutoff (padding particles, second half of diagonal step 16)
template <bool kEnergy, bool kBias, int kUnroll>
__device__ __forceinline__ void sym_steps(const int4 *__restrict__ xyz,
                                            int jb, int s0, int npk, int lane, bool vi, int N, bool diag,
                                            int32_t xi, int32_t yi, int32_t zi, const AzizF32 &E, int32_t zero,
                                            SymAcc &P, f32x2 &n_out2)
{
#pragma unroll kUnroll
    for (int p = 0; p < npk; ++p) {
        const int sa = s0 + 2 * p, sb = sa + 1;
        const int ja = (lane + sa) & 31, jl = (lane + sb) & 31;
        f32x2 bias2 = pk1(0.0f);
        if (kBias) {
            const bool oka = vi && (jb + ja < N);
            const bool okb = vi && (jb + jl < N) && !(diag && sb == 16 && lane >= 16);
            bias2 = pk2(oka ? 0.0f : 0x1p63f, okb ? 0.0f : 0x1p63f);
        }
        const int4 ca = xyz[jb + ja], cb = xyz[jb + jl];             // one 16-byte read per particle
        const Pair2 q = pair_geom(xi, yi, zi, ca.x, cb.x, ca.y, cb.y, ca.z, cb.z, bias2, zero);
        // clamped slots are counted in fp32 (exact far beyond the ~1e4 slots a thread sees): two compares that write
        // 1.0f / 0.0f and one packed add instead of compare + predicated integer add per slot
        if (kEnergy) n_out2 = add2(n_out2, pk2(q.a < 1.0f ? 0.0f : 1.0f, q.b < 1.0f ? 0.0f : 1.0f));
        const f32x2 t = pair_t(q);
        P.si = add2(P.si, t);
        float t0, t1;
        upk2(t, t0, t1);
        // lane m holds j = m: it receives the first pair's terms from lane m - sa, the second's from m - sb
        const int fa = lane - sa, fb = lane - sb;                    // shfl takes the source lane modulo 32
        P.sj = add2(P.sj, pk2(shfl_f(t0, fa), shfl_f(t1, fb)));
        if (kEnergy) {
            // gm = (y^6 - z^6) y;  Laplacian term 2 y^7 + 3 z^7 + z^6 y = 3 (y^7 + z^7) - gm: the two sums are kept apart
            const f32x2 y6 = mul2(q.y4, q.y2), z6 = mul2(q.z4, q.z2);
            const f32x2 gm = mul2(sub2(y6, z6), q.y);
            P.lam = fma2(z6, q.z, fma2(y6, q.y, P.lam));
            P.lg = add2(P.lg, gm);
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
            P.v = add2(P.v, aziz2(q, E));
        }
    }
}

template <int T, bool kEnergy>
__global__ void __launch_bounds__(T, (T <= 128 ? 4 : (T <= 384 ? 2 : 1)))
energy32s_kernel(StateView sv, double Dk, double *__restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = sv.N, ld = sv.ld;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int nwarps = T >> 5;
    // packed pair steps in flight per lane: 4 with 128 registers (T <= 256, T = 512), 2 with the 85 of T = 384
    // (measured: 10.01 against 10.34 ms with 2 at T = 256; 9.05 against 9.12 ms with 4 at T = 384)
    constexpr int kSteps = (T == 384) ? 2 : 4;
    const int w = blockIdx.x;
    const int nblk = (N + 31) >> 5, NP = nblk << 5;

    double  *red = reinterpret_cast<double *>(smem_raw);              // [3][32]
                                                                      // red[97]: opaque zero
    int32_t *ag = reinterpret_cast<int32_t *>(red + 98);              // [4][NP][2]: G_x, G_y, G_z, S as fixed point (hi, lo)
    int4 *xyz = reinterpret_cast<int4 *>(ag + 8 * NP);                // [NP]: fixed-point x, y, z of a particle in one 16-byte word

    const GroupDev g = sv.groups[sv.group_of[w]];
    AzizF32 E;
    E.load(g.az);

    const float *gpos = reinterpret_cast<const float *>(sv.pos) + (size_t)w * 3 * ld;
    for (int j = tid; j < NP; j += T) {
        const bool in = j < N;
        xyz[j] = in ? make_int4(enc_coord(gpos[j]), enc_coord(gpos[ld + j]), enc_coord(gpos[2 * ld + j]), 0) : make_int4(0, 0, 0, 0);
        *reinterpret_cast<int2 *>(ag + 2 * j) = make_int2(0, 0);
        *reinterpret_cast<int2 *>(ag + 2 * (NP + j)) = make_int2(0, 0);
        *reinterpret_cast<int2 *>(ag + 2 * (2 * NP + j)) = make_int2(0, 0);
        *reinterpret_cast<int2 *>(ag + 2 * (3 * NP + j)) = make_int2(0, 0);
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

    // Schedule (deterministic): the block pairs (A, B = A + k), k = 0 .. K (+ the offset n/2 once per pair for
    // even n), form one flat task list that the warps take round-robin -- a fixed set in a fixed order per warp, so the
    // per-thread totals are reproducible.  The per-particle sums of BOTH blocks of a task go to shared memory as 64-bit
    // FIXED-POINT numbers by integer atomic adds: integer addition is associative, so the result does not depend on the
    // order in which the warps arrive, and the main loop needs no barrier at all (round 2's per-offset barrier and
    // thread-local accumulator arrays are gone).  The fixed-point grid is 2^-24 of the kernel's units (kFixS, kFixG):
    // finer than the fp32 partial sums that are added to it (|partial| >= 1 converts exactly), 63 bits of range.
    const int K = (nblk - 1) >> 1;
    const bool even = (nblk & 1) == 0, ragged = (N & 31) != 0;
    double tLam = 0.0, tLg = 0.0, tV = 0.0;
    f32x2 n_out2 = pk1(0.0f);                                         // clamped slots, per packed lane
    bool bad = false;
    int k = warp / nblk, A = warp - k * nblk;                         // task t = warp, warp + nwarps, ...: k = t / n, A = t mod n
#pragma unroll 1
    for (;;) {
        if (k > K && !(even && k == K + 1 && A < (nblk >> 1))) break;   // even n: the offset n/2 once per block pair
        const int i = (A << 5) + lane;
        const bool vi = i < N;
        const int4 ci = xyz[i];
        const int32_t xi = ci.x, yi = ci.y, zi = ci.z;
        int B = A + k;
        if (B >= nblk) B -= nblk;
        const int jb = B << 5;
        const bool diag = (k == 0);
        const bool bias = diag || (ragged && (A == nblk - 1 || B == nblk - 1));
        SymAcc P;
        P.gxi = P.gyi = P.gzi = P.si = P.gxj = P.gyj = P.gzj = P.sj = P.lam = P.lg = P.v = pk1(0.0f);
        const int s0 = diag ? 1 : 0, npk = diag ? 8 : 16;
        if (bias) sym_steps<kEnergy, true, kSteps>(xyz, jb, s0, npk, lane, vi, N, diag, xi, yi, zi, E, zero, P, n_out2);
        else      sym_steps<kEnergy, false, kSteps>(xyz, jb, s0, npk, lane, vi, N, diag, xi, yi, zi, E, zero, P, n_out2);
        if (kEnergy) {
            tLam += (double)hsum2(P.lam);
            tLg += (double)hsum2(P.lg);
            tV += (double)hsum2(P.v);
        }
        if (jb + lane < N) {
            fix_add(ag, 3 * NP + jb + lane, fix_s(hsum2(P.sj), bad));
            if (kEnergy) {
                fix_add(ag, jb + lane, -fix_g(hsum2(P.gxj), bad));         // d_ji = -d_ij
                fix_add(ag, NP + jb + lane, -fix_g(hsum2(P.gyj), bad));
                fix_add(ag, 2 * NP + jb + lane, -fix_g(hsum2(P.gzj), bad));
            }
        }
        if (vi) {
            fix_add(ag, 3 * NP + i, fix_s(hsum2(P.si), bad));
            if (kEnergy) {
                fix_add(ag, i, fix_g(hsum2(P.gxi), bad));
                fix_add(ag, NP + i, fix_g(hsum2(P.gyi), bad));
                fix_add(ag, 2 * NP + i, fix_g(hsum2(P.gzi), bad));
            }
        }
        A += nwarps;
        while (A >= nblk) { A -= nblk; ++k; }
    }
    // a singular configuration: the pair sums come out as NaN, as they would from a floating-point accumulator (for
    // coincident particles the energies below are not finite anyway: the Laplacian and potential totals are floating
    // point); a pair so close that the fixed-point sums could wrap poisons the walker's pair sums, T_PB and E_PB the same way
    // With b = 0 (free particles) every fixed-point sum is multiplied by exactly 0 downstream: nothing to flag.
    const double poison = (__syncthreads_or(bad) && g.b5 != 0.0) ? __longlong_as_double(0x7ff8000000000000LL) : 0.0;

    double tG2 = 0.0;
    for (int i = tid; i < N; i += T) {
        sv.S[(size_t)w * ld + i] = fix_get(ag, 3 * NP + i) * (kSUnit / kFixS) + poison;     // R17: rebuild the running sum
        if (kEnergy) {
            const double a = fix_get(ag, i) * (1.0 / kFixG), b = fix_get(ag, NP + i) * (1.0 / kFixG), c = fix_get(ag, 2 * NP + i) * (1.0 / kFixG);
            tG2 += a * a + b * b + c * c;
        }
    }
    if (kEnergy) {
        const double n_out = (double)hsum2(n_out2);
        tLam = 2.0 * (3.0 * (tLam - 2.0 * n_out) - tLg);              // each unordered pair seen once; a clamped slot adds y^7 + z^7 = 2, gm = 0
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
                const double lam = -5.0 * g.b5 * kGUnit * a;                            // sum_i Lambda_i
                const double g2 = (2.5 * g.b5 * kGUnit * 0x1p-32) * (2.5 * g.b5 * kGUnit * 0x1p-32) * b;   // sum_i |G_i|^2
                const double T_PB = -Dku * (lam + g2);
                const double T_JF = -0.5 * Dku * lam;
                double *o = out + (size_t)w * 4;
                const double V = c * g.az.f32_scale;                                     // the potential was summed in units of f32_scale K
                // V and T_JF are floating-point totals of their own; T_PB holds |G_i|^2 from the fixed-point sums
                o[0] = V + T_PB + poison; o[1] = V; o[2] = T_PB + poison; o[3] = T_JF;
            }
        }
    }
}

int smem_bytes32s(int N) { const int NP = ((N + 31) >> 5) << 5; return 98 * 8 + 4 * NP * 8 + 4 * NP * 4; }

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

#define QMC_E32S_THREADS(X) X(32) X(64) X(128) X(256) X(384) X(512)

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
    if (N >= 1536) T = 384;              // 24 warps per SM at 80 registers beat 16 at 128 (9.32 -> 9.12 ms at N = 1952)
    if (c->tuning.energy_threads > 0) {
        const int v = c->tuning.energy_threads;
        if (v >= 32 && v <= 512 && ((v & (v - 1)) == 0 || v == 384)) T = v;
    }
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
