// qmc_observables.cu -- pair-distance histogram per walker: the raw data of the pair distribution function
// g(r), the paper's second observable ("pair distribution function", l.468; SURVEY.md §8(f)
// NEXT-2).  Integer output, so the arithmetic that decides a bin is specified to the bit (DESIGN.md
// "Observables"): coordinates in Angstrom as fp64 (in FP32C the exact widening qmc_get_positions returns),
//   t = a - b,  d = t - L rint(t / L)   per component,
//   r = sqrt((dx dx + dy dy) + dz dz),  counted iff r < h = L/2,  k = min((int)(r * (nbins / h)), nbins - 1),
// every operation rounded once (no FMA contraction).  For |t| <= L, rint(t / L) is +1 for t > h, -1 for
// t < -h and 0 otherwise (t/L rounds to a double > 1/2 exactly when t > h, and rint(1/2) = 0), so the
// division is replaced by two comparisons with identical results.
//
// One CTA per walker, coordinates and the histogram in shared memory.  The particles are cut into blocks of 32; a warp
// takes a pair of blocks (A, B = A + k mod n) from the flat, statically dealt task list the energy kernels use
// (every unordered pair of blocks once, the diagonal block with j > i), lane l holds particle i = 32 A + l and
// the 32 particles j of block B are read as broadcast 16-byte vectors: no per-lane index arithmetic.
//
// FILTERED evaluation (round 2; the bits above are unchanged).  The specified arithmetic costs ~30 fp64 instructions
// per pair, among them a correctly rounded square root.  The kernel first computes the bin coordinate u = r nbins / h
// in fp32 from 32-bit fixed-point coordinates (the FP32C representation of qmc_f32c.cuh; in FP64 mode the coordinates
// rounded to 2^-32 of the box; the fp64 coordinates stay in global memory): wrapping integer differences, r^2,
// r = sqrt.approx(r^2), u.  Its error against the specified fp64 value is below 2e-6 u (sqrt.approx 2^-22, four fp32
// roundings, coordinate rounding 2^-33 L), i.e.
// below 1e-3 of a bin for nbins <= 512 (4e-4 with the roundings of the floor itself).  If floor(u - kGuard) == floor(u + kGuard) the pair is that far from every bin
// edge and from the cutoff (u = nbins), so the specified arithmetic gives the same bin: it is counted at once.
// Otherwise (2 kGuard = 0.4 % of the pairs) the pair goes to a per-warp queue that evaluates the specified fp64
// arithmetic 32 pairs at a time.  The result is
// bit-identical to the oracle for any input; only the cost depends on the data.
#include "qmc_internal.h"
#include "qmc_f32c.cuh"

namespace qmc {

namespace {

constexpr float kGuard = 0x1p-9f;                      // bins; 5x the fp32 error bound at nbins = 512
constexpr int kMaxFilteredBins = 512;
constexpr int kQueue = 160;                            // entries per warp: 31 left over + 4 x 32 new ones

__device__ __forceinline__ double image_component(double a, double b, double L, double h)
{
    const double t = __dadd_rn(a, -b);
    const double n = t > h ? L : (t < -h ? -L : 0.0);       // L * rint(t / L), exact
    return __dadd_rn(t, -n);
}

// the specified arithmetic: bin of the pair, or -1 beyond the cutoff
__device__ __forceinline__ int exact_bin(double xi, double yi, double zi, double xj, double yj, double zj,
                                         double L, double h, double inv_dr, int nbins)
{
    const double dx = image_component(xi, xj, L, h);
    const double dy = image_component(yi, yj, L, h);
    const double dz = image_component(zi, zj, L, h);
    const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    const double r = __dsqrt_rn(r2);
    if (!(r < h)) return -1;
    const int b = __double2int_rz(__dmul_rn(r, inv_dr));
    return b >= nbins ? nbins - 1 : b;
}

// Angstrom coordinate of particle j as the specification sees it
template <typename Real> struct ExactCoord;
template <> struct ExactCoord<double> {     // FP64: the stored coordinates, re-read from global memory (L2) by the few pairs that need them
    const double *g;
    int ld;
    __device__ __forceinline__ void get(int j, const int32_t *, const int32_t *, const int32_t *, double, double &a, double &b, double &c) const
    { a = g[j]; b = g[ld + j]; c = g[2 * ld + j]; }
};
template <> struct ExactCoord<float> {      // FP32C: s in [1,2) -> (s - 1) L, as qmc_get_positions; s is the fixed-point word
    __device__ __forceinline__ void get(int j, const int32_t *fx, const int32_t *fy, const int32_t *fz, double L, double &a, double &b, double &c) const
    {
        a = __dmul_rn(__dadd_rn((double)dec_coord(fx[j]), -1.0), L);
        b = __dmul_rn(__dadd_rn((double)dec_coord(fy[j]), -1.0), L);
        c = __dmul_rn(__dadd_rn((double)dec_coord(fz[j]), -1.0), L);
    }
};

// x / L in [0, 1] -> 32-bit fixed point (wraps: 1 -> 0, the same point of the periodic box)
__device__ __forceinline__ int32_t fix_coord(double x, double invL)
{
    return (int32_t)(uint32_t)(unsigned long long)__double2ll_rn(x * invL * 4294967296.0);
}

struct HistCtx {
    uint32_t Hs;                    // shared-window byte address of the bins, biased (see hist_pair)
    uint32_t *H, *Q;                // bins; this warp's queue of pairs for the specified arithmetic (i << 16 | j)
    int cnt;                        // entries in the queue (warp-uniform)
    float uscale, lo_off, hi_off;
    int in_limit;
};

// Two pairs per lane (particles j, j + 1: the same two j for all lanes) in packed fp32; kMask: some lanes hold no
// valid pair.  A pair that is clear of every bin edge and of the cutoff is counted at once (predicated shared-memory
// reduction: a branch around atomicAdd costs BSSY / BRA / BSYNC per pair; Hs = shared-window address of bin 0 minus
// 4 x 0x4B400000); slow = true: the pair needs the specified arithmetic.
// floor(v) is read from the low bits of fl((v - 1/2) + 1.5 x 2^23).  The constant is 1.5 x 2^23 and not 2^23 because
// v - 1/2 is NEGATIVE for v < 1/2: 2^23 plus a negative number falls into the binade below 2^23, where the fp32 spacing
// is 1/2, and reads as bin -1 (round 2 did that for every pair closer than a quarter bin).  Around 1.5 x 2^23 the
// spacing is 1 on both sides: u - guard - 1/2 < -1/2 rounds to -1 and u + guard - 1/2 to 0, so a pair with u < guard
// (r = 0 included) differs in the two estimates and takes the specified arithmetic like any pair next to a bin edge.
template <bool kMask>
__device__ __forceinline__ void hist_pair2(const HistCtx &C, int32_t xi, int32_t yi, int32_t zi, int32_t X0, int32_t X1,
                                           int32_t Y0, int32_t Y1, int32_t Z0, int32_t Z1, bool valid0, bool valid1,
                                           bool &slow0, bool &slow1)
{
    const f32x2 mx = pk2(__int2float_rn(wsub(xi, X0)), __int2float_rn(wsub(xi, X1)));
    const f32x2 my = pk2(__int2float_rn(wsub(yi, Y0)), __int2float_rn(wsub(yi, Y1)));
    const f32x2 mz = pk2(__int2float_rn(wsub(zi, Z0)), __int2float_rn(wsub(zi, Z1)));
    const f32x2 r2 = fma2(mx, mx, fma2(my, my, mul2(mz, mz)));
    float ra, rb;
    upk2(r2, ra, rb);
    asm("sqrt.approx.ftz.f32 %0, %0;" : "+f"(ra));
    asm("sqrt.approx.ftz.f32 %0, %0;" : "+f"(rb));
    const f32x2 rr = pk2(ra, rb), us = pk1(C.uscale), magic = pk1(12582912.0f);
    float l0, l1, h0, h1;
    upk2(add2(fma2(rr, us, pk1(C.lo_off)), magic), l0, l1);           // 1.5 x 2^23 + floor(u - guard), both pairs
    upk2(add2(fma2(rr, us, pk1(C.hi_off)), magic), h0, h1);           // 1.5 x 2^23 + floor(u + guard)
    const int a0 = __float_as_int(l0), a1 = __float_as_int(l1), b0 = __float_as_int(h0), b1 = __float_as_int(h1);
    slow0 = a0 != b0;
    slow1 = a1 != b1;
    if (kMask) { slow0 = slow0 && valid0; slow1 = slow1 && valid1; }
    const bool c0 = kMask ? (valid0 && !slow0 && b0 < C.in_limit) : (!slow0 && b0 < C.in_limit);
    const bool c1 = kMask ? (valid1 && !slow1 && b1 < C.in_limit) : (!slow1 && b1 < C.in_limit);
    asm volatile("{ .reg .pred p; setp.ne.s32 p, %2, 0; @p red.shared.add.u32 [%0], %1; }"
                 :: "r"(C.Hs + 4u * (uint32_t)b0), "r"(1u), "r"((int)c0) : "memory");
    asm volatile("{ .reg .pred p; setp.ne.s32 p, %2, 0; @p red.shared.add.u32 [%0], %1; }"
                 :: "r"(C.Hs + 4u * (uint32_t)b1), "r"(1u), "r"((int)c1) : "memory");
}
__device__ __forceinline__ void hist_enqueue(HistCtx &C, bool slow, int i, int j, int lane)
{
    const uint32_t m = __ballot_sync(0xffffffffu, slow);
    if (slow) C.Q[C.cnt + __popc(m & ((1u << lane) - 1u))] = ((uint32_t)i << 16) | (uint32_t)j;
    C.cnt += __popc(m);
}

template <typename Real, bool kFilter>
__global__ void __launch_bounds__(256, 4) pair_histogram_kernel(StateView sv, int nbins, uint32_t *__restrict__ hist)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr bool kF32 = sizeof(Real) == 4;
    const int N = sv.N, ld = sv.ld, w = blockIdx.x, tid = threadIdx.x, T = blockDim.x;
    const int lane = tid & 31, warp = tid >> 5, nwarps = T >> 5;
    const int nblk = (N + 31) >> 5, NP = nblk << 5;
    int32_t *fx = reinterpret_cast<int32_t *>(smem_raw), *fy = fx + NP, *fz = fx + 2 * NP;
    uint32_t *H = reinterpret_cast<uint32_t *>(fx + 3 * NP);
    uint32_t *Qall = H + nbins;                                       // [8 warps][kQueue]
    const GroupDev g = sv.groups[sv.group_of[w]];
    const double L = g.L_A, h = 0.5 * L;
    const Real *gpos = reinterpret_cast<const Real *>(sv.pos) + (size_t)w * 3 * ld;
    for (int j = tid; j < NP; j += T) {
        int32_t a = 0, b = 0, c = 0;
        if (j < N) {
            if constexpr (kF32) {
                a = enc_coord((float)gpos[j]); b = enc_coord((float)gpos[ld + j]); c = enc_coord((float)gpos[2 * ld + j]);
            } else {
                const double invL = 1.0 / L;
                a = fix_coord((double)gpos[j], invL); b = fix_coord((double)gpos[ld + j], invL); c = fix_coord((double)gpos[2 * ld + j], invL);
            }
        }
        fx[j] = a; fy[j] = b; fz[j] = c;
    }
    for (int k = tid; k < nbins; k += T) H[k] = 0u;
    __syncthreads();

    ExactCoord<Real> EC;
    if constexpr (!kF32) { EC.g = reinterpret_cast<const double *>(gpos); EC.ld = ld; }
    const double inv_dr = __ddiv_rn((double)nbins, h);
    HistCtx C;
    C.H = H; C.Q = Qall + warp * kQueue; C.cnt = 0;
    C.Hs = (uint32_t)__cvta_generic_to_shared(H) - 4u * 0x4B400000u;
    C.uscale = (float)nbins * 0x1p-31f;                               // u = (r / L) 2 nbins, r / L arrives times 2^32
    // floor(v) for -1/2 <= v < 2^22 not within rounding of an integer: the low bits of fl((v - 1/2) + 1.5 x 2^23)
    C.lo_off = -(0.5f + kGuard); C.hi_off = -(0.5f - kGuard);
    C.in_limit = 0x4B400000 + nbins;                                  // bit pattern of 1.5 x 2^23 + nbins
    // pairs that need the specified arithmetic wait in the warp's queue and are evaluated 32 at a time, one per
    // lane: the fp64 code never runs with a few lanes of a warp only
    auto drain = [&](int first, int n) {                              // entries [first, first + n), n <= 32
        __syncwarp();
        if (lane < n) {
            const uint32_t e = C.Q[first + lane];
            const int a = (int)(e >> 16), c = (int)(e & 0xFFFFu);
            double ax, ay, az, bx, by, bz;
            EC.get(a, fx, fy, fz, L, ax, ay, az);
            EC.get(c, fx, fy, fz, L, bx, by, bz);
            const int bb = exact_bin(ax, ay, az, bx, by, bz, L, h, inv_dr, nbins);
            if (bb >= 0) atomicAdd(&H[bb], 1u);
        }
        __syncwarp();
    };

    const int K = (nblk - 1) >> 1;
    const bool even = (nblk & 1) == 0, ragged = (N & 31) != 0;
    int k = warp / nblk, A = warp - k * nblk;                         // task t = warp, warp + nwarps, ...: k = t / n, A = t mod n
#pragma unroll 1
    for (;;) {
        if (k > K && !(even && k == K + 1 && A < (nblk >> 1))) break;   // even n: the offset n/2 once per block pair
        const int i = (A << 5) + lane;
        const int32_t xi = fx[i], yi = fy[i], zi = fz[i];
        int B = A + k;
        if (B >= nblk) B -= nblk;
        const int jb = B << 5;
        const bool masked = (k == 0) || (ragged && (A == nblk - 1 || B == nblk - 1));
#pragma unroll 2
        for (int jj = 0; jj < 32; jj += 4) {
            const int4 X = *reinterpret_cast<const int4 *>(fx + jb + jj);
            const int4 Y = *reinterpret_cast<const int4 *>(fy + jb + jj);
            const int4 Z = *reinterpret_cast<const int4 *>(fz + jb + jj);
            const int j = jb + jj;
            bool s0, s1, s2, s3;
            if (!kFilter) {
                const bool vi = i < N;
                s0 = vi && j < N && (k != 0 || j > i);
                s1 = vi && j + 1 < N && (k != 0 || j + 1 > i);
                s2 = vi && j + 2 < N && (k != 0 || j + 2 > i);
                s3 = vi && j + 3 < N && (k != 0 || j + 3 > i);
            } else if (masked) {
                const bool vi = i < N;
                hist_pair2<true>(C, xi, yi, zi, X.x, X.y, Y.x, Y.y, Z.x, Z.y, vi && j < N && (k != 0 || j > i),
                                 vi && j + 1 < N && (k != 0 || j + 1 > i), s0, s1);
                hist_pair2<true>(C, xi, yi, zi, X.z, X.w, Y.z, Y.w, Z.z, Z.w, vi && j + 2 < N && (k != 0 || j + 2 > i),
                                 vi && j + 3 < N && (k != 0 || j + 3 > i), s2, s3);
            } else {
                hist_pair2<false>(C, xi, yi, zi, X.x, X.y, Y.x, Y.y, Z.x, Z.y, true, true, s0, s1);
                hist_pair2<false>(C, xi, yi, zi, X.z, X.w, Y.z, Y.w, Z.z, Z.w, true, true, s2, s3);
            }
            if (__any_sync(0xffffffffu, s0 || s1 || s2 || s3)) {     // one vote per four pairs on the common path
                hist_enqueue(C, s0, i, j, lane);
                hist_enqueue(C, s1, i, j + 1, lane);
                hist_enqueue(C, s2, i, j + 2, lane);
                hist_enqueue(C, s3, i, j + 3, lane);
            }
            while (C.cnt >= 32) { C.cnt -= 32; drain(C.cnt, 32); }     // the queue holds 31 + 4 x 32 entries at most
        }
        A += nwarps;
        while (A >= nblk) { A -= nblk; ++k; }
    }
    drain(0, C.cnt);
    __syncthreads();
    for (int kk = tid; kk < nbins; kk += T) hist[(size_t)w * nbins + kk] = H[kk];
}

}  // namespace

template <typename Real, bool kFilter>
static cudaError_t launch_hist(qmc_ctx *c, int nbins, uint32_t *d_hist, int smem)
{
    auto k = pair_histogram_kernel<Real, kFilter>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    k<<<c->W, 256, smem, c->stream>>>(c->sv, nbins, d_hist);
    return cudaGetLastError();
}

// bytes of shared memory: fixed-point coordinates (padded to blocks of 32), the bins, the warps' queues
static long long hist_smem(int N, int nbins)
{
    const long long NP = ((long long)(N + 31) >> 5) << 5;
    return ((3 * NP + nbins + 8 * kQueue) * 4 + 15) & ~15LL;
}

bool pair_histogram_fits(int N, int nbins, int /*mode*/) { return N <= 65535 && hist_smem(N, nbins) <= 227 * 1024; }

cudaError_t launch_pair_histogram(qmc_ctx *c, int nbins, uint32_t *d_hist)
{
    c->launches += 1;
    const bool filter = nbins <= kMaxFilteredBins;      // the guard band is sized for that many bins
    const int smem = (int)hist_smem(c->p.N, nbins);
    if (c->p.mode == QMC_FP64) return filter ? launch_hist<double, true>(c, nbins, d_hist, smem) : launch_hist<double, false>(c, nbins, d_hist, smem);
    return filter ? launch_hist<float, true>(c, nbins, d_hist, smem) : launch_hist<float, false>(c, nbins, d_hist, smem);
}

}  // namespace qmc
