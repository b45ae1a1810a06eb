// qmc_energy_f64.cu -- FP64 local-energy estimator over all pairs and the
// from-scratch rebuild of the running pair sums S_i (R17), every UNORDERED pair evaluated once.
//
// The fp64 pipe is what bounds this mode (64 lanes per SM, every DFMA/DADD/DMUL two issue cycles), so the
// kernel spends shuffles, shared-memory traffic and integer work -- all on other pipes -- to halve the
// fp64 work: the particles are cut into blocks of 32, a warp takes a pair of blocks (A, B), lane l holds
// particle i = 32A + l AND the accumulators of particle j = 32B + l, and in step s lane l evaluates the pair
// (i_l, j_{(l+s) mod 32}).  The i-side sums stay in the lane's registers; the j-side terms travel by one
// indexed shuffle to the lane that holds j.  Block pairs are visited along a ring, B = A + k mod n,
// k = 1 .. (n-1)/2 (+ half of k = n/2 for even n), the diagonal block with steps 1..16: each pair once.
// Block ownership is static and the warps step through k together, so the per-block sums are merged by plain
// shared-memory read-modify-writes in a fixed order: results are reproducible to the bit.
//
//   G_i      = sum_{j != i} u'(r_ij) d_ij / r_ij,     u'/r = 5/2 b^5 (y^7 - z^6 y)
//   Lambda_i = sum_{j != i} [u'' + 2 u'/r]                 = -5 b^5 (2 y^7 + 3 z^7 + z^6 y)
//   V        = sum_{i<j, r<h} V_Aziz(r_ij)                 (HFD-B(HE), truncated at h, R3)
//   T_PB = -Dk sum_i (Lambda_i + |G_i|^2),  T_JF = -Dk/2 sum_i Lambda_i,  E_PB = V + T_PB      (R14)
// with y = 1/r, z = 1/(L-r).
//
// Cutoff: r^2 is clamped to h^2 for the arithmetic (nothing overflows) and the four pair terms of a pair
// beyond the cutoff, of a padding slot, or of the inactive half of the last diagonal step are selected to
// exactly 0 -- comparison (on the bit patterns, less_pos) and selects on the integer pipe.
// The two exponentials of HFD-B(HE) are kept out of the pair loop where that pays (kPend, below).
#include "qmc_internal.h"

namespace qmc {

namespace {

constexpr int kMaxOwn64 = 20;                        // i-blocks one warp can own (planner: ceil(nblk / nwarps) <= kMaxOwn64)

struct Const64 {
    double L, h, h2, sh;
    double eps, inv_rm, rm2, A, alpha, beta, c6, c8, c10, D, Drm;
    __device__ __forceinline__ void load(const GroupDev &g)
    {
        L = g.L; h = g.h; h2 = g.h2; sh = g.sh;
        const AzizDev &a = g.az;
        eps = a.eps; inv_rm = a.inv_rm; rm2 = a.rm2; A = a.A; alpha = a.alpha; beta = a.beta;
        c6 = a.c6; c8 = a.c8; c10 = a.c10; D = a.D; Drm = a.Drm;
    }
};

// signed minimum-image component for |a - b| <= L: magnitude by the fold h - |h - |d||, sign = sign(d)
// flipped when |d| > h (two integer operations on the high word)
__device__ __forceinline__ double min_image(double a, double b, double h)
{
    const double d = a - b;
    const double f = h - fabs(d);
    const double m = h - fabs(f);
    const int hi = __double2hiint(m) | ((__double2hiint(d) ^ __double2hiint(f)) & 0x80000000);
    return __hiloint2double(hi, __double2loint(m));
}

// exp(a) for a <= 0 in fp64: a = n ln2 + r, |r| <= ln2/2, Taylor polynomial of degree 12 (remainder
// < 2e-16 relative), 2^n through the exponent field; results below 2^-1022 come out as ~1e-308 instead
// of a subnormal (they multiply a term that is then < 1e-300 K).  The coefficients sit in constant
// memory so that every DFMA reads its coefficient as an operand (CUDA's exp() rebuilds its 64-bit
// immediates with two uniform moves each inside the pair loop: 22 issue slots per pair).
__constant__ double kExpC[13] = {
    1.0, 1.0, 1.0 / 2, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320, 1.0 / 362880,
    1.0 / 3628800, 1.0 / 39916800, 1.0 / 479001600};
__device__ __forceinline__ double exp_neg(double a)
{
    const double magic = 6755399441055744.0;                       // 2^52 + 2^51
    const double t = fma(a, 1.4426950408889634, magic);
    const double n = t - magic;
    double r = fma(n, -6.93147180369123816490e-01, a);
    r = fma(n, -1.90821492927058770002e-10, r);
    double p = kExpC[12];
#pragma unroll
    for (int k = 11; k >= 0; --k) p = fma(p, r, kExpC[k]);
    const int e = max(__double2loint(t), -1022);
    return __hiloint2double(__double2hiint(p) + (e << 20), __double2loint(p));
}

// HFD-B(HE) in two parts.  Every pair inside the cutoff adds its dispersion sum with F = 1 in straight-line code.
// The two exponentials -- the repulsive term A exp(-alpha x + beta x^2), below 3e-15 of the dispersion term for
// x = r/r_m >= 3 (8.9 A, i.e. for 97 % of the pairs inside the cutoff), and the damping F(x) - 1, which is 0 for
// x >= D -- cost 19 fp64 instructions each in a dependent chain.  A pair with x < 3 (compared on the high word: kRepHi)
// parks (x, D/x - 1, dispersion) in a per-lane pending slot; the exponentials are evaluated for all lanes that hold
// an entry only when some lane is about to park a second one (about every 8th step), and once at the end.  Which
// pairs are evaluated together depends on the data alone: reproducible.  This also leaves the pair arithmetic free
// of branches, so that two pairs per lane are in flight (the kernel waits on fp64 latencies, not on the pipe).
constexpr int kRepHi = 0x40080000;                   // high word of 3.0

struct Pending64 {
    double x = 3.0, q = 0.0, disp = 0.0, rep = 0.0, corr = 0.0;     // rep: sum of exp(..); corr: sum of (1 - F) disp
    bool full = false;
};

struct Pair64 { double mx, my, mz, t, gm, lt, v, x, q, disp; bool in; };   // v = -dispersion sum: F = 1, no repulsive term (Pending64)

// all terms of one pair; bias > 0 pushes the pair beyond the cutoff
template <bool kEnergy, int kPend>
__device__ __forceinline__ Pair64 pair64(double xi, double yi, double zi, double xs, double ys, double zs,
                                         double bias, const Const64 &C)
{
    Pair64 p;
    p.mx = min_image(xi, xs, C.h);
    p.my = min_image(yi, ys, C.h);
    p.mz = min_image(zi, zs, C.h);
    const double r2 = fma(p.mz, p.mz, fma(p.my, p.my, fma(p.mx, p.mx, bias)));
    p.in = less_pos(r2, C.h2);
    const double r2c = p.in ? r2 : C.h2;
    const double y = rsqrt_pos(r2c);
    const double r = r2c * y;
    const double z = rcp_pos(C.L - r);
    const double y2 = y * y, z2 = z * z;
    const double y4 = y2 * y2, z4 = z2 * z2;
    const double t = fma(z4, z, fma(y4, y, -C.sh));
    p.t = p.in ? t : 0.0;
    p.gm = 0.0; p.lt = 0.0; p.v = 0.0; p.x = 0.0; p.q = 0.0; p.disp = 0.0;
    if (kEnergy) {
        const double y6 = y4 * y2, z6 = z4 * z2;
        const double y7 = y6 * y, z6y = z6 * y, z7 = z6 * z;
        p.gm = p.in ? y7 - z6y : 0.0;
        p.lt = p.in ? fma(2.0, y7, fma(3.0, z7, z6y)) : 0.0;
        const double x = r * C.inv_rm;
        const double w = C.rm2 * y2;                                // 1/x^2
        const double disp = w * w * w * fma(w, fma(w, C.c10, C.c8), C.c6);
        if (kPend != 0) {
            p.x = x;
            p.q = fma(C.Drm, y, -1.0);                              // D/x - 1
            p.disp = disp;
            p.v = p.in ? -disp : 0.0;
        } else {                                                    // small boxes: most pairs are near, evaluate in place
            double F = 1.0;
            if (__any_sync(0xffffffffu, x < C.D)) {
                const double q = fma(C.Drm, y, -1.0);
                const double e = exp_neg(-q * q);
                F = x < C.D ? e : 1.0;
            }
            const double rep = C.A * exp_neg(x * fma(C.beta, x, -C.alpha));
            p.v = p.in ? fma(-F, disp, rep) : 0.0;
        }
    }
    return p;
}

__device__ __forceinline__ double shfl_from(double v, int src)
{
    return __hiloint2double(__shfl_sync(0xffffffffu, __double2hiint(v), src), __shfl_sync(0xffffffffu, __double2loint(v), src));
}

// evaluate the exponentials of every lane's pending entry (warp-uniform call)
__device__ __forceinline__ void pending_flush(Pending64 &Q, const Const64 &C)
{
    const double e = exp_neg(Q.x * fma(C.beta, Q.x, -C.alpha));
    Q.rep += Q.full ? e : 0.0;
    const bool damped = Q.full && Q.x < C.D;
    if (__any_sync(0xffffffffu, damped)) {
        const double F = exp_neg(-Q.q * Q.q);
        Q.corr += damped ? (1.0 - F) * Q.disp : 0.0;
    }
    Q.full = false;
}
__device__ __forceinline__ void pending_park(Pending64 &Q, const Pair64 &p, const Const64 &C)
{
    const bool hit = p.in && __double2hiint(p.x) < kRepHi;
    if (__any_sync(0xffffffffu, hit && Q.full)) pending_flush(Q, C);
    if (hit) { Q.x = p.x; Q.q = p.q; Q.disp = p.disp; Q.full = true; }
}

// kPend = 2, boxes small enough that a lane's pending slot would be evaluated almost every step (N = 512: 12.5 % of
// the pairs have x < 3) and with room in shared memory: the warp COMPACTS such pairs into a queue of (x, dispersion)
// and evaluates the exponentials 32 entries at a time, one per lane, so that their cost is paid once per near pair
// instead of once per warp step.  The queue holds at most 31 + 64 entries.
constexpr int kQueue64 = 96;
struct Queue64 {
    double *x, *d;
    int cnt = 0;
    double rep = 0.0, corr = 0.0;                    // sum of exp(..); sum of (1 - F) disp
};
__device__ __forceinline__ void queue_drain(Queue64 &Q, const Const64 &C, int first, int n, int lane)
{
    __syncwarp();
    const bool act = lane < n;
    const double x = act ? Q.x[first + lane] : 3.0;
    const double e = exp_neg(x * fma(C.beta, x, -C.alpha));
    Q.rep += act ? e : 0.0;
    const bool damped = act && x < C.D;
    if (__any_sync(0xffffffffu, damped)) {
        const double d = act ? Q.d[first + lane] : 0.0;
        double z;                                    // 1/x to third order
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(z) : "d"(x));
        const double e1 = fma(-x, z, 1.0);
        z = fma(z, fma(e1, e1, e1), z);
        const double q = fma(C.D, z, -1.0);          // D/x - 1
        const double F = exp_neg(-q * q);
        Q.corr += damped ? (1.0 - F) * d : 0.0;
    }
    __syncwarp();
}
__device__ __forceinline__ void queue_push(Queue64 &Q, const Pair64 &p, int lane)
{
    const bool hit = p.in && __double2hiint(p.x) < kRepHi;
    const unsigned m = __ballot_sync(0xffffffffu, hit);
    if (m != 0u) {
        if (hit) {
            const int pos = Q.cnt + __popc(m & ((1u << lane) - 1u));
            Q.x[pos] = p.x;
            Q.d[pos] = p.disp;
        }
        Q.cnt += __popc(m);
    }
}

template <int T, bool kEnergy, int kPend>
__global__ void __launch_bounds__(T, (T <= 128 ? 4 : (T <= 256 ? 2 : 1)))
energy64_kernel(StateView sv, double Dk, double *__restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = sv.N, ld = sv.ld;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int nwarps = T >> 5;
    const int w = blockIdx.x;
    const int nblk = (N + 31) >> 5, NP = nblk << 5;

    double *red = reinterpret_cast<double *>(smem_raw);               // [3][32]
    double *x   = red + 98;                                           // [3][NP]
    double *y = x + NP, *z = x + 2 * NP;
    double *ag = x + 3 * NP;                                          // [4][NP]: G_x, G_y, G_z, S (raw units)

    const GroupDev g = sv.groups[sv.group_of[w]];
    Const64 C;
    C.load(g);

    const double *gpos = reinterpret_cast<const double *>(sv.pos) + (size_t)w * 3 * ld;
    for (int j = tid; j < NP; j += T) {
        const bool in = j < N;
        x[j] = in ? gpos[j] : 0.0;
        y[j] = in ? gpos[ld + j] : 0.0;
        z[j] = in ? gpos[2 * ld + j] : 0.0;
        ag[j] = 0.0; ag[NP + j] = 0.0; ag[2 * NP + j] = 0.0; ag[3 * NP + j] = 0.0;
    }
    __syncthreads();

    const double kBig = 4.0 * C.L * C.L;                              // > any r^2: forces the clamp

    // Schedule (deterministic: the same sums in the same order on every run): warp v owns the i-blocks
    // A = v, v + nwarps, ...; all warps go through the ring offsets k = 0, 1, ... together, one barrier per offset.
    // Within one offset the j-blocks B = A + k mod n of different A are different, so the j-side sums are added
    // to shared memory by plain read-modify-writes of the one warp that holds them, in the order of k; the i-side
    // sums of a warp's own blocks wait in (local-memory) accumulators and are added after the last offset.
    const int K = (nblk - 1) >> 1;                                    // full ring offsets
    const bool even = (nblk & 1) == 0;
    double tLam = 0.0, tV = 0.0;
    Pending64 Q;
    Queue64 W;
    if (kPend == 2) { W.x = ag + 4 * NP + warp * (2 * kQueue64); W.d = W.x + kQueue64; }
    double own[kMaxOwn64][4];                                         // G_x, G_y, G_z, S of this lane's particle in each own block
#pragma unroll 1
    for (int a = 0; a < kMaxOwn64; ++a) { own[a][0] = 0.0; own[a][1] = 0.0; own[a][2] = 0.0; own[a][3] = 0.0; }
    const int kend = K + (even ? 1 : 0);
#pragma unroll 1
    for (int k = 0; k <= kend; ++k) {
        int a = 0;
#pragma unroll 1
        for (int A = warp; A < nblk; A += nwarps, ++a) {
            if (k > K && A >= (nblk >> 1)) break;                    // even n: the offset n/2 once per block pair
            const int i = (A << 5) + lane;
            const bool vi = i < N;
            const double xi = x[i], yi = y[i], zi = z[i];
            double gxi = 0.0, gyi = 0.0, gzi = 0.0, si = 0.0;
            int B = A + k;
            if (B >= nblk) B -= nblk;
            const int jb = B << 5;
            const bool vj = jb + lane < N;
            double gxj = 0.0, gyj = 0.0, gzj = 0.0, sj = 0.0;
            const int s0 = (k == 0) ? 1 : 0, s1 = (k == 0) ? 17 : 32;
            if (kPend != 0) {
#pragma unroll 1
                for (int s = s0; s < s1; s += 2) {                        // two pairs per lane in flight (s1 - s0 is even)
                    const int srcA = (lane + s) & 31, srcB = (lane + s + 1) & 31;
                    const bool okA = vi && (jb + srcA < N);
                    const bool okB = vi && (jb + srcB < N) && !(k == 0 && s + 1 == 16 && lane >= 16);
                    const Pair64 pA = pair64<kEnergy, kPend>(xi, yi, zi, x[jb + srcA], y[jb + srcA], z[jb + srcA], okA ? 0.0 : kBig, C);
                    const Pair64 pB = pair64<kEnergy, kPend>(xi, yi, zi, x[jb + srcB], y[jb + srcB], z[jb + srcB], okB ? 0.0 : kBig, C);
                    si += pA.t;
                    si += pB.t;
                    // the lane that holds j = src gets this pair's terms: lane m receives from lane m - s
                    const int fromA = lane - s, fromB = lane - s - 1;     // shfl takes the source lane modulo 32
                    sj += shfl_from(pA.t, fromA);
                    sj += shfl_from(pB.t, fromB);
                    if (kEnergy) {
                        const double ax = pA.gm * pA.mx, ay = pA.gm * pA.my, az = pA.gm * pA.mz;
                        const double bx = pB.gm * pB.mx, by = pB.gm * pB.my, bz = pB.gm * pB.mz;
                        gxi += ax; gyi += ay; gzi += az;
                        gxi += bx; gyi += by; gzi += bz;
                        tLam += pA.lt; tLam += pB.lt;
                        tV += pA.v; tV += pB.v;
                        gxj -= shfl_from(ax, fromA); gyj -= shfl_from(ay, fromA); gzj -= shfl_from(az, fromA);
                        gxj -= shfl_from(bx, fromB); gyj -= shfl_from(by, fromB); gzj -= shfl_from(bz, fromB);
                        if (kPend == 1) { pending_park(Q, pA, C); pending_park(Q, pB, C); }
                        if (kPend == 2) {
                            queue_push(W, pA, lane);
                            queue_push(W, pB, lane);
                            while (W.cnt >= 32) { W.cnt -= 32; queue_drain(W, C, W.cnt, 32, lane); }
                        }
                    }
                }
            } else {
#pragma unroll 1
                for (int s = s0; s < s1; ++s) {                       // one pair per lane and step
                    const int src = (lane + s) & 31;
                    const bool ok = vi && (jb + src < N) && !(k == 0 && s == 16 && lane >= 16);
                    const Pair64 p = pair64<kEnergy, 0>(xi, yi, zi, x[jb + src], y[jb + src], z[jb + src], ok ? 0.0 : kBig, C);
                    si += p.t;
                    double cx = 0.0, cy = 0.0, cz = 0.0;
                    if (kEnergy) {
                        cx = p.gm * p.mx; cy = p.gm * p.my; cz = p.gm * p.mz;
                        gxi += cx; gyi += cy; gzi += cz;
                        tLam += p.lt;
                        tV += p.v;
                    }
                    const int from = lane - s;                        // lane m receives from lane m - s (modulo 32)
                    sj += shfl_from(p.t, from);
                    if (kEnergy) {
                        gxj -= shfl_from(cx, from);
                        gyj -= shfl_from(cy, from);
                        gzj -= shfl_from(cz, from);
                    }
                }
            }
            if (vj) {
                ag[3 * NP + jb + lane] += sj;
                if (kEnergy) {
                    ag[jb + lane] += gxj;
                    ag[NP + jb + lane] += gyj;
                    ag[2 * NP + jb + lane] += gzj;
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
        if (kPend == 1) { pending_flush(Q, C); tV = fma(C.A, Q.rep, tV) + Q.corr; }
        if (kPend == 2) { queue_drain(W, C, 0, W.cnt, lane); tV = fma(C.A, W.rep, tV) + W.corr; }
        tV *= C.eps;
        // each unordered pair was seen once: the Laplacian sum over i counts it twice
        tLam *= 2.0;
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
                const double lam = -5.0 * g.b5 * a;                            // sum_i Lambda_i
                const double g2 = (2.5 * g.b5) * (2.5 * g.b5) * b;             // sum_i |G_i|^2
                const double T_PB = -Dku * (lam + g2);
                const double T_JF = -0.5 * Dku * lam;
                double *o = out + (size_t)w * 4;
                o[0] = c + T_PB; o[1] = c; o[2] = T_PB; o[3] = T_JF;
            }
        }
    }
}

int smem_bytes64(int N) { return 98 * 8 + 7 * (((N + 31) >> 5) << 5) * 8; }

template <int T, bool kEnergy, int kPend>
cudaError_t launch64k(qmc_ctx *c, double *d_out, int smem)
{
    auto k = energy64_kernel<T, kEnergy, kPend>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    k<<<c->W, T, smem, c->stream>>>(c->sv, c->p.hbar2_over_2m, d_out);
    return cudaGetLastError();
}

// fraction of the particles inside the sphere x < 3 around a particle (the pairs that need the exponentials)
double near_pair_fraction(const qmc_ctx *c)
{
    double Lmin = c->box_L[0];
    for (double L : c->box_L) Lmin = L < Lmin ? L : Lmin;
    const double r = 3.0 * c->p.aziz[1];                 // r_m, Angstrom like box_L
    return 4.18879 * r * r * r / (Lmin * Lmin * Lmin);
}

// The pending-slot and queue forms (kPend 1, 2) leave the repulsive term and the damping out for x >= 3.  That is a
// property of the CONSTANTS: with HFD-B(HE)'s the repulsive term is below 3e-15 of the dispersion sum there and
// F = 1 beyond D = 1.4; qmc_params.aziz is the caller's, so the assumption is checked for the numbers supplied
// (ADVICE r2): D <= 3, and A exp(-alpha x + beta x^2) below 1e-14 of |c6/x^6 + c8/x^8 + c10/x^10| at 65 points from
// x = 3 to the cutoff of the largest box.  Anything else (a softer repulsion, a wider damping, no dispersion at all)
// takes the in-place evaluation of both exponentials for every pair (kPend 0).
bool far_terms_negligible(const qmc_ctx *c)
{
    const double *a = c->p.aziz;                         // eps, r_m, A, alpha, beta, c6, c8, c10, D
    if (!(a[8] <= 3.0)) return false;
    double Lmax = 0.0;
    for (double L : c->box_L) Lmax = L > Lmax ? L : Lmax;
    const double x_hi = fmax(3.0, 0.5 * Lmax / a[1]);
    for (int k = 0; k <= 64; ++k) {
        const double x = 3.0 + (x_hi - 3.0) * (double)k / 64.0;
        const double w = 1.0 / (x * x);
        const double disp = fabs(w * w * w * (a[5] + w * (a[6] + w * a[7])));
        const double rep = fabs(a[2]) * exp(x * (a[4] * x - a[3]));
        if (!(rep <= 1e-14 * disp)) return false;
    }
    return true;
}

// How the exponentials are evaluated: 1 (per-lane pending slot) while few pairs are near (N = 1952 at liquid density:
// 3.3 %); 2 (warp queue) for smaller boxes if two CTAs with their queues still fit an SM (N = 512: 12.5 %, N = 256:
// 25 %); 0 (in place) when most pairs are near anyway (N = 64).
template <int T>
cudaError_t launch64(qmc_ctx *c, double *d_out, bool energy)
{
    const int smem = smem_bytes64(c->p.N);
    if (!energy) return launch64k<T, false, 0>(c, d_out, smem);
    if (!far_terms_negligible(c)) return launch64k<T, true, 0>(c, d_out, smem);
    const double f = near_pair_fraction(c);
    const int qbytes = (T >> 5) * 2 * kQueue64 * 8;
    if (f < 0.05) return launch64k<T, true, 1>(c, d_out, smem);
    if (f < 0.5 && 2 * (smem + qbytes + 1024) <= 228 * 1024) return launch64k<T, true, 2>(c, d_out, smem + qbytes);
    return launch64k<T, true, 0>(c, d_out, smem);
}

template <int T>
int occupancy64(int smem)
{
    int occ = 0;
    auto k = energy64_kernel<T, true, 1>;
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, T, smem);
    return occ;
}

}  // namespace

#define QMC_E64_THREADS(X) X(32) X(64) X(128) X(256) X(384) X(512)

cudaError_t launch_energy_f64(qmc_ctx *c, double *d_out, bool energy)
{
    const int T = c->energy_plan.threads;
#define X(TT) if (T == TT) return launch64<TT>(c, d_out, energy);
    QMC_E64_THREADS(X)
#undef X
    return cudaErrorInvalidValue;
}

// 1 to 8 warps;
// qmc_set_tuning("energy_threads") overrides (tuning experiments).  false: N too large for the per-particle
// accumulators in shared memory -- the caller falls back to the ordered-pair kernel of qmc_energy.cu.
bool plan_energy_f64(qmc_ctx *c, EnergyPlan *out)
{
    const int N = c->p.N;
    const int smem = smem_bytes64(N);
    if (smem > 227 * 1024) return false;
    // measured (c2, c5, c3): 128 threads up to N ~ 1000 (N = 512: 13.6 ms against 13.9 with 256), 256 above
    int T = N <= 64 ? 32 : (N <= 128 ? 64 : (N <= 1024 ? 128 : 256));
    if (c->tuning.energy_threads > 0) {
        const int v = c->tuning.energy_threads;
        if (v >= 32 && v <= 512 && ((v & (v - 1)) == 0 || v == 384)) T = v;
    }
    const int nblk = (N + 31) >> 5;
    while ((nblk + (T >> 5) - 1) / (T >> 5) > kMaxOwn64 && T < 512) T *= 2;     // own-block accumulators per warp
    if ((nblk + (T >> 5) - 1) / (T >> 5) > kMaxOwn64) return false;
    out->threads = T;
    out->smem_bytes = smem;
    out->variant = 1;
    out->ctas_per_sm = 0;
#define X(TT) if (T == TT) out->ctas_per_sm = occupancy64<TT>(smem);
    QMC_E64_THREADS(X)
#undef X
    return true;
}

}  // namespace qmc
