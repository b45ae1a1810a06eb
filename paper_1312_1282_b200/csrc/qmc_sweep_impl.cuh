// qmc_sweep_impl.cuh -- the Metropolis sweep kernel.
//
// One CTA per walker ("each thread block serves one walker").  The walker's
// coordinates (SoA) and running pair sums stay in shared memory for the whole call (l.175, l.323
// "shared memory persistence"); global memory is touched once on entry and once on exit.
//
// Pair sums are kept in RAW units: t(r) = y^5 + z^5 - sh with y = 1/r, z = 1/(L-r), sh = 2/h^5, so that
// u(r) = c1 t(r) (Eq.(8)/(9), R1) and t(h) = 0; S_i = sum_{j != i} t(r_ij); Delta = c1 (sum_j t_new - S_s).
//
// Per move (particle s, sweep t):
//   a2  variates from Philox4x32-10(counter (s,t,walker,0), key seed), prepared 32 moves at a time
//       by warp 0 (one move per lane, including log(xi)) into a double-buffered shared array;
//   a3  thread tid evaluates t(|r'_s - r_j|) for its own particles (J of them, in packs of V consecutive
//       ones read as one shared-memory vector) and keeps the values in registers;
//   a4  the old sum is the running S_s (only the thread that owns s reads it);
//   a5  xor-butterfly warp sums, one shared-memory exchange, then every thread adds the warp totals in
//       the same fixed order: every thread ends with the same bits;
//   a6  every thread takes the same decision 2*Delta > log(xi): ONE __syncthreads per move;
//   a7  on accept each thread re-evaluates the OLD terms of its own particles and updates its own
//       S_j += t_new - t_old; the owner of s commits the position and S_s.
// Ownership is static, so S and the pair loops need no synchronisation.  The pair loops carry no index
// test: the owner of s "poisons" the stored x of particle s for the duration of the move (half a box away
// from the point the distances are taken from in FP32C, NaN in FP64) so that the self term is exactly 0;
// r_s itself was read by every thread BEFORE the previous move's barrier (prefetch).
//
// FP32C (R20): a coordinate is the 23-bit grid index k of s = 1 + x/L in [1,2), held in shared memory as the
// 32-bit fixed-point number k << 9.  a - b in wrapping 32-bit integer arithmetic IS the minimum image
// (l.325), exactly; one I2FP gives it as fp32.  Everything after that is fp32 in box units.
#pragma once
#include "qmc_internal.h"
#include "qmc_f32c.cuh"

namespace qmc {

constexpr int kChunk = 32;                       // moves prepared at a time (one per lane of warp 0)

template <typename Real> struct ModeT;
template <> struct ModeT<double> { using Coord = double;  using Disp = double; };
template <> struct ModeT<float>  { using Coord = int32_t; using Disp = int32_t; };

// Displacement (coordinate units, already times step) and log(xi) of one move.
template <typename Real> struct MoveRand { double logxi; typename ModeT<Real>::Disp dx, dy, dz; int32_t s; };
// bytes of one record in the shared-memory variate ring (16-byte aligned)
template <typename Real> struct MoveSlot { static constexpr int bytes = (int)((sizeof(MoveRand<Real>) + 15) / 16 * 16); };

// V consecutive values as one shared-memory vector access.
template <typename E, int V> struct alignas(sizeof(E) * V) Pack { E v[V]; };

// ---- per-mode constants of the pair function -----------------------------------------------------
template <typename Real> struct SweepConst;
template <> struct SweepConst<double> {
    double L, h, h2, sh;
    __device__ __forceinline__ void load(const GroupDev &g) { L = g.L; h = g.h; h2 = g.h2; sh = g.sh; }
};
template <> struct SweepConst<float> {
    __device__ __forceinline__ void load(const GroupDev &) {}      // box units: L = 1, h = 1/2, sh = 64
};

// t(r) between the point (px,py,pz) and the stored particle (X,Y,Z).
// FP64: fold m = h - |h - |a-b|| per component (exact minimum image for |a-b| <= L), select on r^2 < h^2
// (R2; NaN -- poison or padding -- selects 0).
__device__ __forceinline__ double pair_t(double px, double py, double pz, double X, double Y, double Z,
                                         double /*bias*/, const SweepConst<double> &P)
{
    const double mx = P.h - fabs(P.h - fabs(px - X));
    const double my = P.h - fabs(P.h - fabs(py - Y));
    const double mz = P.h - fabs(P.h - fabs(pz - Z));
    const double r2 = fma(mz, mz, fma(my, my, mx * mx));
    const double y = rsqrt_pos(r2);
    const double z = rcp_pos(fma(-r2, y, P.L));                // L - r, r = r^2 y
    const double y2 = y * y, z2 = z * z;
    const double y4 = y2 * y2, z4 = z2 * z2;
    const double t = fma(z4, z, fma(y4, y, -P.sh));
    return r2 < P.h2 ? t : 0.0;
}
// FP32C: wrapping integer difference = minimum image * 2^32; r^2 is clamped to h^2 = 1/4, where
// y = z = 2 and t = 16*2 + (16*2 - 64) = 0 exactly, so pairs at and beyond the cutoff add exactly 0.
// bias = 0 for a real particle, 1 for a padding slot (clamps).
__device__ __forceinline__ float pair_t(int32_t px, int32_t py, int32_t pz, int32_t X, int32_t Y, int32_t Z,
                                        float bias, const SweepConst<float> &)
{
    const float mx = __int2float_rn(wsub(px, X));
    const float my = __int2float_rn(wsub(py, Y));
    const float mz = __int2float_rn(wsub(pz, Z));
    const float r2p = fmaf(mx, mx, fmaf(my, my, mz * mz));
    const float r2 = fminf(fmaf(r2p, 0x1p-64f, bias), 0.25f);
    const float y = rsqrt_pos(r2);
    const float r = r2 * y;
    const float z = rcp_pos(1.0f - r);
    const float y2 = y * y, z2 = z * z;
    const float y4 = y2 * y2, z4 = z2 * z2;
    return fmaf(z4, z, fmaf(y4, y, -64.0f));
}

// Two FP32C pair terms at once.  r^2 arrives as d^2 2^64 (integer differences); ONE integer instruction (VIADDMNMX:
// add to the exponent field, then min) rescales it by 2^-64 and clamps it: a = min(r^2, 1/4).  With a + b = 1 one has
// a^-5 + b^-5 = (1 - 5ab + 5 (ab)^2) / (ab)^5, so with r = sqrt(a), p = r (1 - r) = r - r^2 and w = 1/p
//   t = y^5 + z^5 - 64 = w^3 (w^2 - 5w + 5) - 64:
// one square root, one reciprocal and SIX packed multiply-adds (the form with y = 1/r and z = 1/(1-r) separately takes
// eight).  At the clamp r = 1/2, p = 1/4, w = 4 and t = 64 (16 - 20 + 5) - 64 = 0 exactly (MUFU.SQRT and MUFU.RCP are
// exact on powers of two; tests/test_gpu_parity.py checks the zero through the padding slots).  bias2 holds 0 or 2^63
// per lane (padding: clamps).  d = 0 (two particles on one grid point) gives a negative number, sqrt = NaN, and the
// move is rejected.  Relative error of a term ~5e-7 near contact, absolute error ~2e-5 near the cutoff (where t -> 0
// quadratically): inside the R23 budget.
constexpr double kT2Unit = 1.0;
__device__ __forceinline__ float scale_clamp_r2(float a)
{
    return __int_as_float(__viaddmin_s32(__float_as_int(a), -(64 << 23), 0x3E800000));      // min(a 2^-64, 1/4)
}
__device__ __forceinline__ float sqrt_pos(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ f32x2 pair_t2(int32_t px, int32_t py, int32_t pz, int32_t X0, int32_t X1, int32_t Y0, int32_t Y1,
                                         int32_t Z0, int32_t Z1, f32x2 bias2, int32_t zero)
{
    const f32x2 mx = pk2(__int2float_rn(wsub3(px, X0, zero)), __int2float_rn(wsub3(px, X1, zero)));
    const f32x2 my = pk2(__int2float_rn(wsub3(py, Y0, zero)), __int2float_rn(wsub3(py, Y1, zero)));
    const f32x2 mz = pk2(__int2float_rn(wsub3(pz, Z0, zero)), __int2float_rn(wsub3(pz, Z1, zero)));
    const f32x2 r2p = fma2(mx, mx, fma2(my, my, fma2(mz, mz, bias2)));
    float a, b;
    upk2(r2p, a, b);
    a = scale_clamp_r2(a);
    b = scale_clamp_r2(b);
    const f32x2 r = pk2(sqrt_pos(a), sqrt_pos(b));
    const f32x2 p = sub2(r, pk2(a, b));                                 // r - r^2 = r (1 - r)
    float pa, pb;
    upk2(p, pa, pb);
    const f32x2 w = pk2(rcp_pos(pa), rcp_pos(pb));
    const f32x2 w2 = mul2(w, w), w3 = mul2(w2, w);
    const f32x2 u = fma2(w, w, fma2(w, pk2(-5.0f, -5.0f), pk2(5.0f, 5.0f)));
    return fma2(w3, u, pk2(-64.0f, -64.0f));
}

template <typename Real> __device__ __forceinline__ typename ModeT<Real>::Coord poison_of(typename ModeT<Real>::Coord p);
template <> __device__ __forceinline__ double poison_of<double>(double) { return __longlong_as_double(0x7ff8000000000000LL); }
template <> __device__ __forceinline__ int32_t poison_of<float>(int32_t p) { return (int32_t)((uint32_t)p + 0x80000000u); }

// trial coordinate.  FP64: ONE rounding (bit-identical to the oracle).  FP32C: grid index + displacement
// rounded to the grid (a symmetric proposal on the lattice of representable positions), periodic by wrap-around.
__device__ __forceinline__ double trial_coord(double x, double d) { return __dadd_rn(x, d); }
__device__ __forceinline__ int32_t trial_coord(int32_t x, int32_t d) { return wadd(x, d); }

__device__ __forceinline__ double commit_coord(double x, double L)      // R10
{
    if (x >= L) x -= L;
    if (x < 0.0) x += L;
    return x;
}
__device__ __forceinline__ int32_t commit_coord(int32_t x, double) { return x; }

// position of particle j in the shared S array: the V doubles of a pack are stored as V/2 chunks of 16 bytes,
// chunk c of group g at ((g*(V/2) + c)*T + tid)*2, so that a warp's 16-byte accesses are contiguous.
template <int T, int V>
__device__ __forceinline__ int s_index(int j)
{
    if (V == 1) return j;
    const int gi = j / (T * V), rem = j - gi * (T * V);
    const int tid = rem / V, e = rem - tid * V;
    return ((gi * (V / 2) + (e >> 1)) * T + tid) * 2 + (e & 1);
}

static inline int sweep_smem_bytes(int T, int J, int mode, int P)
{
    const int real = (mode == QMC_FP64) ? 8 : 4;
    const int slot = (mode == QMC_FP64) ? MoveSlot<double>::bytes : MoveSlot<float>::bytes;
    const int NP = T * J;
    (void)P;                                             // hi + lo takes the room of the fp64 sums
    return NP * 8 + 2 * kChunk * slot + 64 * 8 + 3 * NP * real;
}

// Resident CTAs per SM the register allocator should leave room for: what shared memory allows for
// this (T,J), capped so that fp64 code keeps >= ~80 and fp32 code >= ~48 registers plus the J retained terms.
template <typename Real, int T, int J, int P>
constexpr int sweep_min_ctas()
{
    const int real = (int)sizeof(Real);
    const int smem = J * T * (8 + 3 * real) + 2 * kChunk * 48 + 64 * 8 + 1024;
    const int by_smem = (228 * 1024) / smem;
    const int regs = (real == 8 ? 96 + 3 * J : 40 + 3 * J);
    const int by_regs = 65536 / (regs * T);
    int n = by_smem < by_regs ? by_smem : by_regs;
    return n < 1 ? 1 : (n > 32 ? 32 : n);
}

// sum of the NW warp totals in a fixed pairwise order (same bits in every thread)
template <int NW>
__device__ __forceinline__ double sum_parts(const double *pb)
{
    double v[NW];
    if (NW >= 2) {
#pragma unroll
        for (int i = 0; i < NW; i += 2) {
            const double2 p = *reinterpret_cast<const double2 *>(pb + i);
            v[i] = p.x; v[i + 1] = p.y;
        }
    } else {
        v[0] = pb[0];
    }
#pragma unroll
    for (int st = 1; st < NW; st *= 2)
#pragma unroll
        for (int i = 0; i + st < NW; i += 2 * st) v[i] += v[i + st];
    return v[0];
}

__device__ __forceinline__ double coord_to_angstrom(double v, double) { return v; }
__device__ __forceinline__ double coord_to_angstrom(int32_t k, double L_A) { return __dmul_rn(__dadd_rn((double)dec_coord(k), -1.0), L_A); }

// coordinates + accepted-move count of this CTA's walker -> write-out slot; called by ALL threads at a sweep boundary
template <int T, typename Coord>
__device__ __forceinline__ void writeout_walker(const WriteoutView &wo, int slot, int w, int W, int N, double L_A,
                                                const Coord *x, const Coord *y, const Coord *z,
                                                unsigned long long n_acc_total)
{
    __syncthreads();                                          // the last commits of the sweep are in shared memory
    double *dst = wo.xyz + ((size_t)slot * W + w) * 3 * N;
    for (int j = threadIdx.x; j < N; j += T) {
        dst[j]         = coord_to_angstrom(x[j], L_A);
        dst[N + j]     = coord_to_angstrom(y[j], L_A);
        dst[2 * N + j] = coord_to_angstrom(z[j], L_A);
    }
    if (threadIdx.x == 0 && wo.n_acc) wo.n_acc[(size_t)slot * W + w] = n_acc_total;
    __threadfence_system();                                   // data before the flag, as seen from the host
    __syncthreads();
    if (threadIdx.x == 0) wo.flag[(size_t)slot * W + w] = 1;
}

// T threads per CTA; each thread owns J particles in G = J/V packs of V consecutive ones:
// particle j = (g*T + tid)*V + e, g < G, e < V.  Shared arrays are padded to NP = T*J entries.
// PD = 1 (FP32C, V >= 2): a running pair sum is held on chip as the unevaluated sum of two fp32 numbers
// hi + lo (the same 8 bytes per particle as an fp64 sum).  An accepted move adds its fp32 changes
// t_new - t_old to lo with packed adds; every kFold moves each thread renormalises its own sums with an
// error-free TwoSum (hi + lo unchanged as a real number, |lo| <= ulp(hi)/2 again).  Between two
// renormalisations lo has collected the changes of at most kFold moves in fp32 (R20: <= 16 fp32 terms are
// summed in fp32 before they reach the wide accumulator); hi + lo carries 48 significant bits against the 24
// of the pair terms that go into it.  This takes the fp32 -> fp64 conversions, which run at 1/8 rate on the
// unit that also serves rsqrt and rcp, off the per-pair path of an accepted move; fp64 appears where a sum is
// read (the owner of the moved particle) and when the state is stored.
constexpr int kFold = 16;
template <typename Real, int T, int J, int V, int PD, bool DBG>
__global__ void __launch_bounds__(T, (sweep_min_ctas<Real, T, J, PD>()))
sweep_kernel(StateView sv, TraceView tr, WriteoutView wo, uint2 key, uint32_t t0, int n_sweeps)
{
    static_assert(J % V == 0, "J must be a multiple of the vector width");
    static_assert(PD == 0 || (sizeof(Real) == 4 && V >= 2), "pending sums exist only in the packed FP32C path");
    constexpr bool kPend = (PD != 0);
    static_assert(V == 1 || V == 2 || V == 4, "vector width");
    using Coord = typename ModeT<Real>::Coord;
    using PackC = Pack<Coord, V>;
    constexpr bool kF32 = (sizeof(Real) == 4);
    constexpr bool kPacked = kF32 && V >= 2;              // two pair terms per FFMA2-class instruction
    constexpr int NP = T * J, G = J / V, nwarps = T >> 5, kSlot = MoveSlot<Real>::bytes;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = sv.N, ld = sv.ld;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int w = blockIdx.x;

    double         *S    = reinterpret_cast<double *>(smem_raw);                              // [NP], permuted (s_index)
    unsigned char  *rnd  = smem_raw + NP * 8;                                                 // [2][kChunk] 32-byte slots
    double         *part = reinterpret_cast<double *>(smem_raw + NP * 8 + 2 * kChunk * kSlot);   // [2][32]
    Coord          *x    = reinterpret_cast<Coord *>(part + 64);                              // [3][NP]
    Coord *y = x + NP, *z = x + 2 * NP;
    float *Shi = reinterpret_cast<float *>(S), *Slo = Shi + NP;                               // PD = 1: S as hi + lo, [NP] each
    static_assert(sizeof(MoveRand<Real>) <= kSlot, "variate record must fit its slot");

    const GroupDev g = sv.groups[sv.group_of[w]];
    SweepConst<Real> P;
    P.load(g);
    // 2 Delta = c2 * (sum t_new - S_s); the packed FP32C path keeps every sum in units of kT2Unit
    constexpr double kUnit = kPacked ? kT2Unit : 1.0, kInvUnit = 1.0 / kUnit;
    const double c2 = 2.0 * g.c1 * kUnit;
    // proposal half-width: FP64 exactly the caller's step [A]; FP32C in grid units (2^-23 box)
    const double step = kF32 ? g.step * g.inv_unit * 8388608.0 : g.step;
    const uint32_t wid = sv.walker_id_base + (uint32_t)w;

    // a1: walker state global -> shared, once per call
    Real *gpos = reinterpret_cast<Real *>(sv.pos) + (size_t)w * 3 * ld;
    double *gS = sv.S + (size_t)w * ld;
    for (int j = tid; j < NP; j += T) {
        Coord cx, cy, cz;
        double s = 0.0;
        if (j < N) {
            if constexpr (kF32) { cx = enc_coord(gpos[j]); cy = enc_coord(gpos[ld + j]); cz = enc_coord(gpos[2 * ld + j]); }
            else                { cx = gpos[j]; cy = gpos[ld + j]; cz = gpos[2 * ld + j]; }
            s = gS[j] * kInvUnit;
        } else {                                            // padding: NaN selects 0 in FP64; FP32C uses the bias
            if constexpr (kF32) { cx = 0; cy = 0; cz = 0; }
            else                { cx = cy = cz = poison_of<Real>(Coord(0)); }
        }
        x[j] = cx; y[j] = cy; z[j] = cz;
        if constexpr (kPend) {
            const float hi = __double2float_rn(s);
            Shi[j] = hi;
            Slo[j] = __double2float_rn(s - (double)hi);
        } else {
            S[s_index<T, V>(j)] = s;
        }
    }

    // per-pack clamp bias of this thread (FP32C): 1 for padding packs.  Requires N % V == 0 (planner).
    float bias[G];
#pragma unroll
    for (int gi = 0; gi < G; ++gi) bias[gi] = ((gi * T + tid) * V < N) ? 0.0f : 1.0f;
    f32x2 bias2[G];
#pragma unroll
    for (int gi = 0; gi < G; ++gi) bias2[gi] = ((gi * T + tid) * V < N) ? pk2(0.0f, 0.0f) : pk2(0x1p63f, 0x1p63f);

    const uint32_t total = (uint32_t)n_sweeps * (uint32_t)N;

    // a2: variates of moves [chunk*32, chunk*32+32) -> rnd[buf]
    auto produce = [&](uint32_t chunk, int buf) {
        if (warp != 0) return;
        const uint32_t m = chunk * kChunk + lane;
        if (m >= total) return;
        const uint32_t q = m / (uint32_t)N;
        const uint32_t idx = m - q * (uint32_t)N;
        MoveRand<Real> mr;
        double ax, ay, az;
        uint32_t wxi;
        if (DBG && sv.proposal == 1) {                     // random particle, Gaussian displacement (l.144, l.325)
            const uint4 A = philox4x32_10(make_uint4(idx, t0 + q, wid, 2u), key);
            const uint4 B = philox4x32_10(make_uint4(idx, t0 + q, wid, 3u), key);
            mr.s = (int32_t)__umulhi(A.x, (uint32_t)N);
            double z0, z1, z2, z3;
            normal_pair(A.y, A.z, z0, z1);
            normal_pair(B.x, B.y, z2, z3);
            ax = __dmul_rn(step, z0); ay = __dmul_rn(step, z1); az = __dmul_rn(step, z2);
            wxi = A.w;
        } else {                                           // particles in order, uniform cube (R7)
            const uint4 r = philox4x32_10(make_uint4(idx, t0 + q, wid, 0u), key);
            mr.s = (int32_t)idx;
            ax = __dmul_rn(step, word_to_pm1(r.x));
            ay = __dmul_rn(step, word_to_pm1(r.y));
            az = __dmul_rn(step, word_to_pm1(r.z));
            wxi = r.w;
        }
        if constexpr (kF32) {
            mr.dx = (int32_t)((uint32_t)__double2int_rn(ax) << 9);
            mr.dy = (int32_t)((uint32_t)__double2int_rn(ay) << 9);
            mr.dz = (int32_t)((uint32_t)__double2int_rn(az) << 9);
        } else {
            mr.dx = ax; mr.dy = ay; mr.dz = az;
        }
        mr.logxi = log(word_to_unit(wxi));
        *reinterpret_cast<MoveRand<Real> *>(rnd + (buf * kChunk + lane) * kSlot) = mr;
    };
    auto fetch = [&](uint32_t m) {
        return *reinterpret_cast<const MoveRand<Real> *>(rnd + ((int)((m >> 5) & 1) * kChunk + (int)(m & (kChunk - 1))) * kSlot);
    };
    produce(0, 0);
    if (tid == 0) *reinterpret_cast<int32_t *>(part + 63) = 0;
    __syncthreads();
    const int32_t zero = opaque_zero(reinterpret_cast<int32_t *>(part + 63));   // part[32..63] is used from move 1 on

    unsigned long long n_acc = 0;
    MoveRand<Real> mr = fetch(0);
    int s = DBG ? mr.s : 0;
    Coord xs = x[s], ys = y[s], zs = z[s];                 // the moved particle (prefetched one move ahead)
    int sp = -1;                                           // DBG: particle of the previous move and where it ended up
    Coord pxp = xs, pyp = ys, pzp = zs;
    __syncthreads();                                       // ... before its owner poisons it
    // Moves unrolled: the chunk test, the buffer parities and the loop control become static (10.21 -> 9.98 ms at
    // config 3 with 4, 45.2 -> 44.2 ms at config 4); 8 moves of the FP32C kernel and 4 of the fp64 kernel overflow the
    // instruction cache (12.4 ms; fp64: 24 -> 43 ms), 2 of the fp64 kernel gain nothing at config 3 and lose at config 5.
    constexpr int kMoveUnroll = (kF32 && !DBG) ? 4 : 1;
#pragma unroll kMoveUnroll
    for (uint32_t m = 0; m < total; ++m) {
        if ((m & (kChunk - 1)) == 0) produce((m >> 5) + 1, (int)(((m >> 5) + 1) & 1));   // published by this move's barrier
        const Coord tx = trial_coord(xs, mr.dx);
        const Coord ty = trial_coord(ys, mr.dy);
        const Coord tz = trial_coord(zs, mr.dz);
        const double logxi = mr.logxi;
        const bool owner = ((unsigned)tid == (((unsigned)s / (unsigned)V) & (unsigned)(T - 1)));
        if (owner) x[s] = poison_of<Real>(tx);             // self term = 0 (nobody else reads x[s] during this move)

        // prefetch the next move.  Lean kernel: particles in order, N >= 3 -- the next particle is touched
        // neither by this move nor by the previous one.  DBG kernel (any N, random particle): the next
        // particle may be this move's (resolved after the decision) or the previous move's (whose commit
        // by its owner is not ordered against this read: every thread kept the outcome in registers).
        MoveRand<Real> mrn = mr;
        if (m + 1 < total) mrn = fetch(m + 1);
        int sn;
        if constexpr (DBG) sn = mrn.s; else sn = (s + 1 == N) ? 0 : s + 1;
        Coord xn = x[sn], yn = y[sn], zn = z[sn];
        if constexpr (DBG) { if (sn == sp) { xn = pxp; yn = pyp; zn = pzp; } }

        // a3: trial terms of this thread's particles
        Real un[kPacked ? 1 : J];
        f32x2 un2[kPacked ? J / 2 : 1];
        Real accr = (Real)0;
        if constexpr (kPacked) {
            f32x2 acc2 = pk2(0.0f, 0.0f);
#pragma unroll
            for (int gi = 0; gi < G; ++gi) {
                const int base = (gi * T + tid) * V;
                const PackC X = *reinterpret_cast<const PackC *>(x + base);
                const PackC Y = *reinterpret_cast<const PackC *>(y + base);
                const PackC Z = *reinterpret_cast<const PackC *>(z + base);
#pragma unroll
                for (int e = 0; e < V; e += 2) {
                    const f32x2 t2 = pair_t2(tx, ty, tz, X.v[e], X.v[e + 1], Y.v[e], Y.v[e + 1], Z.v[e], Z.v[e + 1], bias2[gi], zero);
                    un2[(gi * V + e) / 2] = t2;
                    acc2 = add2(acc2, t2);
                }
            }
            float a0, a1;
            upk2(acc2, a0, a1);
            accr = a0 + a1;
        } else {
#pragma unroll
            for (int gi = 0; gi < G; ++gi) {
                const int base = (gi * T + tid) * V;
                const PackC X = *reinterpret_cast<const PackC *>(x + base);
                const PackC Y = *reinterpret_cast<const PackC *>(y + base);
                const PackC Z = *reinterpret_cast<const PackC *>(z + base);
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    un[gi * V + e] = pair_t(tx, ty, tz, X.v[e], Y.v[e], Z.v[e], bias[gi], P);
                    accr += un[gi * V + e];
                }
            }
        }
        double acc = (double)accr;
        if (owner) {                                       // a4: sum_j t_new - S_s
            double Ss;
            if constexpr (kPend) Ss = (double)Shi[s] + (double)Slo[s];
            else                 Ss = S[s_index<T, V>(s)];
            acc -= Ss;
        }

        // a5: block sum, identical bits in every thread
        double tot = warp_sum(acc);
        if (nwarps > 1) {
            double *pb = part + (int)(m & 1) * 32;
            if (lane == 0) pb[warp] = tot;
            __syncthreads();
            tot = sum_parts<nwarps>(pb);
        } else {
            __syncwarp();
        }

        // a6: decision (Eq.(5), strict, log form: R8)
        const double margin = fma(c2, tot, -logxi);
        const bool accept = margin > 0.0;
        if (DBG && tr.dec != nullptr) {
            if (tid == 0 && w >= tr.w_begin && w < tr.w_end) {
                const long long k = tr.offset + m;
                if (k < tr.capacity) {
                    const long long idx = (long long)(w - tr.w_begin) * tr.capacity + k;
                    tr.dec[idx] = accept ? 1 : 0;
                    if (tr.margin != nullptr) tr.margin[idx] = margin;
                }
            }
        }

        // a7: commit and update the running pair sums
        if (accept) {
            if (kF32 && owner) x[s] = poison_of<Real>(xs);  // distances are now taken from the old position
#pragma unroll
            for (int gi = 0; gi < G; ++gi) {
                const int base = (gi * T + tid) * V;
                const PackC X = *reinterpret_cast<const PackC *>(x + base);
                const PackC Y = *reinterpret_cast<const PackC *>(y + base);
                const PackC Z = *reinterpret_cast<const PackC *>(z + base);
                if constexpr (V == 1) {
                    const Real to = pair_t(xs, ys, zs, X.v[0], Y.v[0], Z.v[0], bias[gi], P);
                    S[base] += (double)(un[gi] - to);
                } else if constexpr (kPend) {
                    using PackF = Pack<float, V>;
                    PackF pd = *reinterpret_cast<const PackF *>(Slo + base);
#pragma unroll
                    for (int c = 0; c < V / 2; ++c) {
                        const f32x2 to2 = pair_t2(xs, ys, zs, X.v[2 * c], X.v[2 * c + 1], Y.v[2 * c], Y.v[2 * c + 1],
                                                  Z.v[2 * c], Z.v[2 * c + 1], bias2[gi], zero);
                        const f32x2 nw = add2(pk2(pd.v[2 * c], pd.v[2 * c + 1]), sub2(un2[(gi * V) / 2 + c], to2));
                        upk2(nw, pd.v[2 * c], pd.v[2 * c + 1]);
                    }
                    *reinterpret_cast<PackF *>(Slo + base) = pd;
                } else {
#pragma unroll
                    for (int c = 0; c < V / 2; ++c) {
                        double2 *sp = reinterpret_cast<double2 *>(S + ((gi * (V / 2) + c) * T + tid) * 2);
                        double2 sv2 = *sp;
                        if constexpr (kPacked) {
                            const f32x2 to2 = pair_t2(xs, ys, zs, X.v[2 * c], X.v[2 * c + 1], Y.v[2 * c], Y.v[2 * c + 1],
                                                      Z.v[2 * c], Z.v[2 * c + 1], bias2[gi], zero);
                            float d0, d1;
                            upk2(sub2(un2[(gi * V) / 2 + c], to2), d0, d1);
                            sv2.x += (double)d0;
                            sv2.y += (double)d1;
                        } else {
                            const Real t0o = pair_t(xs, ys, zs, X.v[2 * c], Y.v[2 * c], Z.v[2 * c], bias[gi], P);
                            const Real t1o = pair_t(xs, ys, zs, X.v[2 * c + 1], Y.v[2 * c + 1], Z.v[2 * c + 1], bias[gi], P);
                            sv2.x += (double)(un[gi * V + 2 * c] - t0o);
                            sv2.y += (double)(un[gi * V + 2 * c + 1] - t1o);
                        }
                        *sp = sv2;
                    }
                }
            }
            if (owner) {
                if constexpr (kPend) {
                    const double ns = (double)Shi[s] + (double)Slo[s] + tot;
                    const float hi = __double2float_rn(ns);
                    Shi[s] = hi;
                    Slo[s] = __double2float_rn(ns - (double)hi);
                } else {
                    S[s_index<T, V>(s)] += tot;
                }
                x[s] = commit_coord(tx, g.L);
                y[s] = commit_coord(ty, g.L);
                z[s] = commit_coord(tz, g.L);
            }
            ++n_acc;
        } else if (owner) {
            x[s] = xs;                                      // undo the poison
        }
        if constexpr (kPend) {
            if ((m & (kFold - 1)) == kFold - 1) {             // renormalise this thread's sums: TwoSum(hi, lo)
#pragma unroll
                for (int gi = 0; gi < G; ++gi) {
                    using PackF = Pack<float, V>;
                    const int base = (gi * T + tid) * V;
                    PackF ph = *reinterpret_cast<const PackF *>(Shi + base);
                    PackF pl = *reinterpret_cast<const PackF *>(Slo + base);
#pragma unroll
                    for (int c = 0; c < V / 2; ++c) {
                        const f32x2 h2 = pk2(ph.v[2 * c], ph.v[2 * c + 1]), l2 = pk2(pl.v[2 * c], pl.v[2 * c + 1]);
                        const f32x2 sm = add2(h2, l2);
                        const f32x2 bb = sub2(sm, h2);
                        const f32x2 er = add2(sub2(h2, sub2(sm, bb)), sub2(l2, bb));
                        upk2(sm, ph.v[2 * c], ph.v[2 * c + 1]);
                        upk2(er, pl.v[2 * c], pl.v[2 * c + 1]);
                    }
                    *reinterpret_cast<PackF *>(Shi + base) = ph;
                    *reinterpret_cast<PackF *>(Slo + base) = pl;
                }
            }
        }
        if constexpr (DBG) {
            const Coord cx = accept ? commit_coord(tx, g.L) : xs;
            const Coord cy = accept ? commit_coord(ty, g.L) : ys;
            const Coord cz = accept ? commit_coord(tz, g.L) : zs;
            if (sn == s) { xn = cx; yn = cy; zn = cz; }
            sp = s; pxp = cx; pyp = cy; pzp = cz;
        }
        if constexpr (DBG) {                               // end of a sweep: optional in-kernel write-out (NEXT-4)
            if (wo.xyz != nullptr && wo.every > 0 && (m + 1) % (uint32_t)N == 0) {
                const uint32_t done = (m + 1) / (uint32_t)N;
                if (done % (uint32_t)wo.every == 0 && (int)(done / (uint32_t)wo.every) <= wo.n_out)
                    writeout_walker<T>(wo, (int)(done / (uint32_t)wo.every) - 1, w, sv.W, N, g.L_A, x, y, z, sv.n_acc[w] + n_acc);
            }
        }
        s = sn;
        xs = xn; ys = yn; zs = zn;
        mr = mrn;
    }
    __syncthreads();

    // a8: shared -> global, once per call
    for (int j = tid; j < N; j += T) {
        if constexpr (kF32) { gpos[j] = dec_coord(x[j]); gpos[ld + j] = dec_coord(y[j]); gpos[2 * ld + j] = dec_coord(z[j]); }
        else                { gpos[j] = x[j]; gpos[ld + j] = y[j]; gpos[2 * ld + j] = z[j]; }
        if constexpr (kPend) gS[j] = ((double)Shi[j] + (double)Slo[j]) * kUnit;
        else                 gS[j] = S[s_index<T, V>(j)] * kUnit;
    }
    if (tid == 0) sv.n_acc[w] += n_acc;
}

// ---- host side: one table entry per compiled (T, J, V, PD, K) shape -----------------------------------
// K = 1: this file's one-move kernel; K > 1: the tile kernel of qmc_sweep_tile.cuh (FP32C, PD = 1).
struct SweepShape {
    int T, J, V, P, K;
    cudaError_t (*launch)(qmc_ctx *c, int n_sweeps, int smem);
    int (*occupancy)(int smem);
    int smem;
};

template <typename Real, int T, int J, int V, int PD>
static cudaError_t shape_launch(qmc_ctx *c, int n_sweeps, int smem)
{
    const uint2 key = make_uint2((uint32_t)(c->seed & 0xFFFFFFFFull), (uint32_t)(c->seed >> 32));
    // the lean instantiation has neither the decision trace, the write-outs nor the general next-particle
    // handling (N < 3, proposal 1)
    const bool dbg = c->trace.dec != nullptr || c->p.N < 3 || c->sv.proposal != 0 || c->wo.xyz != nullptr;
    auto kern = dbg ? sweep_kernel<Real, T, J, V, PD, true> : sweep_kernel<Real, T, J, V, PD, false>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    kern<<<c->W, T, smem, c->stream>>>(c->sv, c->trace, c->wo, key, c->t, n_sweeps);
    return cudaGetLastError();
}

template <typename Real, int T, int J, int V, int PD>
static int shape_occupancy(int smem)
{
    int n = 0;
    auto kern = sweep_kernel<Real, T, J, V, PD, false>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, T, smem) != cudaSuccess) return 0;
    return n;
}

#define QMC_SHAPE_ENTRY(Real, TT, JJ, VV, PP) {TT, JJ, VV, PP, 1, shape_launch<Real, TT, JJ, VV, PP>, shape_occupancy<Real, TT, JJ, VV, PP>, \
                                               sweep_smem_bytes(TT, JJ, sizeof(Real) == 8 ? QMC_FP64 : QMC_FP32C, PP)},

const SweepShape *sweep_shapes_f32(int *n);
const SweepShape *sweep_shapes_f64(int *n);
const SweepShape *sweep_shapes_tile(int *n);       // qmc_sweep_tile_f32.cu

}  // namespace qmc
