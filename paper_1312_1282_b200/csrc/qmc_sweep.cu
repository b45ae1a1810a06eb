// qmc_sweep.cu -- the Metropolis sweep kernel.
//
// One CTA per walker ("each thread block serves one walker").  The walker's
// coordinates (SoA) and running pair sums S_i stay in shared memory for the whole call (l.175, l.323
// "shared memory persistence"); global memory is touched once on entry and once on exit.
//
// Per move (particle s, sweep t):
//   a2  variates from Philox4x32-10(counter (s,t,walker,0), key seed), prepared 32 moves at a time
//       by warp 0 (one move per lane, including log(xi)) into a double-buffered shared array;
//   a3  thread tid evaluates u(|r'_s - r_j|) for its own particles j = tid, tid+T, ... (J of them),
//       keeps the values in registers;
//   a4  the old sum is the running S_s (only the thread that owns s reads it);
//   a5  xor-butterfly warp sums + one shared-memory exchange: every thread ends with the same bits;
//   a6  every thread takes the same decision 2*Delta > log(xi): ONE __syncthreads per move;
//   a7  on accept each thread re-evaluates the OLD terms of its own particles and updates its own
//       S_j += u_new - u_old; the owner of s commits the wrapped position and S_s.
// Ownership of particle j by thread (j mod T) is static, so S and the pair loops need no
// synchronisation at all; the only cross-thread data are r_s (read by all at the start of move s,
// written by its owner after the decision, at least one barrier earlier) and the partial sums.
#include "qmc_internal.h"

namespace qmc {

constexpr int kChunk = 32;                       // moves prepared at a time (one per lane of warp 0)

// Displacement (in coordinate units, already times step) and log(xi) of one move.
template <typename Real> struct MoveRand { double logxi; Real dx, dy, dz; };

// FP64: trial = r_s + delta with ONE rounding (bit-identical to the oracle).  FP32C: the displacement is
// rounded to fp32 once per move and added in fp32; on the uniform 2^-23 grid of [1,2) this is a symmetric
// proposal (R20).
template <typename Real> __device__ __forceinline__ Real trial_coord(Real x, Real d);
template <> __device__ __forceinline__ double trial_coord<double>(double x, double d) { return __dadd_rn(x, d); }
template <> __device__ __forceinline__ float trial_coord<float>(float x, float d) { return __fadd_rn(x, d); }

template <typename Real> __device__ __forceinline__ Real wrap_coord(Real x, Real lo, Real hi, Real L)   // R10
{
    if (x >= hi) x -= L;
    if (x < lo) x += L;
    return x;
}

template <typename Real> __device__ __forceinline__ Real quiet_nan();
template <> __device__ __forceinline__ double quiet_nan<double>() { return __longlong_as_double(0x7ff8000000000000LL); }
template <> __device__ __forceinline__ float quiet_nan<float>() { return __int_as_float(0x7fc00000); }

__device__ __forceinline__ void copy16(void *dst, const void *src, int bytes, int tid, int nthreads)
{
    uint4 *d = reinterpret_cast<uint4 *>(dst);
    const uint4 *s = reinterpret_cast<const uint4 *>(src);
    for (int i = tid; i < bytes / 16; i += nthreads) d[i] = s[i];
}

// V consecutive values as one shared-memory vector access.
template <typename Real, int V> struct alignas(sizeof(Real) * V) Pack { Real v[V]; };

static int sweep_smem_bytes(int T, int J, int mode)
{
    const int real = (mode == QMC_FP64) ? 8 : 4;
    const int NP = T * J;
    return NP * 8 + 2 * kChunk * 32 + 64 * 8 + 3 * NP * real;
}

// Resident CTAs per SM the register allocator should leave room for: what shared memory allows for
// this (T,J), capped so that fp64 code keeps >= ~80 and fp32 code >= ~48 registers.
template <typename Real, int T, int J>
constexpr int sweep_min_ctas()
{
    const int real = (int)sizeof(Real);
    const int smem = J * T * (8 + 3 * real) + 2 * kChunk * 32 + 64 * 8 + 1024;
    const int by_smem = (228 * 1024) / smem;
    const int by_regs = (real == 8 ? 768 : 1280) / T;
    int n = by_smem < by_regs ? by_smem : by_regs;
    return n < 1 ? 1 : (n > 32 ? 32 : n);
}

// T threads per CTA; each thread owns J particles in J/V groups of V consecutive ones:
// particle j = ((g*T + tid)*V + e), g < J/V, e < V.  Shared arrays are padded to NP = T*J entries;
// the padding holds NaN coordinates, for which every pair term selects 0 -- no bounds checks in the loops.
template <typename Real, int T, int J, int V, bool kTrace>
__global__ void __launch_bounds__(T, (sweep_min_ctas<Real, T, J>()))
sweep_kernel(StateView sv, TraceView tr, uint2 key, uint32_t t0, int n_sweeps)
{
    static_assert(J % V == 0, "J must be a multiple of the vector width");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NP = T * J, G = J / V, nwarps = T >> 5;
    using PackR = Pack<Real, V>;
    using PackD = Pack<double, V>;
    const int N = sv.N, ld = sv.ld;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int w = blockIdx.x;

    double         *S    = reinterpret_cast<double *>(smem_raw);                         // [NP]
    MoveRand<Real> *rnd  = reinterpret_cast<MoveRand<Real> *>(S + NP);                   // [2][kChunk] (32 B slots)
    double         *part = reinterpret_cast<double *>(smem_raw + NP * 8 + 2 * kChunk * 32);   // [2][32]
    Real           *x    = reinterpret_cast<Real *>(part + 64);                          // [3][NP]
    Real *y = x + NP, *z = x + 2 * NP;
    static_assert(sizeof(MoveRand<Real>) <= 32, "variate record must fit its 32-byte slot");

    const GroupDev g = sv.groups[sv.group_of[w]];
    PairConst<Real> P;
    P.load(g);
    // proposal half-width in coordinate units; FP64: exactly the caller's step
    const double step = (sizeof(Real) == 8) ? g.step : g.step * g.inv_unit;
    const Real lo = (Real)g.origin, hi = (Real)(g.origin + g.L);
    const uint32_t wid = sv.walker_id_base + (uint32_t)w;

    // a1: walker state global -> shared, once per call, 16-byte vectors; NaN / 0 in the padding
    Real *gpos = reinterpret_cast<Real *>(sv.pos) + (size_t)w * 3 * ld;
    double *gS = sv.S + (size_t)w * ld;
    copy16(x, gpos, ld * (int)sizeof(Real), tid, T);
    copy16(y, gpos + ld, ld * (int)sizeof(Real), tid, T);
    copy16(z, gpos + 2 * ld, ld * (int)sizeof(Real), tid, T);
    copy16(S, gS, ld * 8, tid, T);
    __syncthreads();
    for (int j = N + tid; j < NP; j += T) {
        x[j] = quiet_nan<Real>(); y[j] = quiet_nan<Real>(); z[j] = quiet_nan<Real>();
        S[j] = 0.0;
    }

    const uint32_t total = (uint32_t)n_sweeps * (uint32_t)N;

    // a2: variates of moves [chunk*32, chunk*32+32) -> rnd[buf]
    auto produce = [&](uint32_t chunk, int buf) {
        if (warp != 0) return;
        const uint32_t m = chunk * kChunk + lane;
        if (m >= total) return;
        const uint32_t q = m / (uint32_t)N;
        const uint32_t s = m - q * (uint32_t)N;
        const uint4 r = philox4x32_10(make_uint4(s, t0 + q, wid, 0u), key);
        MoveRand<Real> mr;
        mr.dx = (Real)__dmul_rn(step, word_to_pm1(r.x));
        mr.dy = (Real)__dmul_rn(step, word_to_pm1(r.y));
        mr.dz = (Real)__dmul_rn(step, word_to_pm1(r.z));
        mr.logxi = log(word_to_unit(r.w));
        *reinterpret_cast<MoveRand<Real> *>(reinterpret_cast<unsigned char *>(rnd) + (buf * kChunk + lane) * 32) = mr;
    };
    produce(0, 0);
    __syncthreads();

    unsigned long long n_acc = 0;
    int s = 0;
    for (uint32_t m = 0; m < total; ++m) {
        const int ci = (int)(m & (kChunk - 1));
        const int buf = (int)((m >> 5) & 1);
        if (ci == 0) produce((m >> 5) + 1, buf ^ 1);      // published by this move's barrier
        const MoveRand<Real> mr =
            *reinterpret_cast<const MoveRand<Real> *>(reinterpret_cast<const unsigned char *>(rnd) + (buf * kChunk + ci) * 32);

        const Real xs = x[s], ys = y[s], zs = z[s];        // broadcast read of the moved particle
        const Real tx = trial_coord<Real>(xs, mr.dx);
        const Real ty = trial_coord<Real>(ys, mr.dy);
        const Real tz = trial_coord<Real>(zs, mr.dz);
        const bool owner = (tid == (s / V) % T);

        // a3: trial terms of this thread's particles
        Real un[J];
        Real accr = (Real)0;
#pragma unroll
        for (int gi = 0; gi < G; ++gi) {
            const int base = (gi * T + tid) * V;
            const PackR X = *reinterpret_cast<const PackR *>(x + base);
            const PackR Y = *reinterpret_cast<const PackR *>(y + base);
            const PackR Z = *reinterpret_cast<const PackR *>(z + base);
#pragma unroll
            for (int e = 0; e < V; ++e) {
                const Real r2 = min_image_r2<Real>(tx, ty, tz, X.v[e], Y.v[e], Z.v[e], P);
                const Real u = pair_u_raw<Real>(r2, P);
                const bool keep = (r2 < P.h2) && (base + e != s);      // cutoff (R2), j != s by index (R9), NaN padding
                un[gi * V + e] = keep ? u : (Real)0;
                accr += un[gi * V + e];
            }
        }
        double acc = (double)accr;
        if (owner) acc -= S[s];                            // a4: Delta = sum_j u_new - S_s

        // a5: block sum, identical bits in every thread
        double tot = warp_sum(acc);
        if (nwarps > 1) {
            double *pb = part + (int)(m & 1) * 32;
            if (lane == 0) pb[warp] = tot;
            __syncthreads();
            tot = warp_sum(lane < nwarps ? pb[lane] : 0.0);
        } else {
            __syncwarp();
        }

        // a6: decision (Eq.(5), strict, log form: R8)
        const double margin = 2.0 * tot - mr.logxi;
        const bool accept = margin > 0.0;
        if (kTrace) {
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
#pragma unroll
            for (int gi = 0; gi < G; ++gi) {
                const int base = (gi * T + tid) * V;
                const PackR X = *reinterpret_cast<const PackR *>(x + base);
                const PackR Y = *reinterpret_cast<const PackR *>(y + base);
                const PackR Z = *reinterpret_cast<const PackR *>(z + base);
                PackD Sv = *reinterpret_cast<const PackD *>(S + base);
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    const Real r2 = min_image_r2<Real>(xs, ys, zs, X.v[e], Y.v[e], Z.v[e], P);
                    const Real u = pair_u_raw<Real>(r2, P);
                    const bool keep = (r2 < P.h2) && (base + e != s);
                    const Real uo = keep ? u : (Real)0;
                    Sv.v[e] += (double)(un[gi * V + e] - uo);
                }
                *reinterpret_cast<PackD *>(S + base) = Sv;
            }
            if (owner) {
                S[s] += tot;
                x[s] = wrap_coord<Real>(tx, lo, hi, P.L);
                y[s] = wrap_coord<Real>(ty, lo, hi, P.L);
                z[s] = wrap_coord<Real>(tz, lo, hi, P.L);
            }
            ++n_acc;
        }
        if (++s == N) s = 0;
    }
    __syncthreads();

    // a8: shared -> global, once per call
    copy16(gpos, x, ld * (int)sizeof(Real), tid, T);
    copy16(gpos + ld, y, ld * (int)sizeof(Real), tid, T);
    copy16(gpos + 2 * ld, z, ld * (int)sizeof(Real), tid, T);
    __syncthreads();
    for (int j = N + tid; j < ld; j += T) {               // keep the row padding of the global state clean
        gpos[j] = (Real)g.origin; gpos[ld + j] = (Real)g.origin; gpos[2 * ld + j] = (Real)g.origin;
    }
    copy16(gS, S, ld * 8, tid, T);
    if (tid == 0) sv.n_acc[w] += n_acc;
}

// (T, J, V) shapes compiled: threads per CTA x particles per thread (J*T >= N) x vector width.
// V = 1 shapes serve small N (every lane busy); vector shapes use 16-byte shared-memory accesses.
#define QMC_SWEEP_SHAPES_F(X) \
    X(32, 1, 1) X(64, 1, 1) X(128, 1, 1) X(128, 2, 1) X(128, 4, 1) \
    X(128, 16, 4) X(256, 4, 4) X(256, 8, 4) X(512, 4, 4) X(512, 8, 4) X(1024, 8, 4) X(1024, 10, 2)
#define QMC_SWEEP_SHAPES_D(X) \
    X(32, 1, 1) X(64, 1, 1) X(128, 1, 1) X(128, 2, 1) X(128, 4, 1) \
    X(128, 16, 2) X(256, 4, 2) X(256, 8, 2) X(512, 4, 2) X(512, 8, 2) X(1024, 8, 2) X(1024, 10, 2)

template <typename Real, int T, int J, int V>
static cudaError_t launch_one(qmc_ctx *c, int n_sweeps)
{
    const SweepPlan &pl = c->sweep_plan;
    const uint2 key = make_uint2((uint32_t)(c->seed & 0xFFFFFFFFull), (uint32_t)(c->seed >> 32));
    cudaError_t e;
    if (c->trace.dec != nullptr) {
        auto kern = sweep_kernel<Real, T, J, V, true>;
        if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, pl.smem_bytes)) != cudaSuccess) return e;
        kern<<<c->W, T, pl.smem_bytes, c->stream>>>(c->sv, c->trace, key, c->t, n_sweeps);
    } else {
        auto kern = sweep_kernel<Real, T, J, V, false>;
        if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, pl.smem_bytes)) != cudaSuccess) return e;
        kern<<<c->W, T, pl.smem_bytes, c->stream>>>(c->sv, c->trace, key, c->t, n_sweeps);
    }
    return cudaGetLastError();
}

cudaError_t launch_sweep(qmc_ctx *c, int n_sweeps)
{
    c->launches += 1;
    const int T = c->sweep_plan.threads, J = c->sweep_plan.J, V = c->sweep_plan.V;
    if (c->p.mode == QMC_FP64) {
#define X(TT, JJ, VV) if (T == TT && J == JJ && V == VV) return launch_one<double, TT, JJ, VV>(c, n_sweeps);
        QMC_SWEEP_SHAPES_D(X)
#undef X
    } else {
#define X(TT, JJ, VV) if (T == TT && J == JJ && V == VV) return launch_one<float, TT, JJ, VV>(c, n_sweeps);
        QMC_SWEEP_SHAPES_F(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

template <typename Real, int T, int J, int V>
static int occupancy_of(int smem)
{
    int n = 0;
    auto kern = sweep_kernel<Real, T, J, V, false>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, T, smem) != cudaSuccess) return 0;
    return n;
}

// vector width of the compiled shape (T,J) in this mode, 0 if there is none
static int shape_V(int mode, int T, int J)
{
    if (mode == QMC_FP64) {
#define X(TT, JJ, VV) if (T == TT && J == JJ) return VV;
        QMC_SWEEP_SHAPES_D(X)
#undef X
    } else {
#define X(TT, JJ, VV) if (T == TT && J == JJ) return VV;
        QMC_SWEEP_SHAPES_F(X)
#undef X
    }
    return 0;
}

// Threads per CTA and particles per thread J (J*T >= N) for this N.
// QMC_SWEEP_SHAPE="T,J" overrides the heuristic (tuning experiments).
bool plan_sweep(qmc_ctx *c, SweepPlan *out)
{
    const int N = c->p.N, mode = c->p.mode;
    int T = 0, J = 0;
    if (N <= 32)         { T = 32;   J = 1; }
    else if (N <= 64)    { T = 64;   J = 1; }
    else if (N <= 128)   { T = 128;  J = 1; }
    else if (N <= 256)   { T = 128;  J = 2; }
    else if (N <= 512)   { T = 128;  J = 4; }
    else if (N <= 1024)  { T = 256;  J = 4; }
    else if (N <= 2048)  { T = 256;  J = 8; }
    else if (N <= 4096)  { T = 512;  J = 8; }
    else if (N <= 8192)  { T = 1024; J = 8; }
    else if (N <= 10240) { T = 1024; J = 10; }
    if (const char *env = getenv("QMC_SWEEP_SHAPE")) {
        int t = 0, j = 0;
        if (sscanf(env, "%d,%d", &t, &j) == 2 && (long long)t * j >= N && shape_V(mode, t, j) > 0) { T = t; J = j; }
    }
    out->threads = T; out->J = J; out->V = 0; out->smem_bytes = 0; out->ctas_per_sm = 0;
    if (T == 0) { out->smem_bytes = N * (8 + 3 * (mode == QMC_FP64 ? 8 : 4)); return false; }
    out->V = shape_V(mode, T, J);
    out->smem_bytes = sweep_smem_bytes(T, J, mode);
    if (out->V == 0 || out->smem_bytes > 227 * 1024) return false;
    int occ = 0;
    if (mode == QMC_FP64) {
#define X(TT, JJ, VV) if (T == TT && J == JJ) occ = occupancy_of<double, TT, JJ, VV>(out->smem_bytes);
        QMC_SWEEP_SHAPES_D(X)
#undef X
    } else {
#define X(TT, JJ, VV) if (T == TT && J == JJ) occ = occupancy_of<float, TT, JJ, VV>(out->smem_bytes);
        QMC_SWEEP_SHAPES_F(X)
#undef X
    }
    out->ctas_per_sm = occ;
    return true;
}

}  // namespace qmc
