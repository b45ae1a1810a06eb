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

struct MoveRand { double dx, dy, dz, logxi; };   // displacement (already times step) and log(xi)

template <typename Real> __device__ __forceinline__ Real trial_coord(Real x, double d);
template <> __device__ __forceinline__ double trial_coord<double>(double x, double d) { return __dadd_rn(x, d); }
template <> __device__ __forceinline__ float trial_coord<float>(float x, double d)   // R20: one rounding to fp32
{
    return __double2float_rn(__dadd_rn((double)x, d));
}
template <typename Real> __device__ __forceinline__ Real wrap_coord(Real x, Real L)   // R10
{
    if (x >= L) x -= L;
    if (x < (Real)0) x += L;
    return x;
}

__device__ __forceinline__ void copy16(void *dst, const void *src, int bytes, int tid, int nthreads)
{
    uint4 *d = reinterpret_cast<uint4 *>(dst);
    const uint4 *s = reinterpret_cast<const uint4 *>(src);
    for (int i = tid; i < bytes / 16; i += nthreads) d[i] = s[i];
}

static int sweep_smem_bytes(int ld, int mode)
{
    const int real = (mode == QMC_FP64) ? 8 : 4;
    return ld * 8 + 2 * kChunk * (int)sizeof(MoveRand) + 64 * 8 + 3 * ld * real;
}

// Resident CTAs per SM the register allocator should leave room for: what shared memory allows at
// the largest N this (T,J) serves, capped so that fp64 code keeps >= ~80 and fp32 code >= ~48 registers.
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

template <typename Real, int T, int J>
__global__ void __launch_bounds__(T, (sweep_min_ctas<Real, T, J>()))
sweep_kernel(StateView sv, TraceView tr, uint2 key, uint32_t t0, int n_sweeps)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = sv.N, ld = sv.ld;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int nwarps = T >> 5;
    const int w = blockIdx.x;

    double   *S    = reinterpret_cast<double *>(smem_raw);                       // [ld]
    MoveRand *rnd  = reinterpret_cast<MoveRand *>(S + ld);                       // [2][kChunk]
    double   *part = reinterpret_cast<double *>(rnd + 2 * kChunk);               // [2][32]
    Real     *X    = reinterpret_cast<Real *>(part + 64);                        // [3][ld]
    Real *x = X, *y = X + ld, *z = X + 2 * ld;

    const GroupDev g = sv.groups[sv.group_of[w]];
    PairConst<Real> P;
    P.load(g);
    const double step = g.step;
    const uint32_t wid = sv.walker_id_base + (uint32_t)w;

    // a1: walker state global -> shared, once per call, 16-byte vectors
    Real *gpos = reinterpret_cast<Real *>(sv.pos) + (size_t)w * 3 * ld;
    double *gS = sv.S + (size_t)w * ld;
    copy16(X, gpos, 3 * ld * (int)sizeof(Real), tid, T);
    copy16(S, gS, ld * 8, tid, T);

    const long long total = (long long)n_sweeps * N;

    // a2: variates of moves [chunk*32, chunk*32+32) -> rnd[buf]
    auto produce = [&](long long chunk, int buf) {
        if (warp != 0) return;
        const long long m = chunk * kChunk + lane;
        if (m >= total) return;
        const uint32_t t = t0 + (uint32_t)(m / N);
        const uint32_t s = (uint32_t)(m % N);
        const uint4 r = philox4x32_10(make_uint4(s, t, wid, 0u), key);
        MoveRand mr;
        mr.dx = __dmul_rn(step, word_to_pm1(r.x));
        mr.dy = __dmul_rn(step, word_to_pm1(r.y));
        mr.dz = __dmul_rn(step, word_to_pm1(r.z));
        mr.logxi = log(word_to_unit(r.w));
        rnd[buf * kChunk + lane] = mr;
    };
    produce(0, 0);
    __syncthreads();

    unsigned long long n_acc = 0;
    int s = 0;
    for (long long m = 0; m < total; ++m) {
        const int ci = (int)(m & (kChunk - 1));
        const int buf = (int)((m >> 5) & 1);
        if (ci == 0) produce((m >> 5) + 1, buf ^ 1);      // published by this move's barrier
        const MoveRand mr = rnd[buf * kChunk + ci];

        const Real xs = x[s], ys = y[s], zs = z[s];        // broadcast read of the moved particle
        const Real tx = trial_coord<Real>(xs, mr.dx);
        const Real ty = trial_coord<Real>(ys, mr.dy);
        const Real tz = trial_coord<Real>(zs, mr.dz);
        const bool owner = (tid == (s & (T - 1)));

        // a3: trial terms of this thread's particles
        Real un[J];
        Real accr = (Real)0;
#pragma unroll
        for (int i = 0; i < J; ++i) {
            const int j = tid + i * T;
            Real u = (Real)0;
            if (j < N) {
                Real r2 = min_image_r2<Real>(tx, ty, tz, x[j], y[j], z[j], P);
                if (j == s) r2 = P.h2;                     // R9: exclude by index
                u = pair_u<Real>(r2, P);
            }
            un[i] = u;
            accr += u;
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
        if (tr.dec != nullptr && tid == 0 && w >= tr.w_begin && w < tr.w_end) {
            const long long k = tr.offset + m;
            if (k < tr.capacity) {
                const long long idx = (long long)(w - tr.w_begin) * tr.capacity + k;
                tr.dec[idx] = accept ? 1 : 0;
                if (tr.margin != nullptr) tr.margin[idx] = margin;
            }
        }

        // a7: commit and update the running pair sums
        if (accept) {
#pragma unroll
            for (int i = 0; i < J; ++i) {
                const int j = tid + i * T;
                if (j < N && j != s) {
                    const Real r2 = min_image_r2<Real>(xs, ys, zs, x[j], y[j], z[j], P);
                    const Real uo = pair_u<Real>(r2, P);
                    S[j] += (double)(un[i] - uo);
                }
            }
            if (owner) {
                S[s] += tot;
                x[s] = wrap_coord<Real>(tx, P.L);
                y[s] = wrap_coord<Real>(ty, P.L);
                z[s] = wrap_coord<Real>(tz, P.L);
            }
            ++n_acc;
        }
        if (++s == N) s = 0;
    }
    __syncthreads();

    // a8: shared -> global, once per call
    copy16(gpos, X, 3 * ld * (int)sizeof(Real), tid, T);
    copy16(gS, S, ld * 8, tid, T);
    if (tid == 0) sv.n_acc[w] += n_acc;
}

// (T, J) combinations compiled: threads per CTA x particles per thread, J*T >= N.
#define QMC_SWEEP_SHAPES(X) \
    X(32, 1) X(64, 1) X(64, 2) X(64, 4) X(128, 1) X(128, 2) X(128, 4) X(128, 8) X(128, 16) \
    X(256, 1) X(256, 2) X(256, 4) X(256, 8) X(512, 4) X(512, 8) X(1024, 2) X(1024, 4) X(1024, 8) \
    X(1024, 10) X(1024, 12) X(1024, 16)

template <typename Real, int T, int J>
static cudaError_t launch_one(qmc_ctx *c, int n_sweeps)
{
    auto kern = sweep_kernel<Real, T, J>;
    const SweepPlan &pl = c->sweep_plan;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, pl.smem_bytes);
    if (e != cudaSuccess) return e;
    const uint2 key = make_uint2((uint32_t)(c->seed & 0xFFFFFFFFull), (uint32_t)(c->seed >> 32));
    kern<<<c->W, T, pl.smem_bytes, c->stream>>>(c->sv, c->trace, key, c->t, n_sweeps);
    return cudaGetLastError();
}

template <typename Real>
static cudaError_t launch_shape(qmc_ctx *c, int n_sweeps)
{
    const int T = c->sweep_plan.threads, J = c->sweep_plan.J;
#define X(TT, JJ) if (T == TT && J == JJ) return launch_one<Real, TT, JJ>(c, n_sweeps);
    QMC_SWEEP_SHAPES(X)
#undef X
    return cudaErrorInvalidValue;
}

cudaError_t launch_sweep(qmc_ctx *c, int n_sweeps)
{
    c->launches += 1;
    return c->p.mode == QMC_FP64 ? launch_shape<double>(c, n_sweeps) : launch_shape<float>(c, n_sweeps);
}

template <typename Real, int T, int J>
static int occupancy_of(int smem)
{
    int n = 0;
    auto kern = sweep_kernel<Real, T, J>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, T, smem) != cudaSuccess) return 0;
    return n;
}

static bool shape_exists(int T, int J)
{
#define X(TT, JJ) if (T == TT && J == JJ) return true;
    QMC_SWEEP_SHAPES(X)
#undef X
    return false;
}

// Threads per CTA (power of two) and particles per thread J (J*T >= N) for this N.
// QMC_SWEEP_THREADS=<T> overrides the heuristic (tuning experiments).
bool plan_sweep(qmc_ctx *c, SweepPlan *out)
{
    const int N = c->p.N;
    int T;
    if (N <= 32)         T = 32;
    else if (N <= 64)    T = 64;
    else if (N <= 512)   T = 128;
    else if (N <= 2048)  T = 256;
    else if (N <= 4096)  T = 512;
    else                 T = 1024;
    if (const char *env = getenv("QMC_SWEEP_THREADS")) {
        const int v = atoi(env);
        if (v >= 32 && v <= 1024 && (v & (v - 1)) == 0) T = v;
    }
    int J = 0;
    for (; T <= 1024 && J == 0; T *= 2)
        for (int j = 1; j <= 16; ++j)
            if ((long long)j * T >= N && shape_exists(T, j)) { J = j; break; }
    T /= 2;
    if (J == 0) return false;
    out->threads = T;
    out->J = J;
    out->smem_bytes = sweep_smem_bytes(c->ld, c->p.mode);
    if (out->smem_bytes > 227 * 1024) return false;
    int occ = 0;
#define X(TT, JJ) if (T == TT && J == JJ) occ = (c->p.mode == QMC_FP64) ? occupancy_of<double, TT, JJ>(out->smem_bytes) \
                                                                        : occupancy_of<float, TT, JJ>(out->smem_bytes);
    QMC_SWEEP_SHAPES(X)
#undef X
    out->ctas_per_sm = occ;
    return true;
}

}  // namespace qmc
