// qmc_sweep_cluster.cuh -- ONE walker advanced by a thread-block CLUSTER.
//
// "it is possible to use all multiprocessors of a GPU to work on a single walker" -- the
// paper tried a cooperating whole-GPU kernel with a global inter-block barrier (Ref. [26]) and left it out; its
// Kepler kernel reached 40 960 atoms by parking coordinates in registers (l.357, l.527).  On sm_100a the same two
// needs -- a walker larger than one SM's shared memory, and one walker (the equilibration case, l.311, l.490) on
// more than one SM -- are met by a cluster of C <= 8 thread blocks with distributed shared memory:
//
//   * particles are dealt to the C blocks in contiguous slices of Nc; block r keeps the coordinates and running
//     pair sums S_j of ITS slice in its own shared memory for the whole call (l.175 persistence), with the same
//     static thread ownership as the one-block kernel (qmc_sweep_impl.cuh);
//   * the coordinates of the next moved particle are written by the thread that owns it into EVERY block's shared
//     memory (st.shared::cluster through map_shared_rank), one move ahead; every block derives the same Philox
//     variates itself (no traffic);
//   * each block sums the trial terms of its slice (warp shuffles + one __syncthreads), then C threads push the
//     block total into every block's exchange array; ONE cluster barrier (barrier.cluster arrive.release /
//     wait.acquire) per move publishes totals and next coordinates; every thread of every block adds the C totals
//     in the same order and takes the same decision (Eq.(5) l.123) on identical bits;
//   * on accept every thread updates the S_j it owns; the owner of the moved particle commits it.  No other
//     inter-block traffic: 8 C bytes + 3 coordinates per move and block.
//
// Same arithmetic as the one-block kernel per pair term; only the summation order of Delta differs (R12), so fp64
// trajectories still match the oracle move for move (tests) and FP32C margins stay inside the R23 bound.
// Proposal 0 (ordered particles) only; N >= 3.
#pragma once
#include <cooperative_groups.h>

#include "qmc_sweep_impl.cuh"

namespace qmc {

namespace cg = cooperative_groups;

constexpr int kClusterMax = 8;                 // portable cluster size

static inline int sweep_cluster_smem_bytes(int T, int J, int mode)
{
    const int real = (mode == QMC_FP64) ? 8 : 4;
    const int slot = (mode == QMC_FP64) ? MoveSlot<double>::bytes : MoveSlot<float>::bytes;
    const int NP = T * J;
    // S, variate ring, warp partials [2][32], block totals [2][kClusterMax], moved-particle slots [2][4] (8-byte
    // slots in both modes), opaque zero, coordinates
    return NP * 8 + 2 * kChunk * slot + 64 * 8 + 2 * kClusterMax * 8 + 2 * 4 * 8 + 16 + 3 * NP * real;
}

template <typename Real, int T, int J, int V, int PD>
__global__ void __launch_bounds__(T, 1)
sweep_cluster_kernel(StateView sv, TraceView tr, uint2 key, uint32_t t0, int n_sweeps, int Nc)
{
    static_assert(J % V == 0, "J must be a multiple of the vector width");
    static_assert(PD == 0 || (sizeof(Real) == 4 && V >= 2), "pending sums exist only in the packed FP32C path");
    static_assert((T & (T - 1)) == 0, "T is a power of two");
    constexpr bool kPend = (PD != 0);
    using Coord = typename ModeT<Real>::Coord;
    using PackC = Pack<Coord, V>;
    constexpr bool kF32 = (sizeof(Real) == 4);
    constexpr bool kPacked = kF32 && V >= 2;
    constexpr int NP = T * J, G = J / V, nwarps = T >> 5, kSlot = MoveSlot<Real>::bytes;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cg::cluster_group cluster = cg::this_cluster();
    const unsigned C = cluster.num_blocks(), rank = cluster.block_rank();
    const int N = sv.N, ld = sv.ld;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int w = blockIdx.x / C;
    const int j0 = (int)rank * Nc;                                // first particle of this block's slice
    const int cnt = min(max(N - j0, 0), Nc);                      // particles in it

    double         *S     = reinterpret_cast<double *>(smem_raw);                              // [NP], permuted (s_index)
    unsigned char  *rnd   = smem_raw + NP * 8;                                                 // [2][kChunk] slots
    double         *part  = reinterpret_cast<double *>(smem_raw + NP * 8 + 2 * kChunk * kSlot);   // [2][32] warp totals
    double         *cpart = part + 64;                                                         // [2][kClusterMax] block totals (written by every block)
    unsigned long long *mvraw = reinterpret_cast<unsigned long long *>(cpart + 2 * kClusterMax);   // [2][4] moved particle (written by its owner)
    int32_t        *zw    = reinterpret_cast<int32_t *>(mvraw + 8);
    Coord          *x     = reinterpret_cast<Coord *>(zw + 4);                                 // [3][NP]
    Coord *y = x + NP, *z = x + 2 * NP;
    float *Shi = reinterpret_cast<float *>(S), *Slo = Shi + NP;

    const GroupDev g = sv.groups[sv.group_of[w]];
    SweepConst<Real> P;
    P.load(g);
    constexpr double kUnit = kPacked ? kT2Unit : 1.0, kInvUnit = 1.0 / kUnit;   // packed FP32C sums are in units of kT2Unit
    const double c2 = 2.0 * g.c1 * kUnit;
    const double step = kF32 ? g.step * g.inv_unit * 8388608.0 : g.step;
    const uint32_t wid = sv.walker_id_base + (uint32_t)w;

    // a1: this block's slice global -> shared, once per call
    Real *gpos = reinterpret_cast<Real *>(sv.pos) + (size_t)w * 3 * ld;
    double *gS = sv.S + (size_t)w * ld;
    for (int l = tid; l < NP; l += T) {
        Coord cx, cy, cz;
        double s = 0.0;
        if (l < cnt) {
            const int j = j0 + l;
            if constexpr (kF32) { cx = enc_coord(gpos[j]); cy = enc_coord(gpos[ld + j]); cz = enc_coord(gpos[2 * ld + j]); }
            else                { cx = gpos[j]; cy = gpos[ld + j]; cz = gpos[2 * ld + j]; }
            s = gS[j] * kInvUnit;
        } else {
            if constexpr (kF32) { cx = 0; cy = 0; cz = 0; }
            else                { cx = cy = cz = poison_of<Real>(Coord(0)); }
        }
        x[l] = cx; y[l] = cy; z[l] = cz;
        if constexpr (kPend) {
            const float hi = __double2float_rn(s);
            Shi[l] = hi;
            Slo[l] = __double2float_rn(s - (double)hi);
        } else {
            S[s_index<T, V>(l)] = s;
        }
    }
    // clamp bias of padding packs (FP32C; Nc % V == 0: whole packs are real or padding)
    float bias[G];
    f32x2 bias2[G];
#pragma unroll
    for (int gi = 0; gi < G; ++gi) {
        const bool real_pack = (gi * T + tid) * V < cnt;
        bias[gi] = real_pack ? 0.0f : 1.0f;
        bias2[gi] = real_pack ? pk2(0.0f, 0.0f) : pk2(0x1p63f, 0x1p63f);
    }

    const uint32_t total = (uint32_t)n_sweeps * (uint32_t)N;
    auto produce = [&](uint32_t chunk, int buf) {             // every block derives the same variates itself
        if (warp != 0) return;
        const uint32_t m = chunk * kChunk + lane;
        if (m >= total) return;
        const uint32_t q = m / (uint32_t)N;
        const uint32_t idx = m - q * (uint32_t)N;
        MoveRand<Real> mr;
        const uint4 r = philox4x32_10(make_uint4(idx, t0 + q, wid, 0u), key);
        mr.s = (int32_t)idx;
        const double ax = __dmul_rn(step, word_to_pm1(r.x));
        const double ay = __dmul_rn(step, word_to_pm1(r.y));
        const double az = __dmul_rn(step, word_to_pm1(r.z));
        if constexpr (kF32) {
            mr.dx = (int32_t)((uint32_t)__double2int_rn(ax) << 9);
            mr.dy = (int32_t)((uint32_t)__double2int_rn(ay) << 9);
            mr.dz = (int32_t)((uint32_t)__double2int_rn(az) << 9);
        } else {
            mr.dx = ax; mr.dy = ay; mr.dz = az;
        }
        mr.logxi = log(word_to_unit(r.w));
        *reinterpret_cast<MoveRand<Real> *>(rnd + (buf * kChunk + lane) * kSlot) = mr;
    };
    auto fetch = [&](uint32_t m) {
        return *reinterpret_cast<const MoveRand<Real> *>(rnd + ((int)((m >> 5) & 1) * kChunk + (int)(m & (kChunk - 1))) * kSlot);
    };
    // the thread that owns global particle s writes its coordinates into every block's slot `buf`
    auto push_particle = [&](int s, int buf) {
        const int r = s / Nc, l = s - r * Nc;
        if ((int)rank != r || (unsigned)tid != (((unsigned)l / (unsigned)V) & (unsigned)(T - 1))) return;
        unsigned long long vx, vy, vz;
        if constexpr (kF32) { vx = (uint32_t)x[l]; vy = (uint32_t)y[l]; vz = (uint32_t)z[l]; }
        else { vx = (unsigned long long)__double_as_longlong(x[l]); vy = (unsigned long long)__double_as_longlong(y[l]); vz = (unsigned long long)__double_as_longlong(z[l]); }
        for (unsigned q = 0; q < C; ++q) {
            unsigned long long *dst = cluster.map_shared_rank(mvraw, q) + buf * 4;
            dst[0] = vx; dst[1] = vy; dst[2] = vz;
        }
    };
    auto read_particle = [&](int buf, Coord &a, Coord &b, Coord &c) {
        const unsigned long long vx = mvraw[buf * 4], vy = mvraw[buf * 4 + 1], vz = mvraw[buf * 4 + 2];
        if constexpr (kF32) { a = (int32_t)(uint32_t)vx; b = (int32_t)(uint32_t)vy; c = (int32_t)(uint32_t)vz; }
        else { a = __longlong_as_double((long long)vx); b = __longlong_as_double((long long)vy); c = __longlong_as_double((long long)vz); }
    };

    produce(0, 0);
    if (tid == 0) *zw = 0;
    __syncthreads();
    push_particle(0, 0);
    cluster.sync();
    const int32_t zero = opaque_zero(zw);

    unsigned long long n_acc = 0;
    int s = 0;
    constexpr int kMoveUnroll = kF32 ? 4 : 1;                 // as in the one-block kernel (qmc_sweep_impl.cuh)
#pragma unroll kMoveUnroll
    for (uint32_t m = 0; m < total; ++m) {
        if ((m & (kChunk - 1)) == 0) produce((m >> 5) + 1, (int)(((m >> 5) + 1) & 1));
        const MoveRand<Real> mr = fetch(m);
        Coord xs, ys, zs;
        read_particle((int)(m & 1), xs, ys, zs);               // published by the previous move's cluster barrier
        const Coord tx = trial_coord(xs, mr.dx);
        const Coord ty = trial_coord(ys, mr.dy);
        const Coord tz = trial_coord(zs, mr.dz);
        const double logxi = mr.logxi;
        const int rs = s / Nc, ls = s - rs * Nc;
        const bool owner = ((int)rank == rs) && ((unsigned)tid == (((unsigned)ls / (unsigned)V) & (unsigned)(T - 1)));
        const int sn = (s + 1 == N) ? 0 : s + 1;
        push_particle(sn, (int)((m + 1) & 1));                 // next particle: untouched by this move (N >= 3)
        if (owner) x[ls] = poison_of<Real>(tx);                // self term = 0

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
        if (owner) {                                           // a4: sum_j t_new - S_s
            double Ss;
            if constexpr (kPend) Ss = (double)Shi[ls] + (double)Slo[ls];
            else                 Ss = S[s_index<T, V>(ls)];
            acc -= Ss;
        }

        // a5: block total (same bits in every thread of the block), then the C block totals through the cluster
        double tot = warp_sum(acc);
        double *pb = part + (int)(m & 1) * 32;
        if (lane == 0) pb[warp] = tot;
        __syncthreads();
        tot = sum_parts<nwarps>(pb);
        double *cb = cpart + (int)(m & 1) * kClusterMax;
        if ((unsigned)tid < C) cluster.map_shared_rank(cb, (unsigned)tid)[rank] = tot;
        cluster.sync();                                        // totals and the next particle are visible everywhere
        tot = cb[0];
        for (unsigned q = 1; q < C; ++q) tot += cb[q];         // same order in every thread of every block

        // a6: decision (Eq.(5), strict, log form: R8)
        const double margin = fma(c2, tot, -logxi);
        const bool accept = margin > 0.0;
        if (tr.dec != nullptr && rank == 0 && tid == 0 && w >= tr.w_begin && w < tr.w_end) {
            const long long k = tr.offset + m;
            if (k < tr.capacity) {
                const long long idx = (long long)(w - tr.w_begin) * tr.capacity + k;
                tr.dec[idx] = accept ? 1 : 0;
                if (tr.margin != nullptr) tr.margin[idx] = margin;
            }
        }

        // a7: commit and update the running pair sums of this block's slice
        if (accept) {
            if (kF32 && owner) x[ls] = poison_of<Real>(xs);
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
                    const double ns = (double)Shi[ls] + (double)Slo[ls] + tot;
                    const float hi = __double2float_rn(ns);
                    Shi[ls] = hi;
                    Slo[ls] = __double2float_rn(ns - (double)hi);
                } else {
                    S[s_index<T, V>(ls)] += tot;
                }
                x[ls] = commit_coord(tx, g.L);
                y[ls] = commit_coord(ty, g.L);
                z[ls] = commit_coord(tz, g.L);
            }
            ++n_acc;
        } else if (owner) {
            x[ls] = xs;                                        // undo the poison
        }
        if constexpr (kPend) {
            if ((m & (kFold - 1)) == kFold - 1) {               // renormalise this thread's sums: TwoSum(hi, lo)
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
        s = sn;
    }
    cluster.sync();                                            // nobody's shared memory goes away while it may still be written

    // a8: this block's slice shared -> global, once per call
    for (int l = tid; l < cnt; l += T) {
        const int j = j0 + l;
        if constexpr (kF32) { gpos[j] = dec_coord(x[l]); gpos[ld + j] = dec_coord(y[l]); gpos[2 * ld + j] = dec_coord(z[l]); }
        else                { gpos[j] = x[l]; gpos[ld + j] = y[l]; gpos[2 * ld + j] = z[l]; }
        if constexpr (kPend) gS[j] = ((double)Shi[l] + (double)Slo[l]) * kUnit;
        else                 gS[j] = S[s_index<T, V>(l)] * kUnit;
    }
    if (rank == 0 && tid == 0) sv.n_acc[w] += n_acc;
}

// ---- host side -----------------------------------------------------------------------------------------------------
struct ClusterShape {
    int T, J, V, P;
    cudaError_t (*launch)(qmc_ctx *c, int n_sweeps, int smem, int C, int Nc);
    int smem;
};

template <typename Real, int T, int J, int V, int PD>
static cudaError_t cluster_launch(qmc_ctx *c, int n_sweeps, int smem, int C, int Nc)
{
    const uint2 key = make_uint2((uint32_t)(c->seed & 0xFFFFFFFFull), (uint32_t)(c->seed >> 32));
    auto kern = sweep_cluster_kernel<Real, T, J, V, PD>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)c->W * (unsigned)C);
    cfg.blockDim = dim3(T);
    cfg.dynamicSmemBytes = (size_t)smem;
    cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, c->sv, c->trace, key, c->t, n_sweeps, Nc);
}

#define QMC_CLUSTER_ENTRY(Real, TT, JJ, VV, PP) {TT, JJ, VV, PP, cluster_launch<Real, TT, JJ, VV, PP>, \
                                                 sweep_cluster_smem_bytes(TT, JJ, sizeof(Real) == 8 ? QMC_FP64 : QMC_FP32C)},

const ClusterShape *cluster_shapes_f32(int *n);
const ClusterShape *cluster_shapes_f64(int *n);

}  // namespace qmc
