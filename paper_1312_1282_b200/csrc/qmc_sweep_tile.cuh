// qmc_sweep_tile.cuh -- the FP32C Metropolis sweep in TILES of K consecutive moves (SURVEY.md §8(a) rows a1-a8,
// §7 hard part (ii); VERDICT r1 "next" #2).  Oracle-green but slower than the one-move kernel (profiles/r02_tile.md,
// DESIGN.md §6): selectable with qmc_set_tuning("sweep_tile", K), never the planner's choice.
//
// The one-move-at-a-time kernel (qmc_sweep_impl.cuh) pays, per move, one block reduction, one barrier and the
// decision chain (the paper fought the same term with warp-synchronous code and a
// prefetched xi).  With particles moved in order (R7), the K moves s0 .. s0+K-1 of a tile touch K DISTINCT particles,
// so their trial sums against every particle OUTSIDE the tile do not depend on each other's outcome:
//
//   pass 1   every thread evaluates, for each particle j it owns (coordinates read ONCE per tile), the K trial terms
//            t(|r'_i - r_j|), i < K, and keeps them in registers; the K tile particles themselves are left out
//            (their owner forces the clamp on that pack: the terms are exactly 0);
//   intra    the 2 K (K-1) pair terms among the tile's own old and trial positions -- t(r'_i, r_i'), t(r'_i, r'_i'),
//            t(r_i, r_i') -- are evaluated once by the lanes of one warp and published in shared memory;
//   reduce   K block sums behind ONE barrier: a butterfly that halves the number of values per stage
//            (12 shuffles for K = 4 instead of 40), one shared-memory exchange;
//   resolve  every thread takes the K decisions IN ORDER on identical bits: move i sees the tile particles i' < i
//            where their decisions left them (trial or old position) and its own running sum S_i corrected for the
//            accepted ones -- exactly the sequential Metropolis chain (Eq.(5) l.123, Eq.(7) l.146); only the
//            summation order of Delta differs from the one-move kernel (R12);
//   commit   for each accepted move, in order, every thread re-evaluates the OLD terms of its own particles and
//            adds t_new - t_old to its own S_j (hi + lo representation, R20); the owner of the tile's pack
//            updates the K tile particles' sums from the intra-tile terms and writes their coordinates.
//
// Ownership is static (particle j belongs to thread (j / V) mod T), so S and the pair loops need no
// synchronisation, and the tile's particles -- K consecutive indices, K | V -- sit in ONE pack of ONE thread.
// Requirements (the planner falls back to the one-move kernel otherwise): FP32C, proposal 0, N % K == 0, N >= 2 K.
#pragma once
#include "qmc_sweep_impl.cuh"

namespace qmc {

// K values per lane -> block-wide: after the call, lanes with (lane % (32/K)) == 0 hold the warp total of move
// lane / (32/K).  Every stage adds a lane's value to its partner's: identical bits in all lanes of a group.
template <int K>
__device__ __forceinline__ double warp_sum_multi(const double (&v)[K], int lane)
{
    static_assert(K == 1 || K == 2 || K == 4, "tile size");
    double b;
    if (K == 4) {
        const bool up = (lane & 16) != 0;
        const double k0 = up ? v[2] : v[0], k1 = up ? v[3] : v[1];
        const double s0 = up ? v[0] : v[2], s1 = up ? v[1] : v[3];
        const double a0 = k0 + __shfl_xor_sync(0xffffffffu, s0, 16);
        const double a1 = k1 + __shfl_xor_sync(0xffffffffu, s1, 16);
        const bool u8 = (lane & 8) != 0;
        b = (u8 ? a1 : a0) + __shfl_xor_sync(0xffffffffu, u8 ? a0 : a1, 8);
        b += __shfl_xor_sync(0xffffffffu, b, 4);
    } else if (K == 2) {
        const bool up = (lane & 16) != 0;
        b = (up ? v[1] : v[0]) + __shfl_xor_sync(0xffffffffu, up ? v[0] : v[1], 16);
        b += __shfl_xor_sync(0xffffffffu, b, 8);
        b += __shfl_xor_sync(0xffffffffu, b, 4);
    } else {
        b = v[0] + __shfl_xor_sync(0xffffffffu, v[0], 16);
        b += __shfl_xor_sync(0xffffffffu, b, 8);
        b += __shfl_xor_sync(0xffffffffu, b, 4);
    }
    b += __shfl_xor_sync(0xffffffffu, b, 2);
    b += __shfl_xor_sync(0xffffffffu, b, 1);
    return b;
}

// Index of the intra-tile terms: unordered pair q = (i, i') with i > i' at q = i (i-1) / 2 + i'; four terms each.
//   TT: t(r'_i, r'_i')    OO: t(r_i, r_i')    TO(i,i'): t(r'_i, r_i')    TO(i',i): t(r'_i', r_i) = t(r_i, r'_i')
__host__ __device__ constexpr int tq(int i, int ip) { return i > ip ? i * (i - 1) / 2 + ip : ip * (ip - 1) / 2 + i; }
__host__ __device__ constexpr int iTT(int i, int ip) { return 4 * tq(i, ip); }
__host__ __device__ constexpr int iOO(int i, int ip) { return 4 * tq(i, ip) + 1; }
__host__ __device__ constexpr int iTO(int i, int ip) { return 4 * tq(i, ip) + (i > ip ? 2 : 3); }   // trial of i, old of i'

// bytes of shared memory: S as hi + lo [NP] floats each, variate ring (SoA, 2 x 32 moves), block-sum exchange
// [2][K][32] doubles, intra-tile terms [2][32] floats, opaque zero, coordinates [3][NP]
static inline int sweep_tile_smem_bytes(int T, int J, int K)
{
    const int NP = T * J;
    return NP * 8 + 2 * kChunk * 20 + 2 * K * 32 * 8 + 2 * 32 * 4 + 16 + 3 * NP * 4;
}

template <int T, int J, int K>
constexpr int sweep_tile_min_ctas()
{
    const int smem = J * T * 20 + 2 * kChunk * 20 + 2 * K * 32 * 8 + 256 + 16 + 1024;
    const int by_smem = (228 * 1024) / smem;
    const int regs = 64 + K * J + 3 * K;                 // retained trial terms dominate
    const int by_regs = 65536 / (regs * T);
    int n = by_smem < by_regs ? by_smem : by_regs;
    return n < 1 ? 1 : (n > 32 ? 32 : n);
}

template <int T, int J, int V, int K>
__global__ void __launch_bounds__(T, (sweep_tile_min_ctas<T, J, K>()))
sweep_tile_kernel(StateView sv, TraceView tr, WriteoutView wo, uint2 key, uint32_t t0, int n_sweeps)
{
    static_assert(V == 2 || V == 4, "packed FP32C path");
    static_assert(K == 2 || K == 4, "tile size");
    static_assert(J % V == 0 && V % K == 0, "a tile is K consecutive particles inside one pack");
    static_assert((T & (T - 1)) == 0, "T is a power of two");
    using PackC = Pack<int32_t, V>;
    using PackF = Pack<float, V>;
    constexpr int NP = T * J, G = J / V, nwarps = T >> 5, HP = V / 2;      // HP: f32x2 pairs per pack
    constexpr int NC = 2 * K * (K - 1);                                      // intra-tile terms
    constexpr int LPG = 32 / K;                                              // lanes per move group after the reduction
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = sv.N, ld = sv.ld;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int w = blockIdx.x;

    float   *Shi  = reinterpret_cast<float *>(smem_raw);                    // [NP]
    float   *Slo  = Shi + NP;                                               // [NP]
    double  *rlog = reinterpret_cast<double *>(smem_raw + NP * 8);          // [2][32] log xi
    int32_t *rdx  = reinterpret_cast<int32_t *>(rlog + 2 * kChunk);         // [2][32] each
    int32_t *rdy = rdx + 2 * kChunk, *rdz = rdy + 2 * kChunk;
    double  *part = reinterpret_cast<double *>(rdz + 2 * kChunk);           // [2][K][32]
    float   *corr = reinterpret_cast<float *>(part + 2 * K * 32);           // [2][32]
    int32_t *zw   = reinterpret_cast<int32_t *>(corr + 64);                 // opaque zero (+ padding to 16 bytes)
    int32_t *x    = zw + 4;                                                 // [3][NP]
    int32_t *y = x + NP, *z = x + 2 * NP;

    const GroupDev g = sv.groups[sv.group_of[w]];
    const double c2 = 2.0 * g.c1 * kT2Unit;                // 2 Delta = c2 * (sum t_new - S_s), sums in units of kT2Unit (pair_t2)
    const double step = g.step * g.inv_unit * 8388608.0;   // proposal half-width in grid units (2^-23 box)
    const uint32_t wid = sv.walker_id_base + (uint32_t)w;

    // a1: walker state global -> shared, once per call
    float *gpos = reinterpret_cast<float *>(sv.pos) + (size_t)w * 3 * ld;
    double *gS = sv.S + (size_t)w * ld;
    for (int j = tid; j < NP; j += T) {
        int32_t cx = 0, cy = 0, cz = 0;
        double s = 0.0;
        if (j < N) {
            cx = enc_coord(gpos[j]); cy = enc_coord(gpos[ld + j]); cz = enc_coord(gpos[2 * ld + j]);
            s = gS[j] * (1.0 / kT2Unit);
        }
        x[j] = cx; y[j] = cy; z[j] = cz;
        const float hi = __double2float_rn(s);
        Shi[j] = hi;
        Slo[j] = __double2float_rn(s - (double)hi);
    }
    // clamp bias of this thread's packs: 2^63 for padding packs (N % V == 0: whole packs are real or padding)
    f32x2 bias2[G];
#pragma unroll
    for (int gi = 0; gi < G; ++gi) bias2[gi] = ((gi * T + tid) * V < N) ? pk2(0.0f, 0.0f) : pk2(0x1p63f, 0x1p63f);

    const uint32_t total = (uint32_t)n_sweeps * (uint32_t)N;

    // a2: variates of moves [chunk*32, chunk*32+32) -> ring buffer `buf`
    auto produce = [&](uint32_t chunk, int buf) {
        if (warp != 0) return;
        const uint32_t m = chunk * kChunk + lane;
        if (m >= total) return;
        const uint32_t q = m / (uint32_t)N;
        const uint32_t idx = m - q * (uint32_t)N;
        const uint4 r = philox4x32_10(make_uint4(idx, t0 + q, wid, 0u), key);
        const int o = buf * kChunk + lane;
        rdx[o] = (int32_t)((uint32_t)__double2int_rn(__dmul_rn(step, word_to_pm1(r.x))) << 9);
        rdy[o] = (int32_t)((uint32_t)__double2int_rn(__dmul_rn(step, word_to_pm1(r.y))) << 9);
        rdz[o] = (int32_t)((uint32_t)__double2int_rn(__dmul_rn(step, word_to_pm1(r.z))) << 9);
        rlog[o] = log(word_to_unit(r.w));
    };
    produce(0, 0);
    if (tid == 0) *zw = 0;
    __syncthreads();
    const int32_t zero = opaque_zero(zw);

    unsigned long long n_acc = 0;
    int s0 = 0;                                            // first particle of the tile
    uint32_t sweeps_done = 0;
    for (uint32_t m0 = 0; m0 < total; m0 += K) {
        const uint32_t tile = m0 / K;
        const int buf = (int)(tile & 1);
        if ((m0 & (kChunk - 1)) == 0) produce((m0 >> 5) + 1, (int)(((m0 >> 5) + 1) & 1));
        // old and trial coordinates of the tile's particles (last written a sweep ago: no hazard), log xi
        int32_t xo[K], yo[K], zo[K], tx[K], ty[K], tz[K];
        double logxi[K];
        {
            const int r0 = (int)(m0 & (kChunk - 1)) + ((int)((m0 >> 5) & 1)) * kChunk;
            const Pack<int32_t, K> X0 = *reinterpret_cast<const Pack<int32_t, K> *>(x + s0);
            const Pack<int32_t, K> Y0 = *reinterpret_cast<const Pack<int32_t, K> *>(y + s0);
            const Pack<int32_t, K> Z0 = *reinterpret_cast<const Pack<int32_t, K> *>(z + s0);
            const Pack<int32_t, K> DX = *reinterpret_cast<const Pack<int32_t, K> *>(rdx + r0);
            const Pack<int32_t, K> DY = *reinterpret_cast<const Pack<int32_t, K> *>(rdy + r0);
            const Pack<int32_t, K> DZ = *reinterpret_cast<const Pack<int32_t, K> *>(rdz + r0);
#pragma unroll
            for (int i = 0; i < K; ++i) {
                xo[i] = X0.v[i]; yo[i] = Y0.v[i]; zo[i] = Z0.v[i];
                tx[i] = wadd(xo[i], DX.v[i]); ty[i] = wadd(yo[i], DY.v[i]); tz[i] = wadd(zo[i], DZ.v[i]);
                logxi[i] = rlog[r0 + i];
            }
        }
        // the thread that owns the tile's pack, and where the tile sits in it
        const unsigned pk = (unsigned)s0 / (unsigned)V;
        const bool owner = (unsigned)tid == (pk & (unsigned)(T - 1));
        const int g_o = owner ? (int)(pk / (unsigned)T) : -1;
        const int h_o = (s0 & (V - 1)) >> 1;                  // first f32x2 pair of the tile inside the pack (K = 2)

        // intra-tile terms, one per lane of one warp (old coordinates are still in shared memory: the owner
        // commits after this tile's barrier)
        if (K > 1 && warp == (int)(tile & (nwarps - 1)) && lane < NC) {
            const int q = lane >> 2, kind = lane & 3;
            const int i = (q >= 3) ? 3 : ((q >= 1) ? 2 : 1);      // q = i (i-1)/2 + i'
            const int ip = q - i * (i - 1) / 2;
            const int ia = (kind == 3) ? ip : i, ib = (kind == 3) ? i : ip;      // a: first point, b: second
            const bool ta = (kind != 1), tb = (kind == 0);                       // trial (else old) position
            const int ra = (int)(m0 & (kChunk - 1)) + ((int)((m0 >> 5) & 1)) * kChunk + ia;
            const int rb = (int)(m0 & (kChunk - 1)) + ((int)((m0 >> 5) & 1)) * kChunk + ib;
            int32_t ax = x[s0 + ia], ay = y[s0 + ia], az = z[s0 + ia];
            int32_t bx = x[s0 + ib], by = y[s0 + ib], bz = z[s0 + ib];
            if (ta) { ax = wadd(ax, rdx[ra]); ay = wadd(ay, rdy[ra]); az = wadd(az, rdz[ra]); }
            if (tb) { bx = wadd(bx, rdx[rb]); by = wadd(by, rdy[rb]); bz = wadd(bz, rdz[rb]); }
            const SweepConst<float> P0{};
            corr[buf * 32 + lane] = pair_t(ax, ay, az, bx, by, bz, 0.0f, P0) * (float)(1.0 / kT2Unit);
        }

        int s0n = s0 + K;
        if (s0n >= N) s0n = 0;

        // pass 1 (a3): K trial terms per owned particle, coordinates read once
        f32x2 un2[K][J / 2];
        f32x2 acc2[K];
#pragma unroll
        for (int i = 0; i < K; ++i) acc2[i] = pk2(0.0f, 0.0f);
#pragma unroll
        for (int gi = 0; gi < G; ++gi) {
            const int base = (gi * T + tid) * V;
            const PackC X = *reinterpret_cast<const PackC *>(x + base);
            const PackC Y = *reinterpret_cast<const PackC *>(y + base);
            const PackC Z = *reinterpret_cast<const PackC *>(z + base);
#pragma unroll
            for (int c = 0; c < HP; ++c) {
                const bool mine = (gi == g_o) && (K == V || c == h_o);      // the tile's own particles: clamp -> 0
                const f32x2 be = mine ? pk2(0x1p63f, 0x1p63f) : bias2[gi];
#pragma unroll
                for (int i = 0; i < K; ++i) {
                    const f32x2 t2 = pair_t2(tx[i], ty[i], tz[i], X.v[2 * c], X.v[2 * c + 1], Y.v[2 * c], Y.v[2 * c + 1],
                                             Z.v[2 * c], Z.v[2 * c + 1], be, zero);
                    un2[i][gi * HP + c] = t2;
                    acc2[i] = add2(acc2[i], t2);
                }
            }
        }
        double acc[K];
#pragma unroll
        for (int i = 0; i < K; ++i) acc[i] = (double)hsum2(acc2[i]);
        double S0[K];                                              // owner: running sums of the tile's particles
        if (owner) {                                               // a4: sum_j t_new - S_s
#pragma unroll
            for (int i = 0; i < K; ++i) {
                S0[i] = (double)Shi[s0 + i] + (double)Slo[s0 + i];
                acc[i] -= S0[i];
            }
        }

        // a5: K block sums, identical bits in every thread
        {
            const double tot = warp_sum_multi<K>(acc, lane);
            double *pb = part + buf * K * 32;
            if ((lane & (LPG - 1)) == 0) pb[(lane / LPG) * 32 + warp] = tot;
        }
        if (nwarps > 1) __syncthreads(); else __syncwarp();
        double tot[K];
#pragma unroll
        for (int i = 0; i < K; ++i) tot[i] = sum_parts<nwarps>(part + buf * K * 32 + i * 32);
        float ct[NC > 0 ? NC : 1];
        if (K > 1) {
#pragma unroll
            for (int k4 = 0; k4 < NC; k4 += 4) {
                const float4 v4 = *reinterpret_cast<const float4 *>(corr + buf * 32 + k4);
                ct[k4] = v4.x; ct[k4 + 1] = v4.y; ct[k4 + 2] = v4.z; ct[k4 + 3] = v4.w;
            }
        }

        // a6: the K decisions in order (Eq.(5), strict, log form: R8)
        bool accept[K];
        double margin[K];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            float c = 0.0f;                     // tile particles as move i finds them, minus the change of S_i so far
#pragma unroll
            for (int ip = 0; ip < K; ++ip) {
                if (ip == i) continue;
                if (ip < i) {
                    const float seen = accept[ip] ? ct[iTT(i, ip)] : ct[iTO(i, ip)];
                    const float dS = accept[ip] ? ct[iTO(ip, i)] - ct[iOO(i, ip)] : 0.0f;
                    c += seen - dS;
                } else {
                    c += ct[iTO(i, ip)];
                }
            }
            tot[i] += (double)c;
            margin[i] = fma(c2, tot[i], -logxi[i]);
            accept[i] = margin[i] > 0.0;
        }
        if (tr.dec != nullptr && tid == 0 && w >= tr.w_begin && w < tr.w_end) {
#pragma unroll
            for (int i = 0; i < K; ++i) {
                const long long k = tr.offset + m0 + i;
                if (k < tr.capacity) {
                    const long long idx = (long long)(w - tr.w_begin) * tr.capacity + k;
                    tr.dec[idx] = accept[i] ? 1 : 0;
                    if (tr.margin != nullptr) tr.margin[idx] = margin[i];
                }
            }
        }
        bool any = false;
#pragma unroll
        for (int i = 0; i < K; ++i) { any = any || accept[i]; n_acc += accept[i] ? 1 : 0; }

        // a7: running pair sums of the particles outside the tile, S_j += t_new - t_old per accepted move
        if (any) {
#pragma unroll
            for (int gi = 0; gi < G; ++gi) {
                const int base = (gi * T + tid) * V;
                const PackC X = *reinterpret_cast<const PackC *>(x + base);
                const PackC Y = *reinterpret_cast<const PackC *>(y + base);
                const PackC Z = *reinterpret_cast<const PackC *>(z + base);
                PackF pd = *reinterpret_cast<const PackF *>(Slo + base);
#pragma unroll
                for (int c = 0; c < HP; ++c) {
                    const bool mine = (gi == g_o) && (K == V || c == h_o);
                    const f32x2 be = mine ? pk2(0x1p63f, 0x1p63f) : bias2[gi];
                    f32x2 nw = pk2(pd.v[2 * c], pd.v[2 * c + 1]);
#pragma unroll
                    for (int i = 0; i < K; ++i) {
                        if (accept[i]) {
                            const f32x2 to2 = pair_t2(xo[i], yo[i], zo[i], X.v[2 * c], X.v[2 * c + 1], Y.v[2 * c], Y.v[2 * c + 1],
                                                      Z.v[2 * c], Z.v[2 * c + 1], be, zero);
                            nw = add2(nw, sub2(un2[i][gi * HP + c], to2));
                        }
                    }
                    upk2(nw, pd.v[2 * c], pd.v[2 * c + 1]);
                }
                *reinterpret_cast<PackF *>(Slo + base) = pd;
            }
            // the tile's own particles: sums from the intra-tile terms, coordinates
            if (owner) {
#pragma unroll
                for (int i = 0; i < K; ++i) {
                    if (!accept[i]) continue;
#pragma unroll
                    for (int p = 0; p < K; ++p) {
                        if (p == i) continue;
                        float d;
                        if (p < i) d = accept[p] ? ct[iTT(i, p)] - ct[iTO(p, i)] : ct[iTO(i, p)] - ct[iOO(i, p)];
                        else       d = ct[iTO(i, p)] - ct[iOO(i, p)];
                        S0[p] += (double)d;
                    }
                    S0[i] += tot[i];
                }
#pragma unroll
                for (int i = 0; i < K; ++i) {
                    const float hi = __double2float_rn(S0[i]);
                    Shi[s0 + i] = hi;
                    Slo[s0 + i] = __double2float_rn(S0[i] - (double)hi);
                    if (accept[i]) { x[s0 + i] = tx[i]; y[s0 + i] = ty[i]; z[s0 + i] = tz[i]; }
                }
            }
        }
        // renormalise this thread's sums every kFold moves: TwoSum(hi, lo) (R20)
        if (((m0 + K) & (kFold - 1)) == 0) {
#pragma unroll
            for (int gi = 0; gi < G; ++gi) {
                const int base = (gi * T + tid) * V;
                PackF ph = *reinterpret_cast<const PackF *>(Shi + base);
                PackF pl = *reinterpret_cast<const PackF *>(Slo + base);
#pragma unroll
                for (int c = 0; c < HP; ++c) {
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
        // end of a sweep: optional in-kernel write-out (NEXT-4)
        if (s0n == 0) {
            ++sweeps_done;
            if (wo.xyz != nullptr && wo.every > 0 && sweeps_done % (uint32_t)wo.every == 0) {
                const int slot = (int)(sweeps_done / (uint32_t)wo.every) - 1;
                if (slot < wo.n_out) writeout_walker<T>(wo, slot, w, sv.W, N, g.L_A, x, y, z, sv.n_acc[w] + n_acc);
            }
        }
        s0 = s0n;
    }
    __syncthreads();

    // a8: shared -> global, once per call
    for (int j = tid; j < N; j += T) {
        gpos[j] = dec_coord(x[j]); gpos[ld + j] = dec_coord(y[j]); gpos[2 * ld + j] = dec_coord(z[j]);
        gS[j] = ((double)Shi[j] + (double)Slo[j]) * kT2Unit;
    }
    if (tid == 0) sv.n_acc[w] += n_acc;
}

}  // namespace qmc
