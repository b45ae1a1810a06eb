// qmc_energy_f32.cu -- FP32C local-energy estimator over all pairs and the
// from-scratch rebuild of the running pair sums S_i (R17).
//
// One CTA per walker; coordinates in shared memory as 32-bit fixed point (qmc_f32c.cuh), so the signed
// minimum image of a pair is ONE wrapping integer subtraction.  The particles are cut into blocks of 32.
// A warp owns an i-block (lane = particle i; grad_i log psi, lap_i log psi, S_i and V stay in registers --
// the scatter-free layout of PAPER.md l.527's "extra memory to store wavefunction derivatives") and
// streams the j-blocks from shared memory (every lane reads the same j: broadcast).  Two j per
// instruction: all pair arithmetic is packed f32x2.
//
//   G_i      = sum_{j != i} u'(r_ij) d_ij / r_ij,     u'/r = 5/2 b^5 y (y^6 - z^6)
//   Lambda_i = sum_{j != i} [u'' + 2 u'/r]                 = -5 b^5 (2 y^7 + 3 z^7 + z^6 y)
//   V        = sum_{i<j, r<h} V_Aziz(r_ij)                 (HFD-B(HE), truncated at h, R3)
//   T_PB = -Dk sum_i (Lambda_i + |G_i|^2),  T_JF = -Dk/2 sum_i Lambda_i,  E_PB = V + T_PB      (R14)
// with y = 1/r, z = 1/(L-r), box units (L = 1, h = 1/2).
//
// No per-pair cutoff test.  r^2 is CLAMPED to h^2, where y = z = 2 exactly, so a pair at or beyond the
// cutoff contributes exactly 0 to S_i and G_i, and exactly the constants K_L = 768 (lap term / 5 b^5; 6 in the kernel's units, qmc_energy_f32_pair.cuh) and
// K_V = V(h) to the other two sums; the kernel counts the pairs inside the cutoff (one integer compare) and
// removes (pairs - inside) K afterwards in fp64.  Only the j-block that contains the warp's own particles
// (self pair, V for j > i only) and a ragged last block take a slower tile with explicit selects.
// V is evaluated only in tiles with j-block > i-block (+ the diagonal tile), i.e. once per unordered pair.
//
// R20: per-pair terms are fp32; 16 consecutive j are summed in fp32 (two packed lanes of 8) and then added
// to fp64 accumulators.
#include <cstdarg>
#include <cstring>
#include <mutex>

#include "qmc_energy_f32_pair.cuh"

namespace qmc {

namespace {

using namespace e32;

struct Acc32 { f32x2 gx, gy, gz, lam, s, v; };
struct Acc64 { double gx, gy, gz, lam, lamd, s, v; };   // lam: tiles above the diagonal (counted twice), lamd: diagonal tile

// 16 consecutive j (4 vector loads per coordinate) against this lane's particle.
//   kSlow: per-pair selects (self pair, j >= N, V only for j > i); kV: evaluate the potential and the
//   Laplacian term (both are symmetric in i,j and only their totals are needed: tiles below the diagonal skip them).
// Sums kept here: gm = y^7 - z^6 y = (u'/r) / (5/2 b^5);  lt = 2 y^7 + 3 z^7 + z^6 y = -(u'' + 2u'/r) / (5 b^5).
template <bool kEnergy, bool kV, bool kSlow, bool kGlobal = false>
__device__ __forceinline__ void tile16(const int32_t *__restrict__ x, const int32_t *__restrict__ y, const int32_t *__restrict__ z,
                                       int j0, int i, int N, int32_t xi, int32_t yi, int32_t zi, const AzizF32 &E,
                                       int32_t zero, Acc64 &A, double &lam_acc, int &n_in)
{
    Acc32 P;
    P.gx = P.gy = P.gz = P.lam = P.s = P.v = pk1(0.0f);
#pragma unroll 4
    for (int g = 0; g < 4; ++g) {
        // kGlobal: the coordinates stream from global memory through the read-only path (all lanes read the same
        // address; the L1 serves the other warps of the block)
        const int4 X = kGlobal ? __ldg(reinterpret_cast<const int4 *>(x + j0 + 4 * g)) : *reinterpret_cast<const int4 *>(x + j0 + 4 * g);
        const int4 Y = kGlobal ? __ldg(reinterpret_cast<const int4 *>(y + j0 + 4 * g)) : *reinterpret_cast<const int4 *>(y + j0 + 4 * g);
        const int4 Z = kGlobal ? __ldg(reinterpret_cast<const int4 *>(z + j0 + 4 * g)) : *reinterpret_cast<const int4 *>(z + j0 + 4 * g);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int ja = j0 + 4 * g + 2 * h, jb = ja + 1;
            f32x2 bias2 = pk1(0.0f);
            if (kSlow) bias2 = pk2((ja == i || ja >= N) ? 0x1p63f : 0.0f, (jb == i || jb >= N) ? 0x1p63f : 0.0f);
            const Pair2 p = h == 0 ? pair_geom(xi, yi, zi, X.x, X.y, Y.x, Y.y, Z.x, Z.y, bias2, zero)
                                   : pair_geom(xi, yi, zi, X.z, X.w, Y.z, Y.w, Z.z, Z.w, bias2, zero);
            const bool ina = __float_as_int(p.a) < kClampBits, inb = __float_as_int(p.b) < kClampBits;
            P.s = add2(P.s, pair_t(p));
            if (kEnergy) {
                const f32x2 y6 = mul2(p.y4, p.y2), z6 = mul2(p.z4, p.z2);
                const f32x2 y7 = mul2(y6, p.y), z6y = mul2(z6, p.y);
                const f32x2 z7 = kV ? mul2(z6, p.z) : z6;
                const f32x2 gm = sub2(y7, z6y);
                P.gx = fma2(gm, p.mx, P.gx);
                P.gy = fma2(gm, p.my, P.gy);
                P.gz = fma2(gm, p.mz, P.gz);
                if (kV) {
                    f32x2 lt = fma2(y7, pk1(2.0f), fma2(z7, pk1(3.0f), z6y));
                    if (kSlow) {
                        float la, lb;
                        upk2(lt, la, lb);
                        lt = pk2(ina ? la : 0.0f, inb ? lb : 0.0f);
                    } else {
                        n_in += (ina ? 1 : 0) + (inb ? 1 : 0);
                    }
                    P.lam = add2(P.lam, lt);
                    f32x2 vp = aziz2(p, E);
                    if (kSlow) {
                        float va, vb;
                        upk2(vp, va, vb);
                        vp = pk2((ina && ja > i) ? va : 0.0f, (inb && jb > i) ? vb : 0.0f);
                    }
                    P.v = add2(P.v, vp);
                }
            }
        }
    }
    A.s += (double)hsum2(P.s);
    if (kEnergy) {
        A.gx += (double)hsum2(P.gx);
        A.gy += (double)hsum2(P.gy);
        A.gz += (double)hsum2(P.gz);
        if (kV) {
            lam_acc += (double)hsum2(P.lam);
            A.v += (double)hsum2(P.v);
        }
    }
}

template <int T, bool kEnergy>
__global__ void __launch_bounds__(T, (T <= 128 ? 4 : (T <= 256 ? 2 : 1)))
energy32_kernel(StateView sv, double Dk, double *__restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = sv.N, ld = sv.ld;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int nwarps = T >> 5;
    const int w = blockIdx.x;
    const int nblk = (N + 31) >> 5, NP = nblk << 5;

    double  *red = reinterpret_cast<double *>(smem_raw);              // [3][32]
    int32_t *x   = reinterpret_cast<int32_t *>(red + 96);             // [3][NP]
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
    }
    if (tid == 0) *reinterpret_cast<int32_t *>(red + 95) = 0;
    __syncthreads();
    const int32_t zero = opaque_zero(reinterpret_cast<int32_t *>(red + 95));

    // V of a clamped pair, by the same instructions every clamped pair goes through
    float KV = 0.0f;
    if (kEnergy) {
        const Pair2 pc = pair_geom(0, 0, 0, 0, 0, 0, 0, 0, 0, pk1(0x1p63f), zero);
        float va, vb;
        upk2(aziz2(pc, E), va, vb);
        KV = va;
    }

    const bool ragged = (N & 31) != 0;
    double tLam = 0.0, tG2 = 0.0, tV = 0.0;
    for (int A = warp; A < nblk; A += nwarps) {
        const int i = (A << 5) + lane;
        const bool live = i < N;
        const int ic = live ? i : N - 1;
        const int32_t xi = x[ic], yi = y[ic], zi = z[ic];
        Acc64 acc = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        int n_hi = 0, fast_hi = 0, n_none = 0;                 // inside-cutoff pairs / fast tiles above A
        for (int B = 0; B < nblk; ++B) {
            const int j0 = B << 5;
            if (B == A || (ragged && B == nblk - 1)) {
                double &la = (B == A) ? acc.lamd : acc.lam;
                tile16<kEnergy, true, true>(x, y, z, j0, ic, N, xi, yi, zi, E, zero, acc, la, n_none);
                tile16<kEnergy, true, true>(x, y, z, j0 + 16, ic, N, xi, yi, zi, E, zero, acc, la, n_none);
            } else if (B > A) {
                tile16<kEnergy, true, false>(x, y, z, j0, ic, N, xi, yi, zi, E, zero, acc, acc.lam, n_hi);
                tile16<kEnergy, true, false>(x, y, z, j0 + 16, ic, N, xi, yi, zi, E, zero, acc, acc.lam, n_hi);
                ++fast_hi;
            } else {
                tile16<kEnergy, false, false>(x, y, z, j0, ic, N, xi, yi, zi, E, zero, acc, acc.lam, n_none);
                tile16<kEnergy, false, false>(x, y, z, j0 + 16, ic, N, xi, yi, zi, E, zero, acc, acc.lam, n_none);
            }
        }
        if (live) {
            sv.S[(size_t)w * ld + i] = acc.s * kSUnit;                 // R17: rebuild the running sum
            if (kEnergy) {
                const double out_hi = (double)(32 * fast_hi - n_hi);
                tLam += 2.0 * (acc.lam - kLamClamp * out_hi) + acc.lamd;
                tG2 += acc.gx * acc.gx + acc.gy * acc.gy + acc.gz * acc.gz;
                tV += acc.v - (double)KV * out_hi;
            }
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
                // box units -> Angstrom: gradients per box edge; the minimum image carried a factor 2^32
                const double Dku = Dk * g.inv_unit * g.inv_unit;
                const double lam = -5.0 * g.b5 * kGUnit * a;                            // sum_i Lambda_i
                const double g2 = (2.5 * g.b5 * kGUnit * 0x1p-32) * (2.5 * g.b5 * kGUnit * 0x1p-32) * b;   // sum_i |G_i|^2
                const double T_PB = -Dku * (lam + g2);
                const double T_JF = -0.5 * Dku * lam;
                double *o = out + (size_t)w * 4;
                const double V = c * g.az.f32_scale;                                     // the potential was summed in units of f32_scale K
                o[0] = V + T_PB; o[1] = V; o[2] = T_PB; o[3] = T_JF;
            }
        }
    }
}

// ---- gridded variant (energy_plan.variant 3): any N, and one walker on many SMs --------------
// The walker's fixed-point coordinates sit in GLOBAL memory ([W][3][NP] int32, written by encode_kernel) and stream
// through L1/L2 as broadcast 16-byte reads; block (w, part) of the grid takes the i-blocks A = part*nwarps + warp,
// + nparts*nwarps, ... of walker w with the same tiles as energy32_kernel, writes their S_i and its three partial
// sums; finalize_kernel adds the parts of a walker in a fixed order (deterministic) and forms the energies.
__global__ void encode_kernel(StateView sv, int32_t *__restrict__ enc, int NP)
{
    const int w = blockIdx.x;
    const int j = blockIdx.y * blockDim.x + threadIdx.x;
    if (j >= NP) return;
    const float *gpos = reinterpret_cast<const float *>(sv.pos) + (size_t)w * 3 * sv.ld;
    const bool in = j < sv.N;
    int32_t *e = enc + (size_t)w * 3 * NP;
    e[j] = in ? enc_coord(gpos[j]) : 0;
    e[NP + j] = in ? enc_coord(gpos[sv.ld + j]) : 0;
    e[2 * NP + j] = in ? enc_coord(gpos[2 * sv.ld + j]) : 0;
}

template <int T, bool kEnergy>
__global__ void __launch_bounds__(T, (T <= 128 ? 4 : 2))
energy32g_kernel(StateView sv, const int32_t *__restrict__ enc, int NP, int nparts, double *__restrict__ partial)
{
    __shared__ double red[96];
    __shared__ int32_t zw[4];
    const int N = sv.N, ld = sv.ld;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int nwarps = T >> 5;
    const int w = blockIdx.x / nparts, part = blockIdx.x - w * nparts;
    const int nblk = NP >> 5;
    const int32_t *x = enc + (size_t)w * 3 * NP, *y = x + NP, *z = x + 2 * NP;

    const GroupDev g = sv.groups[sv.group_of[w]];
    AzizF32 E;
    E.load(g.az);
    if (tid == 0) zw[0] = 0;
    __syncthreads();
    const int32_t zero = opaque_zero(zw);
    float KV = 0.0f;
    if (kEnergy) {
        const Pair2 pc = pair_geom(0, 0, 0, 0, 0, 0, 0, 0, 0, pk1(0x1p63f), zero);
        float va, vb;
        upk2(aziz2(pc, E), va, vb);
        KV = va;
    }
    const bool ragged = (N & 31) != 0;
    double tLam = 0.0, tG2 = 0.0, tV = 0.0;
    for (int A = part * nwarps + warp; A < nblk; A += nparts * nwarps) {
        const int i = (A << 5) + lane;
        const bool live = i < N;
        const int ic = live ? i : N - 1;
        const int32_t xi = __ldg(x + ic), yi = __ldg(y + ic), zi = __ldg(z + ic);
        Acc64 acc = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        int n_hi = 0, fast_hi = 0, n_none = 0;
        for (int B = 0; B < nblk; ++B) {
            const int j0 = B << 5;
            if (B == A || (ragged && B == nblk - 1)) {
                double &la = (B == A) ? acc.lamd : acc.lam;
                tile16<kEnergy, true, true, true>(x, y, z, j0, ic, N, xi, yi, zi, E, zero, acc, la, n_none);
                tile16<kEnergy, true, true, true>(x, y, z, j0 + 16, ic, N, xi, yi, zi, E, zero, acc, la, n_none);
            } else if (B > A) {
                tile16<kEnergy, true, false, true>(x, y, z, j0, ic, N, xi, yi, zi, E, zero, acc, acc.lam, n_hi);
                tile16<kEnergy, true, false, true>(x, y, z, j0 + 16, ic, N, xi, yi, zi, E, zero, acc, acc.lam, n_hi);
                ++fast_hi;
            } else {
                tile16<kEnergy, false, false, true>(x, y, z, j0, ic, N, xi, yi, zi, E, zero, acc, acc.lam, n_none);
                tile16<kEnergy, false, false, true>(x, y, z, j0 + 16, ic, N, xi, yi, zi, E, zero, acc, acc.lam, n_none);
            }
        }
        if (live) {
            sv.S[(size_t)w * ld + i] = acc.s * kSUnit;                 // R17: rebuild the running sum
            if (kEnergy) {
                const double out_hi = (double)(32 * fast_hi - n_hi);
                tLam += 2.0 * (acc.lam - kLamClamp * out_hi) + acc.lamd;
                tG2 += acc.gx * acc.gx + acc.gy * acc.gy + acc.gz * acc.gz;
                tV += acc.v - (double)KV * out_hi;
            }
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
                double *o = partial + ((size_t)w * nparts + part) * 3;
                o[0] = a; o[1] = b; o[2] = c;
            }
        }
    }
}

__global__ void finalize32g_kernel(StateView sv, double Dk, const double *__restrict__ partial, int nparts, double *__restrict__ out)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= sv.W) return;
    double a = 0.0, b = 0.0, c = 0.0;
    for (int p = 0; p < nparts; ++p) {                                  // fixed order
        const double *o = partial + ((size_t)w * nparts + p) * 3;
        a += o[0]; b += o[1]; c += o[2];
    }
    const GroupDev g = sv.groups[sv.group_of[w]];
    const double Dku = Dk * g.inv_unit * g.inv_unit;
    const double lam = -5.0 * g.b5 * kGUnit * a;                                 // sum_i Lambda_i
    const double g2 = (2.5 * g.b5 * kGUnit * 0x1p-32) * (2.5 * g.b5 * kGUnit * 0x1p-32) * b;   // sum_i |G_i|^2
    const double T_PB = -Dku * (lam + g2);
    const double T_JF = -0.5 * Dku * lam;
    double *o = out + (size_t)w * 4;
    const double V = c * g.az.f32_scale;                                     // the potential was summed in units of f32_scale K
                o[0] = V + T_PB; o[1] = V; o[2] = T_PB; o[3] = T_JF;
}

int smem_bytes32(int N) { return 96 * 8 + 3 * (((N + 31) >> 5) << 5) * 4; }

template <int T>
cudaError_t launch32(qmc_ctx *c, double *d_out, bool energy)
{
    const int smem = smem_bytes32(c->p.N);
    cudaError_t e;
    if (energy) {
        auto k = energy32_kernel<T, true>;
        if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
        k<<<c->W, T, smem, c->stream>>>(c->sv, c->p.hbar2_over_2m, d_out);
    } else {
        auto k = energy32_kernel<T, false>;
        if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
        k<<<c->W, T, smem, c->stream>>>(c->sv, c->p.hbar2_over_2m, d_out);
    }
    return cudaGetLastError();
}

template <int T>
int occupancy32(int smem)
{
    int occ = 0;
    auto k = energy32_kernel<T, true>;
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, T, smem);
    return occ;
}

}  // namespace

cudaError_t launch_energy_f32g(qmc_ctx *c, double *d_out, bool energy)
{
    const int N = c->p.N, NP = ((N + 31) >> 5) << 5, nparts = c->energy_plan.parts;
    if (!c->d_enc) {
        cudaError_t e = cudaMalloc(&c->d_enc, sizeof(int32_t) * (size_t)c->W_total * 3 * NP);
        if (e == cudaSuccess) e = cudaMalloc(&c->d_epart, sizeof(double) * (size_t)c->W_total * nparts * 3);
        if (e != cudaSuccess) return e;
    }
    // a walker sub-range (qmc_step_host's chunks, possibly on concurrent streams) uses its own part of the scratch arrays
    const size_t w_off = (size_t)(c->sv.walker_id_base - c->p.walker_id_base);
    int32_t *enc = c->d_enc + w_off * 3 * NP;
    double *epart = c->d_epart + w_off * nparts * 3;
    encode_kernel<<<dim3((unsigned)c->W, (unsigned)((NP + 127) / 128)), 128, 0, c->stream>>>(c->sv, enc, NP);
    if (energy) {
        energy32g_kernel<256, true><<<(unsigned)c->W * (unsigned)nparts, 256, 0, c->stream>>>(c->sv, enc, NP, nparts, epart);
        finalize32g_kernel<<<(c->W + 127) / 128, 128, 0, c->stream>>>(c->sv, c->p.hbar2_over_2m, epart, nparts, d_out);
    } else {
        energy32g_kernel<256, false><<<(unsigned)c->W * (unsigned)nparts, 256, 0, c->stream>>>(c->sv, enc, NP, nparts, epart);
    }
    c->launches += energy ? 2 : 1;
    return cudaGetLastError();
}

// Gridded kernel: 8 warps per block, as many parts per walker as give every SM ~4 blocks (at most one i-block per warp)
bool plan_energy_f32g(qmc_ctx *c, EnergyPlan *out)
{
    const int N = c->p.N, nblk = (N + 31) >> 5;
    int parts = (4 * c->sm_count + c->W - 1) / c->W;
    const int max_parts = (nblk + 7) / 8;
    if (parts > max_parts) parts = max_parts;
    if (parts < 1) parts = 1;
    out->threads = 256;
    out->smem_bytes = 0;
    out->variant = 3;
    out->parts = parts;
    out->ctas_per_sm = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&out->ctas_per_sm, energy32g_kernel<256, true>, 256, 0);
    return true;
}

#define QMC_E32_THREADS(X) X(32) X(64) X(128) X(256) X(512)

cudaError_t launch_energy_f32(qmc_ctx *c, double *d_out, bool energy)
{
    const int T = c->energy_plan.threads;
#define X(TT) if (T == TT) return launch32<TT>(c, d_out, energy);
    QMC_E32_THREADS(X)
#undef X
    return cudaErrorInvalidValue;
}

// One warp per 32 particles up to 8 warps; qmc_set_tuning("energy_threads") overrides (tuning experiments).
bool plan_energy_f32(qmc_ctx *c, EnergyPlan *out)
{
    const int N = c->p.N;
    int T = 32;
    while (T < N && T < 256) T *= 2;
    if (smem_bytes32(N) > 113 * 1024) T = 512;      // one CTA per SM (N = 10000): fill it with 16 warps
    if (c->tuning.energy_threads > 0) {
        const int v = c->tuning.energy_threads;
        if (v >= 32 && v <= 512 && (v & (v - 1)) == 0) T = v;
    }
    out->threads = T;
    out->smem_bytes = smem_bytes32(N);
    if (out->smem_bytes > 227 * 1024) return false;
    out->ctas_per_sm = 0;
#define X(TT) if (T == TT) out->ctas_per_sm = occupancy32<TT>(out->smem_bytes);
    QMC_E32_THREADS(X)
#undef X
    return true;
}

}  // namespace qmc

// ==========================================================================================================
// qmc_local_energy_fp32c_static (include/qmc.h): the gridded FP32C local-energy pass for callers that must not
// allocate.  The kernels are the ones above, untouched (encode -> energy32g_kernel -> finalize32g_kernel); what
// differs is where their working memory lives.  launch_energy_f32g() takes it from cudaMalloc on first use, and
// everything else a qmc_ctx needs comes from cudaMalloc in qmc_create.  Here ALL of it -- the per-group constants,
// the walker -> group table, the fixed-point coordinates, the rebuilt pair sums and the per-block partial sums --
// sits in ONE file-scope device array that the CUDA module loader places when the library is loaded on a GPU.
//
// g_static_scratch below is, in HOST code, only a handle for the symbol: it is not a device address and must never
// be handed to a kernel.  The device address comes from cudaGetSymbolAddress, asked once per device (with that
// device current) on the first call and cached.
// ==========================================================================================================
namespace qmc {
namespace {

constexpr size_t kStaticGroupBytes = 512;                                         // one GroupDev, padded
constexpr size_t kStaticGroupOfOff = kStaticGroupBytes;                            // int32 [QMC_STATIC_MAX_WALKERS]
constexpr size_t kStaticEncOff = kStaticGroupOfOff + sizeof(int32_t) * QMC_STATIC_MAX_WALKERS;      // int32 [W][3][NP]
constexpr size_t kStaticSOff = kStaticEncOff + sizeof(int32_t) * 3 * (size_t)QMC_STATIC_MAX_SLOTS;  // double [W][ld], ld <= NP
constexpr size_t kStaticPartOff = kStaticSOff + sizeof(double) * (size_t)QMC_STATIC_MAX_SLOTS;      // double [W][parts][3]
// parts <= ceil(NP / 256), so W * parts <= W * NP / 256 + W
constexpr size_t kStaticPartMax = (size_t)QMC_STATIC_MAX_SLOTS / 256 + QMC_STATIC_MAX_WALKERS;
constexpr size_t kStaticBytes = kStaticPartOff + sizeof(double) * 3 * kStaticPartMax;
static_assert(sizeof(GroupDev) <= kStaticGroupBytes, "GroupDev outgrew its slot");
static_assert(kStaticEncOff % 256 == 0 && kStaticSOff % 256 == 0 && kStaticPartOff % 256 == 0, "sub-arrays stay 256-byte aligned");
static_assert(kStaticBytes == QMC_STATIC_SCRATCH_BYTES, "qmc.h states the size of the static scratch array");

static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

// Writes the two small tables the unchanged kernels read through StateView: the constants of the single parameter
// point, and group_of[w] = 0 for every walker (the only part of the scratch that has to hold zeros).
__global__ void static_tables_kernel(GroupDev g, GroupDev *__restrict__ groups, int32_t *__restrict__ group_of, int W)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w == 0) groups[0] = g;
    if (w < W) group_of[w] = 0;
}

// Angstrom [W][3][N] doubles -> fixed-point coordinates [W][3][NP], with exactly the arithmetic of
// set_positions_kernel<float> (wrap into [0, L), s = fl32(1 + x/L) in [1, 2)) followed by encode_kernel.
__global__ void encode_angstrom_kernel(const double *__restrict__ xyz, int N, int NP, double L_A, int32_t *__restrict__ enc)
{
    const int w = blockIdx.x;
    const int j = blockIdx.y * blockDim.x + threadIdx.x;
    if (j >= NP) return;
    const double *src = xyz + (size_t)w * 3 * N;
    int32_t *e = enc + (size_t)w * 3 * NP;
    for (int c = 0; c < 3; ++c) {
        int32_t k = 0;
        if (j < N) {
            double v = src[c * N + j];
            if (v >= L_A) v -= L_A;
            if (v < 0.0) v += L_A;
            float s = __double2float_rn(1.0 + v / L_A);
            if (s >= 2.0f) s -= 1.0f;
            if (s < 1.0f) s += 1.0f;
            k = enc_coord(s);
        }
        e[c * NP + j] = k;
    }
}

struct StaticDevice { bool ready = false; unsigned char *base = nullptr; int sm_count = 0; };
constexpr int kStaticMaxDevices = 64;
StaticDevice g_static_dev[kStaticMaxDevices];
// aziz_f32_scale() is a host search of a few milliseconds: remember the last parameter set it was run for
struct StaticScale { bool valid = false; double aziz[9]; double L; double scale; } g_static_scale;
std::mutex g_static_mu;

int static_fail(char *err, size_t err_len, int code, const char *fmt, ...)
{
    if (err && err_len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

}  // namespace
}  // namespace qmc

extern "C" int qmc_local_energy_fp32c_static(const double *d_xyz, int32_t W, int32_t N, double box_L, double jastrow_b,
                                             const double *aziz, double hbar2_over_2m, double *d_out, void *cuda_stream,
                                             char *err, size_t err_len)
{
    using namespace qmc;
    if (!d_xyz || !d_out || !aziz) return static_fail(err, err_len, QMC_E_ARG, "d_xyz, d_out and aziz are required");
    if (N < 2 || W < 1) return static_fail(err, err_len, QMC_E_ARG, "N >= 2 and W >= 1 required (got N = %d, W = %d)", N, W);
    if (!(box_L > 0.0) || !(jastrow_b >= 0.0) || !(aziz[1] > 0.0))
        return static_fail(err, err_len, QMC_E_ARG, "box_L > 0, jastrow_b >= 0 and aziz r_m > 0 required");
    const long long NP = (((long long)N + 31) >> 5) << 5;
    if (W > QMC_STATIC_MAX_WALKERS || N > QMC_STATIC_MAX_ATOMS || (long long)W * NP > QMC_STATIC_MAX_SLOTS)
        return static_fail(err, err_len, QMC_E_CAPACITY,
                           "W = %d walkers of N = %d atoms exceed the static scratch array: W <= %d, N <= %d and "
                           "W * (N rounded up to a multiple of 32) = %lld <= %d; use a qmc_ctx and qmc_local_energy for larger runs",
                           W, N, QMC_STATIC_MAX_WALKERS, QMC_STATIC_MAX_ATOMS, (long long)W * NP, QMC_STATIC_MAX_SLOTS);

#define STATIC_CUDA(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) \
        return static_fail(err, err_len, QMC_E_CUDA, "%s: %s", #expr, cudaGetErrorString(e__)); } while (0)

    int dev = 0;
    STATIC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return static_fail(err, err_len, QMC_E_ARG, "device ordinal %d not supported", dev);
    unsigned char *base = nullptr;
    int sm_count = 0;
    double f32_scale = 1.0;

    // per-group constants exactly as qmc_create computes them for QMC_FP32C (coordinate unit = the box edge)
    GroupDev G;
    memset(&G, 0, sizeof(G));
    {
        const double unit = box_L;
        G.unit = unit; G.inv_unit = 1.0 / unit; G.origin = 1.0;
        G.L_A = box_L;
        G.L = 1.0;
        G.h = 0.5 * G.L; G.h2 = G.h * G.h;
        const double bu = jastrow_b / unit;
        G.b5 = bu * bu * bu * bu * bu;
        G.c1 = -0.5 * G.b5;
        const double h = G.h;
        G.c0 = G.b5 / (h * h * h * h * h);
        G.sh = 2.0 / (h * h * h * h * h);
        G.step = 0.0;
        long long k = 1;
        while (4 * k * k * k < N) ++k;
        G.k_lat = (int32_t)k;
        G.a_lat = box_L / (double)k;
        G.pad = 0;
        const double rm = aziz[1] / unit;
        G.az.eps = aziz[0]; G.az.inv_rm = 1.0 / rm; G.az.rm2 = rm * rm; G.az.A = aziz[2];
        G.az.alpha = aziz[3]; G.az.beta = aziz[4]; G.az.c6 = aziz[5]; G.az.c8 = aziz[6]; G.az.c10 = aziz[7];
        G.az.D = aziz[8]; G.az.Drm = aziz[8] * rm;
    }
    {
        std::lock_guard<std::mutex> lock(g_static_mu);
        StaticDevice &D = g_static_dev[dev];
        if (!D.ready) {
            // set-up, once per device, with that device current: the device address of the static array
            void *p = nullptr;
            STATIC_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
            STATIC_CUDA(cudaDeviceGetAttribute(&D.sm_count, cudaDevAttrMultiProcessorCount, dev));
            D.base = static_cast<unsigned char *>(p);
            D.ready = true;
        }
        base = D.base;
        sm_count = D.sm_count;
        StaticScale &Sc = g_static_scale;
        if (!(Sc.valid && Sc.L == box_L && memcmp(Sc.aziz, aziz, sizeof(Sc.aziz)) == 0)) {
            Sc.scale = e32::aziz_f32_scale(G.az);
            memcpy(Sc.aziz, aziz, sizeof(Sc.aziz));
            Sc.L = box_L;
            Sc.valid = true;
        }
        f32_scale = Sc.scale;
    }
    G.az.f32_scale = f32_scale;

    GroupDev *groups = reinterpret_cast<GroupDev *>(base);
    int32_t *group_of = reinterpret_cast<int32_t *>(base + kStaticGroupOfOff);
    int32_t *enc = reinterpret_cast<int32_t *>(base + kStaticEncOff);
    double *S = reinterpret_cast<double *>(base + kStaticSOff);
    double *epart = reinterpret_cast<double *>(base + kStaticPartOff);

    // the split of a walker over thread blocks, as plan_energy_f32g chooses it
    const int nblk = (int)(NP >> 5);
    int parts = (4 * sm_count + W - 1) / W;
    const int max_parts = (nblk + 7) / 8;
    if (parts > max_parts) parts = max_parts;
    if (parts < 1) parts = 1;

    StateView sv{};
    sv.pos = nullptr;                       // the gridded kernels read the fixed-point copy only
    sv.S = S;
    sv.n_acc = nullptr;
    sv.group_of = group_of;
    sv.groups = groups;
    sv.W = W; sv.N = N; sv.ld = (N + 3) & ~3;
    sv.walker_id_base = 0;
    sv.proposal = 0;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    static_tables_kernel<<<(W + 255) / 256, 256, 0, st>>>(G, groups, group_of, W);
    encode_angstrom_kernel<<<dim3((unsigned)W, (unsigned)((NP + 127) / 128)), 128, 0, st>>>(d_xyz, N, (int)NP, box_L, enc);
    energy32g_kernel<256, true><<<(unsigned)W * (unsigned)parts, 256, 0, st>>>(sv, enc, (int)NP, parts, epart);
    finalize32g_kernel<<<(W + 127) / 128, 128, 0, st>>>(sv, hbar2_over_2m, epart, parts, d_out);
    STATIC_CUDA(cudaGetLastError());
#undef STATIC_CUDA
    return QMC_OK;
}
