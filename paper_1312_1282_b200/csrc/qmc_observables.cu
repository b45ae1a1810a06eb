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
// One CTA per walker, coordinates and the histogram in shared memory; thread i takes particle i and the
// partners j = i + k mod N, k = 1 .. (N-1)/2 (+ half of k = N/2 for even N): every unordered pair once,
// the same trip count for every thread.
#include "qmc_internal.h"

namespace qmc {

namespace {

__device__ __forceinline__ double image_component(double a, double b, double L, double h)
{
    const double t = __dadd_rn(a, -b);
    const double n = t > h ? L : (t < -h ? -L : 0.0);       // L * rint(t / L), exact
    return __dadd_rn(t, -n);
}

template <typename Real>
__global__ void __launch_bounds__(256) pair_histogram_kernel(StateView sv, int nbins, uint32_t *__restrict__ hist)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = sv.N, ld = sv.ld, w = blockIdx.x, tid = threadIdx.x, T = blockDim.x;
    double *x = reinterpret_cast<double *>(smem_raw), *y = x + N, *z = x + 2 * N;
    uint32_t *H = reinterpret_cast<uint32_t *>(x + 3 * N);
    const GroupDev g = sv.groups[sv.group_of[w]];
    const Real *gpos = reinterpret_cast<const Real *>(sv.pos) + (size_t)w * 3 * ld;
    for (int j = tid; j < N; j += T) {
        if (sizeof(Real) == 4) {                            // FP32C: s in [1,2) -> (s - 1) L, as qmc_get_positions
            x[j] = __dmul_rn(__dadd_rn((double)gpos[j], -1.0), g.L_A);
            y[j] = __dmul_rn(__dadd_rn((double)gpos[ld + j], -1.0), g.L_A);
            z[j] = __dmul_rn(__dadd_rn((double)gpos[2 * ld + j], -1.0), g.L_A);
        } else {
            x[j] = (double)gpos[j]; y[j] = (double)gpos[ld + j]; z[j] = (double)gpos[2 * ld + j];
        }
    }
    for (int k = tid; k < nbins; k += T) H[k] = 0u;
    __syncthreads();

    const double L = g.L_A, h = 0.5 * L;
    const double inv_dr = __ddiv_rn((double)nbins, h);
    const int kfull = (N - 1) >> 1;
    const bool even = (N & 1) == 0;
    for (int i = tid; i < N; i += T) {
        const double xi = x[i], yi = y[i], zi = z[i];
        const int kmax = kfull + ((even && i < (N >> 1)) ? 1 : 0);
        int j = i;
        for (int k = 1; k <= kmax; ++k) {
            j = (j + 1 == N) ? 0 : j + 1;
            const double dx = image_component(xi, x[j], L, h);
            const double dy = image_component(yi, y[j], L, h);
            const double dz = image_component(zi, z[j], L, h);
            const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
            const double r = __dsqrt_rn(r2);
            if (r < h) {
                int b = __double2int_rz(__dmul_rn(r, inv_dr));
                if (b >= nbins) b = nbins - 1;
                atomicAdd(&H[b], 1u);
            }
        }
    }
    __syncthreads();
    for (int k = tid; k < nbins; k += T) hist[(size_t)w * nbins + k] = H[k];
}

}  // namespace

cudaError_t launch_pair_histogram(qmc_ctx *c, int nbins, uint32_t *d_hist)
{
    c->launches += 1;
    const int smem = 3 * c->p.N * 8 + nbins * 4;
    cudaError_t e;
    if (c->p.mode == QMC_FP64) {
        auto k = pair_histogram_kernel<double>;
        if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
        k<<<c->W, 256, smem, c->stream>>>(c->sv, nbins, d_hist);
    } else {
        auto k = pair_histogram_kernel<float>;
        if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
        k<<<c->W, 256, smem, c->stream>>>(c->sv, nbins, d_hist);
    }
    return cudaGetLastError();
}

}  // namespace qmc
