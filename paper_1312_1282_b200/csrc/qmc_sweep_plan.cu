// qmc_sweep_plan.cu -- host side of the sweep: choice of the (T, J, V) kernel shape for N and the launch.
#include <cmath>
#include <cstdlib>

#include "qmc_sweep_impl.cuh"

namespace qmc {

cudaError_t launch_sweep(qmc_ctx *c, int n_sweeps)
{
    c->launches += 1;
    const SweepShape *sh = static_cast<const SweepShape *>(c->sweep_plan.shape);
    if (sh == nullptr) return cudaErrorInvalidValue;
    return sh->launch(c, n_sweeps, c->sweep_plan.smem_bytes);
}

// Threads per walker the heuristic aims at: about 16 particles per thread (measured on B200, profiles/),
// one warp at least.  QMC_SWEEP_SHAPE="T,J[,V[,P]]" overrides the heuristic (tuning experiments).
bool plan_sweep(qmc_ctx *c, SweepPlan *out)
{
    const int N = c->p.N, mode = c->p.mode;
    int n = 0;
    const SweepShape *tab = (mode == QMC_FP64) ? sweep_shapes_f64(&n) : sweep_shapes_f32(&n);
    auto usable = [&](const SweepShape &s) {
        if ((long long)s.T * s.J < N) return false;
        if (s.V > 1 && N % s.V != 0) return false;
        return sweep_smem_bytes(s.T, s.J, mode, s.P) <= 227 * 1024;
    };
    const SweepShape *best = nullptr;
    if (const char *env = getenv("QMC_SWEEP_SHAPE")) {
        int t = 0, j = 0, v = 0, pp = 0;
        const int got = sscanf(env, "%d,%d,%d,%d", &t, &j, &v, &pp);
        for (int k = 0; k < n && got >= 2; ++k)
            if (tab[k].T == t && tab[k].J == j && (got < 3 || tab[k].V == v) && (got < 4 || tab[k].P == pp) && usable(tab[k]))
                if (!best || tab[k].V > best->V || (tab[k].V == best->V && tab[k].P > best->P)) best = &tab[k];
    }
    if (!best) {
        const int per_thread = 16;
        double t_target = std::log2(std::fmax(32.0, std::fmin(1024.0, (double)N / per_thread)));
        double best_score = 1e30;
        for (int k = 0; k < n; ++k) {
            if (!usable(tab[k])) continue;
            const double waste = (double)(tab[k].T * tab[k].J - N) / (double)N;       // idle slots
            const double score = 4.0 * waste + std::fabs(std::log2((double)tab[k].T) - t_target)
                               + (mode == QMC_FP64 ? 0.25 * (2 - tab[k].V) : 0.25 * (4 - tab[k].V)) - 0.1 * tab[k].P;   // hi + lo running sums: 10.5 vs 11.1 ms at N = 1952 (measured)
            if (score < best_score) { best_score = score; best = &tab[k]; }
        }
    }
    out->threads = 0; out->J = 0; out->V = 0; out->ctas_per_sm = 0; out->shape = nullptr;
    out->smem_bytes = N * (8 + 3 * (mode == QMC_FP64 ? 8 : 4));
    if (!best) return false;
    out->threads = best->T; out->J = best->J; out->V = best->V; out->shape = best;
    out->smem_bytes = sweep_smem_bytes(best->T, best->J, mode, best->P);
    out->ctas_per_sm = best->occupancy(out->smem_bytes);
    return true;
}

}  // namespace qmc
