// qmc_sweep_plan.cu -- host side of the sweep: choice of the kernel shape (T threads per walker, J particles per
// thread in packs of V, running-sum representation, tile size K) for N, W and the mode, and the launch.
#include <cmath>
#include <cstdlib>

#include "qmc_sweep_tile.cuh"
#include "qmc_sweep_cluster.cuh"

namespace qmc {

Tuning g_tuning;

cudaError_t launch_sweep(qmc_ctx *c, int n_sweeps)
{
    c->launches += 1;
    if (c->sweep_plan.cluster > 1) {                                 // one walker per thread-block cluster (NEXT-3)
        const ClusterShape *cs = static_cast<const ClusterShape *>(c->sweep_plan.shape);
        if (cs == nullptr || c->p.N < 3) return cudaErrorNotSupported;
        if (c->sv.proposal == 0 && c->wo.xyz == nullptr)
            return cs->launch(c, n_sweeps, c->sweep_plan.smem_bytes, c->sweep_plan.cluster, c->sweep_plan.Nc);
        // proposal 1 and in-kernel write-outs exist in the one-block kernel only: where one block can hold the walker
        // the plan carries that shape as its fallback (slower for few walkers, but it serves the call)
        const SweepShape *fb = static_cast<const SweepShape *>(c->sweep_plan.fallback);
        if (fb == nullptr) return cudaErrorNotSupported;
        return fb->launch(c, n_sweeps, c->sweep_plan.fallback_smem);
    }
    const SweepShape *sh = static_cast<const SweepShape *>(c->sweep_plan.shape);
    int smem = c->sweep_plan.smem_bytes;
    if (sh != nullptr && sh->K > 1 && c->sv.proposal != 0) {       // the tile kernel moves particles in order only
        sh = static_cast<const SweepShape *>(c->sweep_plan.fallback);
        smem = c->sweep_plan.fallback_smem;
    }
    if (sh == nullptr) return cudaErrorInvalidValue;
    return sh->launch(c, n_sweeps, smem);
}

// Cluster plan: C blocks per walker, slices of Nc particles (a multiple of 4), the narrowest block shape that holds
// a slice.  Used when no single block can hold the walker (N > 10240 in FP32C, > 6144 in FP64) and when
// qmc_set_tuning("sweep_cluster") asks for it (e.g. one walker on 8 SMs).
static bool plan_cluster(qmc_ctx *c, SweepPlan *out, int C)
{
    const int N = c->p.N, mode = c->p.mode;
    int n = 0;
    const ClusterShape *tab = (mode == QMC_FP64) ? cluster_shapes_f64(&n) : cluster_shapes_f32(&n);
    const int Nc = (((N + C - 1) / C) + 3) & ~3;
    const ClusterShape *best = nullptr;
    double best_cost = 1e300;
    for (int k = 0; k < n; ++k) {
        const ClusterShape &s = tab[k];
        if (s.T * s.J < Nc || s.smem > 227 * 1024) continue;
        if (mode != QMC_FP64 && N % s.V != 0) continue;
        if ((c->tuning.sweep_threads > 0 && s.T != c->tuning.sweep_threads) || (c->tuning.sweep_per_thread > 0 && s.J != c->tuning.sweep_per_thread)) continue;
        const double cost = (double)s.T * ((double)s.J + (mode == QMC_FP64 ? 4.0 : 12.0)) * (s.V == 2 && mode != QMC_FP64 ? 1.12 : 1.0);
        if (cost < best_cost) { best_cost = cost; best = &s; }
    }
    if (!best) return false;
    out->threads = best->T; out->J = best->J; out->V = best->V; out->P = best->P; out->K = 1;
    out->cluster = C; out->Nc = Nc; out->shape = best; out->smem_bytes = best->smem; out->ctas_per_sm = 1;
    out->fallback = nullptr; out->fallback_smem = 0;
    return true;
}

// What a shape costs (relative; it only has to rank shapes).  Fitted to the shape scans of the five configs in
// profiles/r02_shapes.md:
//   * in the throughput-bound regime a move costs every warp of the CTA  a J + b  pipe cycles (a: pair terms, b: the
//     serial part -- reduction, barrier, decision; b / a = 1.35 in FP64, 4.2 in FP32C), so a sweep costs
//     T (J + b/a): few threads with many particles each win, and padding (T J > N) is paid for;
//   * that only holds while the SM has enough warps to overlap the serial parts of different walkers: below ~10
//     resident warps per SM the time grows like 10 / warps.  W is given (PAPER.md l.484, l.502
//     tuned walkers per SM instead), so with few walkers -- configs 1 and 2 -- threads per walker must grow;
//   * more than 20 particles per thread costs registers (retained trial terms) and loses to the next wider shape.
static double shape_cost(const SweepShape &s, int N, int W, int mode, int sm_count, int ctas_per_sm)
{
    if (ctas_per_sm < 1) return 1e300;
    const double b_over_a = (mode == QMC_FP64) ? 1.35 : 4.2;
    double cost = (double)s.T * ((double)s.J + b_over_a);
    const double resident = std::fmin((double)ctas_per_sm, std::ceil((double)W / sm_count));
    const double warps = resident * (s.T / 32);
    if (warps < 10.0) cost *= 10.0 / warps;
    if (s.J > 20) cost *= 1.15;
    (void)N;
    return cost;
}

bool plan_sweep(qmc_ctx *c, SweepPlan *out)
{
    const int N = c->p.N, mode = c->p.mode, W = c->W;
    int n = 0, nt = 0;
    const SweepShape *tab = (mode == QMC_FP64) ? sweep_shapes_f64(&n) : sweep_shapes_f32(&n);
    const SweepShape *tile = (mode == QMC_FP64) ? nullptr : sweep_shapes_tile(&nt);
    auto usable = [&](const SweepShape &s) {
        if ((long long)s.T * s.J < N) return false;
        if (s.V > 1 && N % s.V != 0) return false;
        if (s.K > 1 && (N % s.K != 0 || N < 2 * s.K)) return false;
        return s.smem <= 227 * 1024;
    };
    const Tuning &tu = c->tuning;
    out->cluster = 1; out->Nc = 0;
    // the one-block, one-move shape the heuristic would take: what a cluster plan falls back to for proposal 1 and
    // in-kernel write-outs (nullptr when no single block holds the walker)
    auto one_block = [&](int *smem) -> const SweepShape * {
        const SweepShape *b = nullptr;
        double b_cost = 1e300;
        for (int k = 0; k < n; ++k) {
            const SweepShape &s = tab[k];
            if (!usable(s) || s.K > 1) continue;
            double cost = shape_cost(s, N, W, mode, c->sm_count, s.occupancy(s.smem));
            if (mode != QMC_FP64) cost *= (s.V == 4 ? 1.0 : (s.V == 2 ? 1.12 : 1.6)) * (s.P ? 1.0 : 1.06);
            else                  cost *= (s.V == 2 ? 1.0 : 1.05);
            if (cost < b_cost) { b_cost = cost; b = &s; }
        }
        *smem = b ? b->smem : 0;
        return b;
    };
    if (tu.sweep_cluster > 1 && N >= 3) {
        int C = tu.sweep_cluster > kClusterMax ? kClusterMax : tu.sweep_cluster;
        if (plan_cluster(c, out, C)) { out->fallback = one_block(&out->fallback_smem); return true; }
    }
    auto wanted = [&](const SweepShape &s) {
        return (tu.sweep_threads <= 0 || s.T == tu.sweep_threads) && (tu.sweep_per_thread <= 0 || s.J == tu.sweep_per_thread)
            && (tu.sweep_vector < 0 || s.V == tu.sweep_vector) && (tu.sweep_pending < 0 || s.P == tu.sweep_pending)
            && (tu.sweep_tile < 0 || s.K == (tu.sweep_tile < 1 ? 1 : tu.sweep_tile));
    };
    const bool forced = tu.sweep_threads > 0 || tu.sweep_per_thread > 0 || tu.sweep_vector >= 0 || tu.sweep_pending >= 0 || tu.sweep_tile >= 0;
    const SweepShape *best = nullptr;
    double best_cost = 1e300;
    int best_occ = 0;
    for (int pass = 0; pass < 2 && !best; ++pass) {
        // pass 0: shapes the tuning overrides ask for (if any); pass 1: the heuristic over the one-move shapes.
        // The tile kernel (K > 1) is never the heuristic's choice: it measured slower than the one-move kernel at
        // every config but config 4 (+0.8 %), see profiles/r02_tile.md; qmc_set_tuning("sweep_tile") selects it.
        if (pass == 0 && !forced) continue;
        for (int k = 0; k < n + nt; ++k) {
            const SweepShape &s = k < n ? tab[k] : tile[k - n];
            if (!usable(s) || (pass == 0 && !wanted(s)) || (pass == 1 && s.K > 1)) continue;
            const int occ = s.occupancy(s.smem);
            double cost = shape_cost(s, N, W, mode, c->sm_count, occ);
            if (mode != QMC_FP64) cost *= (s.V == 4 ? 1.0 : (s.V == 2 ? 1.12 : 1.6)) * (s.P ? 1.0 : 1.06);
            else                  cost *= (s.V == 2 ? 1.0 : 1.05);
            if (cost < best_cost) { best_cost = cost; best = &s; best_occ = occ; }
        }
    }
    out->threads = 0; out->J = 0; out->V = 0; out->P = 0; out->K = 0; out->cluster = 1; out->ctas_per_sm = 0; out->shape = nullptr;
    out->fallback = nullptr; out->fallback_smem = 0;
    out->smem_bytes = N * (8 + 3 * (mode == QMC_FP64 ? 8 : 4));
    // Clusters.  Few walkers of many atoms (the equilibration case): one block per walker
    // would leave most SMs idle, and the cluster kernel's barrier pays off from N ~ 4000 (FP32C) / 2500 (FP64) up
    // (profiles/r02_cluster.md: N = 10000, one walker: 23.0 ms per sweep on one SM, 14.4 ms on 8).  A GPC runs at
    // most two clusters of 8, four of 4: 16 / 32 / 64 walkers at once.
    int c_few = 1;
    if (tu.sweep_cluster < 0 && !forced && N >= (mode == QMC_FP64 ? 2500 : 4000))
        c_few = W <= 16 ? 8 : (W <= 32 ? 4 : (W <= 64 ? 2 : 1));
    if (!best || c_few > 1) {                        // ... or no single block holds the walker: the smallest cluster that does
        for (int C = (best ? c_few : 2); C <= kClusterMax && N >= 3; C *= 2)
            if (C >= c_few && plan_cluster(c, out, C)) { out->fallback = one_block(&out->fallback_smem); return true; }
        if (!best) return false;
        out->cluster = 1; out->Nc = 0;
    }
    out->threads = best->T; out->J = best->J; out->V = best->V; out->P = best->P; out->K = best->K; out->shape = best;
    out->smem_bytes = best->smem;
    out->ctas_per_sm = best_occ;
    out->fallback = best;
    out->fallback_smem = best->smem;
    if (best->K > 1) {                               // the one-move kernel of the same geometry (proposal 1)
        out->fallback = nullptr;
        for (int k = 0; k < n; ++k)
            if (tab[k].T == best->T && tab[k].J == best->J && tab[k].V == best->V && tab[k].P == 1 && usable(tab[k])) {
                out->fallback = &tab[k];
                out->fallback_smem = tab[k].smem;
            }
        if (!out->fallback) return false;
    }
    return true;
}

}  // namespace qmc
