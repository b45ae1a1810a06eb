// qmc_internal.h -- host-side context shared by the translation units of libqmc_b200.so.
#pragma once
#include <cstdint>
#include <cstdio>
#include <vector>
#include <cuda_runtime.h>

#include "../../include/qmc.h"
#include "qmc_device.cuh"

namespace qmc {

// Everything a kernel needs to find a walker's state.  Plain pointers, passed by value.
struct StateView {
    void     *pos;        // Real [W][3][ld]   (Real = double in FP64, float in FP32C)
    double   *S;          // [W][ld]  running pair sums S_i = sum_{j != i} u(r_ij)
    unsigned long long *n_acc;   // [W] accepted moves since init / set_positions
    const int32_t *group_of;     // [W] parameter point of each walker
    const GroupDev *groups;      // [n_groups]
    int32_t   W, N, ld;   // ld = N rounded up to a multiple of 4 (16-byte rows)
    uint32_t  walker_id_base;
    int32_t   proposal;   // 0: particles in order, uniform cube (R7); 1: random particle, Gaussian step (l.144, l.325)
};

struct TraceView {
    uint8_t *dec;         // [(w_end-w_begin)][capacity] or nullptr
    double  *margin;      // same shape or nullptr
    int32_t  w_begin, w_end;
    long long capacity, offset;   // offset = moves already recorded per walker
};

// In-kernel write-outs: every `every` sweeps the CTA writes
// its walker's coordinates and accepted-move count to a buffer the host can read while the kernel runs (mapped
// pinned host memory, or device memory) and then raises the walker's flag of that write-out (the paper's
// sentinel values in write-combined memory, as an explicit flag array).
struct WriteoutView {
    double *xyz;                   // [n_out][W][3][N] Angstrom, or nullptr: no write-outs
    unsigned long long *n_acc;     // [n_out][W] accepted moves since init / set_positions, or nullptr
    volatile int32_t *flag;        // [n_out][W] set to 1 after the data of (write-out, walker) have been written
    int32_t every;                 // sweeps between write-outs (m of Fig. 2)
    int32_t n_out;                 // capacity in write-outs
};

struct SweepPlan  { int threads, J, V, P, K, cluster, Nc, smem_bytes, ctas_per_sm; const void *shape;   // cluster > 1: blocks per walker, slices of Nc particles
                    const void *fallback; int fallback_smem; };   // fallback: one-move shape for what the tile kernel does not take
// Overrides of the launch heuristics; -1 / 0 = heuristic.  Each context carries its own copy (qmc_ctx::tuning), filled at
// creation: from the caller's key/value list (qmc_create_tuned) or from the process-wide default that qmc_set_tuning edits
// (qmc_create).  Nothing reads g_tuning after a context exists.
struct Tuning { int sweep_threads = 0, sweep_per_thread = 0, sweep_vector = -1, sweep_pending = -1, sweep_tile = -1,
                    energy_threads = 0, energy_ordered = 0, sweep_cluster = -1, host_chunks = 0; };
constexpr int kHostChunksMax = 8;
extern Tuning g_tuning;
struct EnergyPlan { int threads, smem_bytes, ctas_per_sm, variant, parts; };   // variant 0 ordered pairs, 1 / 2 unordered pairs (fp64 / fp32c), 3 gridded fp32c (parts blocks per walker)

}  // namespace qmc

struct qmc_ctx {
    qmc_params p;                                  // scalar fields only; arrays below
    std::vector<int32_t> walkers_per_group;
    std::vector<double>  box_L, jastrow_b;
    std::vector<qmc::GroupDev> groups;             // host mirror of d_groups
    int32_t W = 0, ld = 0;
    cudaStream_t stream = nullptr;
    void *d_state = nullptr;
    bool owns_state = false;
    qmc::StateView sv{};
    qmc::GroupDev *d_groups = nullptr;
    int32_t *d_group_of = nullptr;
    int32_t *d_enc = nullptr;                      // gridded FP32C energy: fixed-point coordinates [W][3][NP] (first use)
    double *d_epart = nullptr;                     //   and per-block partial sums [W][parts][3]
    int32_t W_total = 0;                           // W of the whole context (W itself is narrowed by qmc_step_host's chunks)
    double *d_scratch = nullptr;                   // [W][4] + [W] + [W][3][N] staging for *_host calls
    // qmc_run_blocks_host: write-out stream, double-buffered block results, their events (created on first use)
    cudaStream_t out_stream = nullptr;
    double *d_block = nullptr;                     // [2][W][5]
    double *d_block_xyz = nullptr;                 // [2][W][3][N] coordinate write-outs (allocated on first use)
    bool blocks_ready = false;                     // stream, d_block and the events below exist
    cudaEvent_t ev_ready[2] = {nullptr, nullptr}, ev_copied[2] = {nullptr, nullptr};
    // qmc_step_host: copy-in, copy-out and two compute streams, per-chunk events, staging of the pair sums (first use)
    cudaStream_t hs_in = nullptr, hs_out = nullptr, hs_cmp[2] = {nullptr, nullptr};
    cudaEvent_t hs_ev_in[qmc::kHostChunksMax] = {}, hs_ev_cmp[qmc::kHostChunksMax] = {}, hs_ev_fork = nullptr, hs_ev_join = nullptr;
    double *d_hS = nullptr;                        // [W][N]
    bool host_ready = false;
    qmc::TraceView trace{};
    qmc::WriteoutView wo{};                        // in-kernel write-outs of the running qmc_sweep_writeouts call
    qmc::Tuning tuning{};                          // this context's overrides of the launch heuristics
    qmc::SweepPlan sweep_plan{};
    qmc::EnergyPlan energy_plan{};
    uint64_t seed = 0;
    uint32_t t = 0;
    uint32_t t_acc0 = 0;                           // sweep index at which the acceptance counters were zeroed
    bool have_state = false;
    int sm_count = 0;
    uint64_t launches = 0;
    char err[512] = {0};
};

namespace qmc {

// kernels' host launchers (one per translation unit); each returns a cudaError_t
cudaError_t launch_sweep(qmc_ctx *c, int n_sweeps);
cudaError_t launch_energy(qmc_ctx *c, double *d_out, bool energy /*false: only rebuild S_i*/);
cudaError_t launch_init(qmc_ctx *c);
cudaError_t launch_set_positions(qmc_ctx *c, const double *d_xyz);
cudaError_t launch_get_positions(qmc_ctx *c, double *d_xyz);
cudaError_t launch_acceptance(qmc_ctx *c, double *d_out);
cudaError_t launch_pair_histogram(qmc_ctx *c, int nbins, uint32_t *d_hist);   // qmc_observables.cu
bool pair_histogram_fits(int N, int nbins, int mode);                        // shared-memory capacity of that kernel
bool plan_sweep(qmc_ctx *c, SweepPlan *out);
bool plan_energy(qmc_ctx *c, EnergyPlan *out);
cudaError_t launch_energy_f32(qmc_ctx *c, double *d_out, bool energy);
bool plan_energy_f32(qmc_ctx *c, EnergyPlan *out);
cudaError_t launch_energy_f32s(qmc_ctx *c, double *d_out, bool energy);   // unordered pairs (qmc_energy_f32s.cu)
bool plan_energy_f32s(qmc_ctx *c, EnergyPlan *out);
cudaError_t launch_energy_f32g(qmc_ctx *c, double *d_out, bool energy);   // gridded, any N (qmc_energy_f32.cu)
bool plan_energy_f32g(qmc_ctx *c, EnergyPlan *out);
cudaError_t launch_energy_f64(qmc_ctx *c, double *d_out, bool energy);
bool plan_energy_f64(qmc_ctx *c, EnergyPlan *out);

}  // namespace qmc
