// qmc_api.cu -- the C ABI of include/qmc.h: context management, small state kernels
// (initial lattice, position import/export, acceptance), host-buffer step, pipe-peak microbenchmark.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include <nvtx3/nvToolsExt.h>          // header-only NVTX v3: ranges around the hot launches

#include "qmc_internal.h"
#include "qmc_energy_f32_pair.cuh"     // aziz_f32_scale (host)

using namespace qmc;

namespace {
struct NvtxRange {                      // no-op unless a profiler is attached
    explicit NvtxRange(const char *name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};
}  // namespace

static char g_create_err[512] = "no error";

#define QMC_FAIL(c, code, ...)                                         \
    do {                                                               \
        snprintf((c) ? (c)->err : g_create_err, 512, __VA_ARGS__);     \
        return (code);                                                 \
    } while (0)

#define QMC_CUDA(c, expr)                                                                     \
    do {                                                                                      \
        cudaError_t e__ = (expr);                                                             \
        if (e__ != cudaSuccess) QMC_FAIL(c, QMC_E_CUDA, "%s: %s", #expr, cudaGetErrorString(e__)); \
    } while (0)

namespace qmc {

// ------------------------------------------------------------------------------------------
// Initial walkers (R13): particle i on FCC site floor(i*M/N), M = 4k^3, sites ordered
// (ix,iy,iz,basis) with the basis fastest; + jitter * a_c, a_c from Philox counter (i,0,walker,1).
// ------------------------------------------------------------------------------------------
// Angstrom -> stored coordinate.  FP64: the value itself.  FP32C: s = 1 + x/L rounded to fp32, in [1,2).
template <typename Real> __device__ __forceinline__ Real to_stored(double x, const GroupDev &g);
template <> __device__ __forceinline__ double to_stored<double>(double x, const GroupDev &) { return x; }
template <> __device__ __forceinline__ float to_stored<float>(double x, const GroupDev &g)
{
    float s = __double2float_rn(1.0 + x / g.L_A);
    if (s >= 2.0f) s -= 1.0f;
    if (s < 1.0f) s += 1.0f;
    return s;
}
template <typename Real> __device__ __forceinline__ double to_angstrom(Real s, const GroupDev &g);
template <> __device__ __forceinline__ double to_angstrom<double>(double s, const GroupDev &) { return s; }
template <> __device__ __forceinline__ double to_angstrom<float>(float s, const GroupDev &g)
{
    return __dmul_rn(__dadd_rn((double)s, -1.0), g.L_A);
}

template <typename Real>
__global__ void init_kernel(StateView sv, uint2 key, double jitter)
{
    const int N = sv.N, ld = sv.ld;
    const int w = blockIdx.x;
    const int i = blockIdx.y * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const GroupDev g = sv.groups[sv.group_of[w]];
    const long long k = g.k_lat, M = 4 * k * k * k;
    const long long site = ((long long)i * M) / N;
    const int bas = (int)(site & 3);
    const long long cell = site >> 2;
    const long long iz = cell % k, iy = (cell / k) % k, ix = cell / (k * k);
    const double ox = (bas == 1 || bas == 2) ? 0.5 : 0.0;
    const double oy = (bas == 1 || bas == 3) ? 0.5 : 0.0;
    const double oz = (bas == 2 || bas == 3) ? 0.5 : 0.0;
    const uint4 r = philox4x32_10(make_uint4((uint32_t)i, 0u, sv.walker_id_base + (uint32_t)w, 1u), key);
    const double idx[3] = {(double)ix + ox, (double)iy + oy, (double)iz + oz};
    const uint32_t word[3] = {r.x, r.y, r.z};
    Real *pos = reinterpret_cast<Real *>(sv.pos) + (size_t)w * 3 * ld;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double v = __dadd_rn(__dmul_rn(idx[c], g.a_lat), __dmul_rn(jitter, word_to_pm1(word[c])));
        if (v >= g.L_A) v = __dadd_rn(v, -g.L_A);
        if (v < 0.0) v = __dadd_rn(v, g.L_A);
        pos[c * ld + i] = to_stored<Real>(v, g);
    }
}

template <typename Real>
__global__ void set_positions_kernel(StateView sv, const double *__restrict__ xyz)
{
    const int N = sv.N, ld = sv.ld;
    const int w = blockIdx.x;
    const int i = blockIdx.y * blockDim.x + threadIdx.x;
    if (i >= ld) return;
    Real *pos = reinterpret_cast<Real *>(sv.pos) + (size_t)w * 3 * ld;
    const double *src = xyz + (size_t)w * 3 * N;
    const GroupDev g = sv.groups[sv.group_of[w]];
    for (int c = 0; c < 3; ++c) {
        Real q = (Real)g.origin;
        if (i < N) {
            double v = src[c * N + i];
            if (v >= g.L_A) v -= g.L_A;
            if (v < 0.0) v += g.L_A;
            q = to_stored<Real>(v, g);
        }
        pos[c * ld + i] = q;
    }
    if (i == 0) sv.n_acc[w] = 0ull;
}

template <typename Real>
__global__ void get_positions_kernel(StateView sv, double *__restrict__ xyz)
{
    const int N = sv.N, ld = sv.ld;
    const int w = blockIdx.x;
    const int i = blockIdx.y * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const Real *pos = reinterpret_cast<const Real *>(sv.pos) + (size_t)w * 3 * ld;
    double *dst = xyz + (size_t)w * 3 * N;
    const GroupDev g = sv.groups[sv.group_of[w]];
    for (int c = 0; c < 3; ++c) dst[c * N + i] = to_angstrom<Real>(pos[c * ld + i], g);
}

__global__ void get_pair_sums_kernel(StateView sv, double *__restrict__ S)
{
    const int w = blockIdx.x;
    const int i = blockIdx.y * blockDim.x + threadIdx.x;
    // the state holds raw sums of t = y^5 + z^5 - sh; u = c1 t (qmc_sweep_impl.cuh)
    if (i < sv.N) S[(size_t)w * sv.N + i] = sv.groups[sv.group_of[w]].c1 * sv.S[(size_t)w * sv.ld + i];
}

// running pair sums in the state's own unit (sum_j t(r_ij), u = c1 t), [W][N] <-> [W][ld]: qmc_step_host's h_S_in / h_S_out
__global__ void export_raw_sums_kernel(StateView sv, double *__restrict__ S)
{
    const int w = blockIdx.x;
    const int i = blockIdx.y * blockDim.x + threadIdx.x;
    if (i < sv.N) S[(size_t)w * sv.N + i] = sv.S[(size_t)w * sv.ld + i];
}
__global__ void import_raw_sums_kernel(StateView sv, const double *__restrict__ S)
{
    const int w = blockIdx.x;
    const int i = blockIdx.y * blockDim.x + threadIdx.x;
    if (i < sv.N) sv.S[(size_t)w * sv.ld + i] = S[(size_t)w * sv.N + i];
}

__global__ void acceptance_kernel(StateView sv, double attempted, double *__restrict__ out)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w < sv.W) out[w] = attempted > 0.0 ? (double)sv.n_acc[w] / attempted : 0.0;
}

__global__ void zero_state_kernel(StateView sv, size_t pos_bytes)
{
    // zero the padding of every row once so that vector copies never move uninitialised bytes
    const size_t n = pos_bytes / 4;
    uint32_t *p = reinterpret_cast<uint32_t *>(sv.pos);
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = 0u;
    double *S = sv.S;
    const size_t ns = (size_t)sv.W * sv.ld;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < ns; i += (size_t)gridDim.x * blockDim.x) S[i] = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < (size_t)sv.W; i += (size_t)gridDim.x * blockDim.x) sv.n_acc[i] = 0ull;
}

// walkers on gridDim.x (limit 2^31 - 1), particle tiles of 128 on gridDim.y
static dim3 grid_wn(const qmc_ctx *c, int n) { return dim3((unsigned)c->W, (unsigned)((n + 127) / 128)); }

cudaError_t launch_init(qmc_ctx *c)
{
    c->launches += 1;
    const uint2 key = make_uint2((uint32_t)(c->seed & 0xFFFFFFFFull), (uint32_t)(c->seed >> 32));
    if (c->p.mode == QMC_FP64) init_kernel<double><<<grid_wn(c, c->p.N), 128, 0, c->stream>>>(c->sv, key, c->p.jitter);
    else                       init_kernel<float><<<grid_wn(c, c->p.N), 128, 0, c->stream>>>(c->sv, key, c->p.jitter);
    return cudaGetLastError();
}
cudaError_t launch_set_positions(qmc_ctx *c, const double *d_xyz)
{
    c->launches += 1;
    if (c->p.mode == QMC_FP64) set_positions_kernel<double><<<grid_wn(c, c->ld), 128, 0, c->stream>>>(c->sv, d_xyz);
    else                       set_positions_kernel<float><<<grid_wn(c, c->ld), 128, 0, c->stream>>>(c->sv, d_xyz);
    return cudaGetLastError();
}
cudaError_t launch_get_positions(qmc_ctx *c, double *d_xyz)
{
    c->launches += 1;
    if (c->p.mode == QMC_FP64) get_positions_kernel<double><<<grid_wn(c, c->p.N), 128, 0, c->stream>>>(c->sv, d_xyz);
    else                       get_positions_kernel<float><<<grid_wn(c, c->p.N), 128, 0, c->stream>>>(c->sv, d_xyz);
    return cudaGetLastError();
}
cudaError_t launch_acceptance(qmc_ctx *c, double *d_out)
{
    c->launches += 1;
    acceptance_kernel<<<(c->W + 127) / 128, 128, 0, c->stream>>>(c->sv, (double)(c->t - c->t_acc0) * (double)c->p.N, d_out);
    return cudaGetLastError();
}
static cudaError_t launch_acceptance_attempted(qmc_ctx *c, double attempted, double *d_out)
{
    c->launches += 1;
    acceptance_kernel<<<(c->W + 127) / 128, 128, 0, c->stream>>>(c->sv, attempted, d_out);
    return cudaGetLastError();
}
static cudaError_t launch_raw_sums(qmc_ctx *c, double *d_S, bool import)
{
    c->launches += 1;
    if (import) import_raw_sums_kernel<<<grid_wn(c, c->p.N), 128, 0, c->stream>>>(c->sv, d_S);
    else        export_raw_sums_kernel<<<grid_wn(c, c->p.N), 128, 0, c->stream>>>(c->sv, d_S);
    return cudaGetLastError();
}

}  // namespace qmc

// ==========================================================================================
// C ABI
// ==========================================================================================
static bool valid_params(const qmc_params *p, char *err)
{
    if (!p) { snprintf(err, 512, "params is NULL"); return false; }
    if (p->N < 2) { snprintf(err, 512, "N must be >= 2 (got %d)", p->N); return false; }
    if (p->n_groups < 1 || !p->walkers_per_group || !p->box_L || !p->jastrow_b) {
        snprintf(err, 512, "n_groups >= 1 and the three per-group arrays are required"); return false;
    }
    if (p->mode != QMC_FP64 && p->mode != QMC_FP32C) { snprintf(err, 512, "unknown mode %d", p->mode); return false; }
    long long W = 0;
    for (int g = 0; g < p->n_groups; ++g) {
        if (p->walkers_per_group[g] < 0) { snprintf(err, 512, "walkers_per_group[%d] < 0", g); return false; }
        if (!(p->box_L[g] > 0.0) || !(p->jastrow_b[g] >= 0.0)) { snprintf(err, 512, "box_L > 0 and jastrow_b >= 0 required (group %d)", g); return false; }
        W += p->walkers_per_group[g];
    }
    if (W < 1 || W > 0x7fffffffLL) { snprintf(err, 512, "total walker count %lld out of range", W); return false; }
    if (!(p->aziz[1] > 0.0)) { snprintf(err, 512, "aziz r_m must be > 0"); return false; }
    return true;
}

static int round_up4(int n) { return (n + 3) & ~3; }

static void state_layout(const qmc_params *p, long long W, size_t *pos_bytes, size_t *S_off, size_t *acc_off, size_t *total)
{
    const size_t ld = (size_t)round_up4(p->N);
    const size_t real = p->mode == QMC_FP64 ? 8 : 4;
    auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
    *pos_bytes = (size_t)W * 3 * ld * real;
    *S_off = up(*pos_bytes);
    *acc_off = up(*S_off + (size_t)W * ld * 8);
    *total = up(*acc_off + (size_t)W * 8);
}

extern "C" size_t qmc_state_bytes(const qmc_params *p)
{
    char err[512];
    if (!valid_params(p, err)) return 0;
    long long W = 0;
    for (int g = 0; g < p->n_groups; ++g) W += p->walkers_per_group[g];
    size_t pb, so, ao, tot;
    state_layout(p, W, &pb, &so, &ao, &tot);
    return tot;
}

static bool tuning_set(Tuning &t, const char *key, int32_t value)
{
    struct { const char *name; int *field; } tab[] = {
        {"sweep_threads", &t.sweep_threads}, {"sweep_per_thread", &t.sweep_per_thread}, {"sweep_vector", &t.sweep_vector},
        {"sweep_pending", &t.sweep_pending}, {"sweep_tile", &t.sweep_tile}, {"sweep_cluster", &t.sweep_cluster},
        {"energy_threads", &t.energy_threads}, {"energy_ordered", &t.energy_ordered}, {"host_chunks", &t.host_chunks},
    };
    for (auto &e : tab)
        if (strcmp(key, e.name) == 0) { *e.field = value; return true; }
    return false;
}

static int create_impl(const qmc_params *p, void *cuda_stream, void *d_state, size_t state_bytes, const Tuning &tuning, qmc_ctx **out);

extern "C" int qmc_create(const qmc_params *p, void *cuda_stream, void *d_state, size_t state_bytes, qmc_ctx **out)
{
    return create_impl(p, cuda_stream, d_state, state_bytes, g_tuning, out);
}

extern "C" int qmc_create_tuned(const qmc_params *p, void *cuda_stream, void *d_state, size_t state_bytes,
                                const char *const *keys, const int32_t *values, int32_t n_keys, qmc_ctx **out)
{
    if (out) *out = nullptr;
    if (n_keys < 0 || (n_keys > 0 && (!keys || !values))) QMC_FAIL((qmc_ctx *)nullptr, QMC_E_ARG, "qmc_create_tuned: keys and values are required");
    Tuning t{};                                          // the heuristics, whatever qmc_set_tuning has been told
    for (int k = 0; k < n_keys; ++k)
        if (!keys[k] || !tuning_set(t, keys[k], values[k]))
            QMC_FAIL((qmc_ctx *)nullptr, QMC_E_ARG, "qmc_create_tuned: unknown key '%s'", keys[k] ? keys[k] : "(null)");
    return create_impl(p, cuda_stream, d_state, state_bytes, t, out);
}

static int create_impl(const qmc_params *p, void *cuda_stream, void *d_state, size_t state_bytes, const Tuning &tuning, qmc_ctx **out)
{
    if (!out) QMC_FAIL((qmc_ctx *)nullptr, QMC_E_ARG, "out is NULL");
    *out = nullptr;
    if (!valid_params(p, g_create_err)) return QMC_E_ARG;
    qmc_ctx *c = new (std::nothrow) qmc_ctx();
    if (!c) QMC_FAIL((qmc_ctx *)nullptr, QMC_E_ARG, "out of host memory");
    c->tuning = tuning;
    c->p = *p;
    c->walkers_per_group.assign(p->walkers_per_group, p->walkers_per_group + p->n_groups);
    c->box_L.assign(p->box_L, p->box_L + p->n_groups);
    c->jastrow_b.assign(p->jastrow_b, p->jastrow_b + p->n_groups);
    c->p.walkers_per_group = c->walkers_per_group.data();
    c->p.box_L = c->box_L.data();
    c->p.jastrow_b = c->jastrow_b.data();
    c->stream = (cudaStream_t)cuda_stream;
    c->ld = round_up4(p->N);
    long long W = 0;
    for (int g = 0; g < p->n_groups; ++g) W += p->walkers_per_group[g];
    c->W = (int32_t)W;
    c->W_total = (int32_t)W;

#define CREATE_FAIL(code, ...) do { snprintf(g_create_err, 512, __VA_ARGS__); qmc_destroy(c); return (code); } while (0)
#define CREATE_CUDA(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) CREATE_FAIL(QMC_E_CUDA, "%s: %s", #expr, cudaGetErrorString(e__)); } while (0)

    int dev = 0;
    CREATE_CUDA(cudaGetDevice(&dev));
    CREATE_CUDA(cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev));

    // per-group constants
    c->groups.resize(p->n_groups);
    for (int g = 0; g < p->n_groups; ++g) {
        GroupDev &G = c->groups[g];
        const double LA = p->box_L[g], b = p->jastrow_b[g];
        // coordinate unit: Angstrom in FP64, the box edge in FP32C
        const double unit = (p->mode == QMC_FP64) ? 1.0 : LA;
        G.unit = unit; G.inv_unit = 1.0 / unit; G.origin = (p->mode == QMC_FP64) ? 0.0 : 1.0;
        G.L_A = LA;
        G.L = (p->mode == QMC_FP64) ? LA : 1.0;
        G.h = 0.5 * G.L; G.h2 = G.h * G.h;
        const double bu = b / unit;
        G.b5 = bu * bu * bu * bu * bu;
        G.c1 = -0.5 * G.b5;
        const double h = G.h;
        G.c0 = G.b5 / (h * h * h * h * h);
        G.sh = 2.0 / (h * h * h * h * h);
        G.step = 0.0;
        long long k = 1;
        while (4 * k * k * k < p->N) ++k;
        G.k_lat = (int32_t)k;
        G.a_lat = LA / (double)k;
        G.pad = 0;
        const double *a = p->aziz;
        const double rm = a[1] / unit;
        G.az.eps = a[0]; G.az.inv_rm = 1.0 / rm; G.az.rm2 = rm * rm; G.az.A = a[2];
        G.az.alpha = a[3]; G.az.beta = a[4]; G.az.c6 = a[5]; G.az.c8 = a[6]; G.az.c10 = a[7];
        G.az.D = a[8]; G.az.Drm = a[8] * rm;
        G.az.f32_scale = (p->mode == QMC_FP64) ? 1.0 : e32::aziz_f32_scale(G.az);
    }

    // state buffer
    size_t pos_bytes, S_off, acc_off, total;
    state_layout(p, W, &pos_bytes, &S_off, &acc_off, &total);
    if (d_state) {
        if (state_bytes < total) CREATE_FAIL(QMC_E_ARG, "state buffer too small: %zu < %zu bytes", state_bytes, total);
        if (((uintptr_t)d_state & 255) != 0) CREATE_FAIL(QMC_E_ARG, "state buffer must be 256-byte aligned");
        c->d_state = d_state;
    } else {
        CREATE_CUDA(cudaMalloc(&c->d_state, total));
        c->owns_state = true;
    }
    std::vector<int32_t> group_of((size_t)W);
    {
        size_t w = 0;
        for (int g = 0; g < p->n_groups; ++g)
            for (int k = 0; k < p->walkers_per_group[g]; ++k) group_of[w++] = g;
    }
    CREATE_CUDA(cudaMalloc(&c->d_groups, sizeof(GroupDev) * p->n_groups));
    CREATE_CUDA(cudaMalloc(&c->d_group_of, sizeof(int32_t) * (size_t)W));
    CREATE_CUDA(cudaMalloc(&c->d_scratch, sizeof(double) * ((size_t)W * 5 + (size_t)W * 3 * p->N)));
    CREATE_CUDA(cudaMemcpyAsync(c->d_groups, c->groups.data(), sizeof(GroupDev) * p->n_groups, cudaMemcpyHostToDevice, c->stream));
    CREATE_CUDA(cudaMemcpyAsync(c->d_group_of, group_of.data(), sizeof(int32_t) * (size_t)W, cudaMemcpyHostToDevice, c->stream));
    CREATE_CUDA(cudaStreamSynchronize(c->stream));

    c->sv.pos = c->d_state;
    c->sv.S = reinterpret_cast<double *>((char *)c->d_state + S_off);
    c->sv.n_acc = reinterpret_cast<unsigned long long *>((char *)c->d_state + acc_off);
    c->sv.group_of = c->d_group_of;
    c->sv.groups = c->d_groups;
    c->sv.W = c->W; c->sv.N = p->N; c->sv.ld = c->ld;
    c->sv.walker_id_base = p->walker_id_base;
    c->sv.proposal = 0;

    if (!plan_sweep(c, &c->sweep_plan))
        CREATE_FAIL(QMC_E_CAPACITY, "N = %d does not fit the sweep kernel's shared-memory budget in mode %d "
                    "(needs %d bytes per CTA, limit %d)", p->N, p->mode, c->sweep_plan.smem_bytes, 227 * 1024);
    if (!plan_energy(c, &c->energy_plan))
        CREATE_FAIL(QMC_E_CAPACITY, "N = %d does not fit the energy kernel's shared-memory budget in mode %d", p->N, p->mode);

    zero_state_kernel<<<c->sm_count * 4, 256, 0, c->stream>>>(c->sv, pos_bytes);
    CREATE_CUDA(cudaGetLastError());
    CREATE_CUDA(cudaStreamSynchronize(c->stream));
    c->launches += 1;
    *out = c;
    snprintf(g_create_err, 512, "no error");
    return QMC_OK;
}

extern "C" int qmc_destroy(qmc_ctx *c)
{
    if (!c) return QMC_OK;
    cudaStreamSynchronize(c->stream);
    if (c->owns_state && c->d_state) cudaFree(c->d_state);
    if (c->d_groups) cudaFree(c->d_groups);
    if (c->d_group_of) cudaFree(c->d_group_of);
    if (c->d_scratch) cudaFree(c->d_scratch);
    if (c->d_enc) cudaFree(c->d_enc);
    if (c->d_epart) cudaFree(c->d_epart);
    if (c->out_stream) cudaStreamSynchronize(c->out_stream);
    if (c->d_block) cudaFree(c->d_block);
    if (c->d_block_xyz) cudaFree(c->d_block_xyz);
    for (cudaStream_t st : {c->hs_in, c->hs_out, c->hs_cmp[0], c->hs_cmp[1]}) if (st) { cudaStreamSynchronize(st); cudaStreamDestroy(st); }
    for (int k = 0; k < qmc::kHostChunksMax; ++k) {
        if (c->hs_ev_in[k]) cudaEventDestroy(c->hs_ev_in[k]);
        if (c->hs_ev_cmp[k]) cudaEventDestroy(c->hs_ev_cmp[k]);
    }
    if (c->hs_ev_fork) cudaEventDestroy(c->hs_ev_fork);
    if (c->hs_ev_join) cudaEventDestroy(c->hs_ev_join);
    if (c->d_hS) cudaFree(c->d_hS);
    for (int k = 0; k < 2; ++k) {
        if (c->ev_ready[k]) cudaEventDestroy(c->ev_ready[k]);
        if (c->ev_copied[k]) cudaEventDestroy(c->ev_copied[k]);
    }
    if (c->out_stream) cudaStreamDestroy(c->out_stream);
    delete c;
    return QMC_OK;
}

extern "C" const char *qmc_last_error(const qmc_ctx *c) { return c ? c->err : g_create_err; }

extern "C" int qmc_init_walkers(qmc_ctx *c, uint64_t seed)
{
    if (!c) return QMC_E_ARG;
    c->seed = seed;
    c->t = 0;
    c->t_acc0 = 0;
    c->trace.offset = 0;
    QMC_CUDA(c, cudaMemsetAsync(c->sv.n_acc, 0, sizeof(unsigned long long) * (size_t)c->W, c->stream));
    QMC_CUDA(c, launch_init(c));
    QMC_CUDA(c, launch_energy(c, nullptr, false));       // build S_i
    c->have_state = true;
    return QMC_OK;
}

extern "C" int qmc_set_seed(qmc_ctx *c, uint64_t seed, uint32_t t)
{
    if (!c) return QMC_E_ARG;
    c->seed = seed;
    c->t_acc0 += t - c->t;       // keep the attempted-move count of qmc_acceptance unchanged
    c->t = t;
    return QMC_OK;
}

extern "C" int qmc_set_proposal(qmc_ctx *c, int32_t kind)
{
    if (!c) return QMC_E_ARG;
    if (kind != 0 && kind != 1) QMC_FAIL(c, QMC_E_ARG, "unknown proposal kind %d", kind);
    c->sv.proposal = kind;
    return QMC_OK;
}

extern "C" int qmc_sweep(qmc_ctx *c, int32_t n_sweeps, const double *steps)
{
    if (!c) return QMC_E_ARG;
    if (!c->have_state) QMC_FAIL(c, QMC_E_STATE, "qmc_sweep before qmc_init_walkers / qmc_set_positions");
    if (n_sweeps < 0 || !steps) QMC_FAIL(c, QMC_E_ARG, "n_sweeps >= 0 and steps != NULL required");
    if (n_sweeps == 0) return QMC_OK;
    if ((long long)n_sweeps * c->p.N >= (1LL << 31)) QMC_FAIL(c, QMC_E_ARG, "n_sweeps * N must stay below 2^31 per call");
    bool changed = false;
    for (int g = 0; g < c->p.n_groups; ++g) {
        // proposal 1: |z| <= sqrt(66 ln 2) < 6.77 with 32-bit uniforms; the displacement must stay below L/2
        const double reach = c->sv.proposal == 1 ? 6.77 : 1.0;
        if (!(steps[g] > 0.0) || !(steps[g] * reach < 0.5 * c->box_L[g]))
            QMC_FAIL(c, QMC_E_ARG, "steps[%d] = %g must lie in (0, L/2 = %g)%s", g, steps[g], 0.5 * c->box_L[g],
                     c->sv.proposal == 1 ? " after multiplication by 6.77 (largest Gaussian variate)" : "");
        if (c->groups[g].step != steps[g]) { c->groups[g].step = steps[g]; changed = true; }
    }
    if (changed)   // stream-ordered update of the small constant table (host mirror is ours, pageable copy is synchronous to the host)
        QMC_CUDA(c, cudaMemcpyAsync(c->d_groups, c->groups.data(), sizeof(GroupDev) * c->p.n_groups, cudaMemcpyHostToDevice, c->stream));
    if (c->sweep_plan.cluster > 1 && c->sweep_plan.fallback == nullptr && (c->sv.proposal != 0 || c->wo.xyz != nullptr))
        QMC_FAIL(c, QMC_E_ARG, "the cluster sweep kernel (N = %d on %d blocks per walker) takes proposal 0 and no in-kernel write-outs, "
                 "and no single thread block can hold a walker of this size", c->p.N, c->sweep_plan.cluster);
    {
        NvtxRange r("qmc_sweep");
        QMC_CUDA(c, launch_sweep(c, n_sweeps));
    }
    c->t += (uint32_t)n_sweeps;
    if (c->trace.dec) c->trace.offset += (long long)n_sweeps * c->p.N;
    return QMC_OK;
}

extern "C" int qmc_sweep_writeouts(qmc_ctx *c, int32_t n_sweeps, const double *steps, int32_t every,
                                   double *xyz_out, uint64_t *n_acc_out, int32_t *flags)
{
    if (!c) return QMC_E_ARG;
    if (every < 1 || !xyz_out || !flags) QMC_FAIL(c, QMC_E_ARG, "every >= 1, xyz_out and flags are required");
    c->wo.xyz = xyz_out;
    c->wo.n_acc = reinterpret_cast<unsigned long long *>(n_acc_out);
    c->wo.flag = flags;
    c->wo.every = every;
    c->wo.n_out = n_sweeps / every;
    const int rc = qmc_sweep(c, n_sweeps, steps);
    c->wo = WriteoutView{};
    return rc;
}

extern "C" int qmc_local_energy(qmc_ctx *c, double *d_out)
{
    if (!c || !d_out) return QMC_E_ARG;
    if (!c->have_state) QMC_FAIL(c, QMC_E_STATE, "qmc_local_energy before qmc_init_walkers / qmc_set_positions");
    NvtxRange r("qmc_local_energy");
    QMC_CUDA(c, launch_energy(c, d_out, true));
    return QMC_OK;
}

extern "C" int qmc_pair_histogram(qmc_ctx *c, int32_t nbins, uint32_t *d_hist)
{
    if (!c || !d_hist) return QMC_E_ARG;
    if (!c->have_state) QMC_FAIL(c, QMC_E_STATE, "qmc_pair_histogram before qmc_init_walkers / qmc_set_positions");
    if (nbins < 1 || nbins > 8192) QMC_FAIL(c, QMC_E_ARG, "nbins = %d must lie in [1, 8192]", nbins);
    if (!pair_histogram_fits(c->p.N, nbins, c->p.mode))
        QMC_FAIL(c, QMC_E_CAPACITY, "N = %d with %d bins does not fit the histogram kernel's shared memory", c->p.N, nbins);
    QMC_CUDA(c, launch_pair_histogram(c, nbins, d_hist));
    return QMC_OK;
}

extern "C" int qmc_refresh_pair_sums(qmc_ctx *c)
{
    if (!c) return QMC_E_ARG;
    if (!c->have_state) QMC_FAIL(c, QMC_E_STATE, "no walker state yet");
    QMC_CUDA(c, launch_energy(c, nullptr, false));
    return QMC_OK;
}

extern "C" int qmc_acceptance(qmc_ctx *c, double *d_out)
{
    if (!c || !d_out) return QMC_E_ARG;
    QMC_CUDA(c, launch_acceptance(c, d_out));
    return QMC_OK;
}

extern "C" int qmc_get_positions(qmc_ctx *c, double *d_xyz)
{
    if (!c || !d_xyz) return QMC_E_ARG;
    QMC_CUDA(c, launch_get_positions(c, d_xyz));
    return QMC_OK;
}

extern "C" int qmc_set_positions(qmc_ctx *c, const double *d_xyz)
{
    if (!c || !d_xyz) return QMC_E_ARG;
    QMC_CUDA(c, launch_set_positions(c, d_xyz));
    QMC_CUDA(c, launch_energy(c, nullptr, false));
    c->t_acc0 = c->t;
    c->have_state = true;
    return QMC_OK;
}

extern "C" int qmc_get_pair_sums(qmc_ctx *c, double *d_S)
{
    if (!c || !d_S) return QMC_E_ARG;
    c->launches += 1;
    get_pair_sums_kernel<<<grid_wn(c, c->p.N), 128, 0, c->stream>>>(c->sv, d_S);
    QMC_CUDA(c, cudaGetLastError());
    return QMC_OK;
}

extern "C" int qmc_trace_decisions(qmc_ctx *c, int32_t w_begin, int32_t w_end, uint8_t *d_dec, double *d_margin,
                                   int64_t moves_capacity)
{
    if (!c) return QMC_E_ARG;
    if (d_dec && (w_begin < 0 || w_end > c->W || w_begin >= w_end || moves_capacity <= 0))
        QMC_FAIL(c, QMC_E_ARG, "bad trace window [%d,%d) or capacity", w_begin, w_end);
    c->trace.dec = d_dec;
    c->trace.margin = d_dec ? d_margin : nullptr;
    c->trace.w_begin = w_begin;
    c->trace.w_end = w_end;
    c->trace.capacity = moves_capacity;
    c->trace.offset = 0;
    return QMC_OK;
}

// A walker sub-range [w0, w0 + wc) of the context as a context of its own for the launch helpers: state pointers
// advanced, W and walker_id_base adjusted, work on `stream`.  Restores everything on destruction.
namespace {
struct RangeGuard {
    qmc_ctx *c; StateView sv0; int32_t W0; cudaStream_t st0;
    RangeGuard(qmc_ctx *ctx, int w0, int wc, cudaStream_t stream) : c(ctx), sv0(ctx->sv), W0(ctx->W), st0(ctx->stream)
    {
        const size_t real = c->p.mode == QMC_FP64 ? 8 : 4;
        c->sv.pos = (char *)sv0.pos + (size_t)w0 * 3 * c->ld * real;
        c->sv.S = sv0.S + (size_t)w0 * c->ld;
        c->sv.n_acc = sv0.n_acc + w0;
        c->sv.group_of = sv0.group_of + w0;
        c->sv.W = wc;
        c->sv.walker_id_base = sv0.walker_id_base + (uint32_t)w0;
        c->W = wc;
        c->stream = stream;
    }
    ~RangeGuard() { c->sv = sv0; c->W = W0; c->stream = st0; }
};
}  // namespace

extern "C" int qmc_step_host(qmc_ctx *c, const double *h_xyz_in, const double *h_S_in, int32_t n_sweeps, const double *steps,
                             double *h_energy, double *h_acc, double *h_xyz_out, double *h_S_out)
{
    if (!c) return QMC_E_ARG;
    if (h_S_in && !h_xyz_in) QMC_FAIL(c, QMC_E_ARG, "h_S_in needs h_xyz_in (the pair sums belong to the uploaded coordinates)");
    if (!h_xyz_in && !c->have_state) QMC_FAIL(c, QMC_E_STATE, "qmc_step_host without coordinates before qmc_init_walkers / qmc_set_positions");
    if (n_sweeps < 0 || (n_sweeps > 0 && !steps)) QMC_FAIL(c, QMC_E_ARG, "n_sweeps >= 0 and steps != NULL required");
    if ((long long)n_sweeps * c->p.N >= (1LL << 31)) QMC_FAIL(c, QMC_E_ARG, "n_sweeps * N must stay below 2^31 per call");
    const size_t Wt = (size_t)c->W, N = (size_t)c->p.N;
    // first use: copy-in / copy-out / two compute streams and the per-chunk events (all or nothing)
    if (!c->host_ready) {
        cudaError_t e = cudaSuccess;
        cudaStream_t *st[4] = {&c->hs_in, &c->hs_out, &c->hs_cmp[0], &c->hs_cmp[1]};
        for (auto p : st) if (e == cudaSuccess) e = cudaStreamCreateWithFlags(p, cudaStreamNonBlocking);
        for (int k = 0; k < kHostChunksMax && e == cudaSuccess; ++k) {
            e = cudaEventCreateWithFlags(&c->hs_ev_in[k], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->hs_ev_cmp[k], cudaEventDisableTiming);
        }
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->hs_ev_fork, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->hs_ev_join, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaMalloc(&c->d_hS, sizeof(double) * Wt * N);
        if (e != cudaSuccess) {
            for (auto p : st) if (*p) { cudaStreamDestroy(*p); *p = nullptr; }
            for (int k = 0; k < kHostChunksMax; ++k) {
                if (c->hs_ev_in[k]) { cudaEventDestroy(c->hs_ev_in[k]); c->hs_ev_in[k] = nullptr; }
                if (c->hs_ev_cmp[k]) { cudaEventDestroy(c->hs_ev_cmp[k]); c->hs_ev_cmp[k] = nullptr; }
            }
            if (c->hs_ev_fork) { cudaEventDestroy(c->hs_ev_fork); c->hs_ev_fork = nullptr; }
            if (c->hs_ev_join) { cudaEventDestroy(c->hs_ev_join); c->hs_ev_join = nullptr; }
            if (c->d_hS) { cudaFree(c->d_hS); c->d_hS = nullptr; }
            QMC_FAIL(c, QMC_E_CUDA, "qmc_step_host set-up: %s", cudaGetErrorString(e));
        }
        c->host_ready = true;
    }
    // proposal steps -> constant table (once, before the fork)
    if (n_sweeps > 0) {
        bool changed = false;
        for (int g = 0; g < c->p.n_groups; ++g) {
            const double reach = c->sv.proposal == 1 ? 6.77 : 1.0;
            if (!(steps[g] > 0.0) || !(steps[g] * reach < 0.5 * c->box_L[g]))
                QMC_FAIL(c, QMC_E_ARG, "steps[%d] = %g must lie in (0, L/2 = %g)", g, steps[g], 0.5 * c->box_L[g]);
            if (c->groups[g].step != steps[g]) { c->groups[g].step = steps[g]; changed = true; }
        }
        if (changed)
            QMC_CUDA(c, cudaMemcpyAsync(c->d_groups, c->groups.data(), sizeof(GroupDev) * c->p.n_groups, cudaMemcpyHostToDevice, c->stream));
    }
    // walkers in chunks (l.175, l.319-323: transfers masked by computation): chunk k's upload, compute and download
    // run on three streams, so that chunk k+1 uploads and chunk k-1 downloads while chunk k computes; two compute
    // streams let the sweep of one chunk share the GPU with the energy pass of the previous one.  A decision trace
    // (walker indices of the whole context) or few walkers keep everything in one chunk.
    int nchunk = c->tuning.host_chunks > 0 ? c->tuning.host_chunks : 4;
    if (nchunk > kHostChunksMax) nchunk = kHostChunksMax;
    while (nchunk > 1 && (int)Wt / nchunk < c->sm_count) --nchunk;
    if (c->trace.dec) nchunk = 1;
    if (h_xyz_in) c->t_acc0 = c->t;                             // set_positions zeroes the counters
    const double attempted = (double)(c->t + (uint32_t)n_sweeps - c->t_acc0) * (double)N;
    double *d_e = c->d_scratch, *d_a = c->d_scratch + 4 * Wt, *d_x = c->d_scratch + 5 * Wt;
    NvtxRange range("qmc_step_host");
    QMC_CUDA(c, cudaEventRecord(c->hs_ev_fork, c->stream));
    for (cudaStream_t st : {c->hs_in, c->hs_out, c->hs_cmp[0], c->hs_cmp[1]}) QMC_CUDA(c, cudaStreamWaitEvent(st, c->hs_ev_fork, 0));
    for (int k = 0; k < nchunk; ++k) {
        const int w0 = (int)((long long)Wt * k / nchunk), w1 = (int)((long long)Wt * (k + 1) / nchunk), wc = w1 - w0;
        cudaStream_t cs = c->hs_cmp[k & 1];
        double *dxk = d_x + (size_t)w0 * 3 * N, *dSk = c->d_hS + (size_t)w0 * N;
        if (h_xyz_in) {
            QMC_CUDA(c, cudaMemcpyAsync(dxk, h_xyz_in + (size_t)w0 * 3 * N, sizeof(double) * wc * 3 * N, cudaMemcpyHostToDevice, c->hs_in));
            if (h_S_in) QMC_CUDA(c, cudaMemcpyAsync(dSk, h_S_in + (size_t)w0 * N, sizeof(double) * wc * N, cudaMemcpyHostToDevice, c->hs_in));
            QMC_CUDA(c, cudaEventRecord(c->hs_ev_in[k], c->hs_in));
            QMC_CUDA(c, cudaStreamWaitEvent(cs, c->hs_ev_in[k], 0));
        }
        {
            RangeGuard view(c, w0, wc, cs);
            if (h_xyz_in) {
                QMC_CUDA(c, launch_set_positions(c, dxk));
                if (h_S_in) QMC_CUDA(c, launch_raw_sums(c, dSk, true));
                else        QMC_CUDA(c, launch_energy(c, nullptr, false));      // rebuild S_i from the coordinates
            }
            if (n_sweeps > 0) QMC_CUDA(c, launch_sweep(c, n_sweeps));
            if (h_energy) QMC_CUDA(c, launch_energy(c, d_e + (size_t)w0 * 4, true));
            if (h_acc) QMC_CUDA(c, launch_acceptance_attempted(c, attempted, d_a + w0));
            if (h_xyz_out) QMC_CUDA(c, launch_get_positions(c, dxk));
            if (h_S_out) QMC_CUDA(c, launch_raw_sums(c, dSk, false));
        }
        QMC_CUDA(c, cudaEventRecord(c->hs_ev_cmp[k], cs));
        QMC_CUDA(c, cudaStreamWaitEvent(c->hs_out, c->hs_ev_cmp[k], 0));
        if (h_energy) QMC_CUDA(c, cudaMemcpyAsync(h_energy + (size_t)w0 * 4, d_e + (size_t)w0 * 4, sizeof(double) * 4 * wc, cudaMemcpyDeviceToHost, c->hs_out));
        if (h_acc) QMC_CUDA(c, cudaMemcpyAsync(h_acc + w0, d_a + w0, sizeof(double) * wc, cudaMemcpyDeviceToHost, c->hs_out));
        if (h_xyz_out) QMC_CUDA(c, cudaMemcpyAsync(h_xyz_out + (size_t)w0 * 3 * N, dxk, sizeof(double) * wc * 3 * N, cudaMemcpyDeviceToHost, c->hs_out));
        if (h_S_out) QMC_CUDA(c, cudaMemcpyAsync(h_S_out + (size_t)w0 * N, dSk, sizeof(double) * wc * N, cudaMemcpyDeviceToHost, c->hs_out));
    }
    // join: the context's stream continues after everything; then the host waits
    for (cudaStream_t st : {c->hs_in, c->hs_out, c->hs_cmp[0], c->hs_cmp[1]}) {
        QMC_CUDA(c, cudaEventRecord(c->hs_ev_join, st));
        QMC_CUDA(c, cudaStreamWaitEvent(c->stream, c->hs_ev_join, 0));
    }
    c->t += (uint32_t)n_sweeps;
    if (c->trace.dec) c->trace.offset += (long long)n_sweeps * c->p.N;
    if (h_xyz_in) c->have_state = true;
    QMC_CUDA(c, cudaStreamSynchronize(c->stream));
    return QMC_OK;
}

// Host function of the write-out stream: the block's data have landed, raise its flag.
static void CUDART_CB raise_flag(void *flag) { *reinterpret_cast<volatile int32_t *>(flag) = 1; }

extern "C" int qmc_run_blocks_host(qmc_ctx *c, int32_t n_blocks, int32_t sweeps_per_block, const double *steps,
                                   double *h_energy, double *h_acc, int32_t xyz_every, double *h_xyz, int32_t *h_done)
{
    if (!c || !h_energy) return QMC_E_ARG;
    if (!c->have_state) QMC_FAIL(c, QMC_E_STATE, "qmc_run_blocks_host before qmc_init_walkers / qmc_set_positions");
    if (n_blocks < 0 || sweeps_per_block < 1) QMC_FAIL(c, QMC_E_ARG, "n_blocks >= 0 and sweeps_per_block >= 1 required");
    if (h_xyz && xyz_every < 1) QMC_FAIL(c, QMC_E_ARG, "xyz_every >= 1 required with h_xyz");
    const size_t W = (size_t)c->W, N = (size_t)c->p.N;
    // first use: write-out stream, double-buffered results, events.  Everything or nothing: a failure half way
    // leaves no half-initialised state behind for the next call.
    if (!c->blocks_ready) {
        auto undo = [&]() {
            if (c->out_stream) { cudaStreamDestroy(c->out_stream); c->out_stream = nullptr; }
            if (c->d_block) { cudaFree(c->d_block); c->d_block = nullptr; }
            for (int k = 0; k < 2; ++k) {
                if (c->ev_ready[k]) { cudaEventDestroy(c->ev_ready[k]); c->ev_ready[k] = nullptr; }
                if (c->ev_copied[k]) { cudaEventDestroy(c->ev_copied[k]); c->ev_copied[k] = nullptr; }
            }
        };
        cudaError_t e = cudaStreamCreateWithFlags(&c->out_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaMalloc(&c->d_block, sizeof(double) * 2 * W * 5);
        for (int k = 0; k < 2 && e == cudaSuccess; ++k) {
            e = cudaEventCreateWithFlags(&c->ev_ready[k], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_copied[k], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) { undo(); QMC_FAIL(c, QMC_E_CUDA, "qmc_run_blocks_host set-up: %s", cudaGetErrorString(e)); }
        c->blocks_ready = true;
    }
    if (h_xyz && !c->d_block_xyz) QMC_CUDA(c, cudaMalloc(&c->d_block_xyz, sizeof(double) * 2 * W * 3 * N));
    for (int32_t b = 0; b < n_blocks; ++b) {
        const int k = b & 1;
        double *d_e = c->d_block + (size_t)k * W * 5, *d_a = d_e + 4 * W;
        int rc = qmc_sweep(c, sweeps_per_block, steps);
        if (rc != QMC_OK) return rc;
        // buffer k is free again once its last copy has finished -- also the copy of an EARLIER call (waiting on an
        // event that was never recorded is a no-op)
        QMC_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_copied[k], 0));
        if ((rc = qmc_local_energy(c, d_e)) != QMC_OK) return rc;
        if ((rc = qmc_acceptance(c, d_a)) != QMC_OK) return rc;
        const bool with_xyz = h_xyz && ((b + 1) % xyz_every == 0);
        double *d_x = c->d_block_xyz ? c->d_block_xyz + (size_t)k * W * 3 * N : nullptr;
        if (with_xyz && (rc = qmc_get_positions(c, d_x)) != QMC_OK) return rc;
        QMC_CUDA(c, cudaEventRecord(c->ev_ready[k], c->stream));
        // write-out while the next block computes (the paper's asynchronous writeouts, l.175, l.323)
        QMC_CUDA(c, cudaStreamWaitEvent(c->out_stream, c->ev_ready[k], 0));
        QMC_CUDA(c, cudaMemcpyAsync(h_energy + (size_t)b * W * 4, d_e, sizeof(double) * 4 * W, cudaMemcpyDeviceToHost, c->out_stream));
        if (h_acc)
            QMC_CUDA(c, cudaMemcpyAsync(h_acc + (size_t)b * W, d_a, sizeof(double) * W, cudaMemcpyDeviceToHost, c->out_stream));
        if (with_xyz)
            QMC_CUDA(c, cudaMemcpyAsync(h_xyz + (size_t)((b + 1) / xyz_every - 1) * W * 3 * N, d_x, sizeof(double) * W * 3 * N,
                                        cudaMemcpyDeviceToHost, c->out_stream));
        QMC_CUDA(c, cudaEventRecord(c->ev_copied[k], c->out_stream));
        if (h_done) QMC_CUDA(c, cudaLaunchHostFunc(c->out_stream, raise_flag, h_done + b));
    }
    return QMC_OK;
}

extern "C" int qmc_wait(qmc_ctx *c)
{
    if (!c) return QMC_E_ARG;
    QMC_CUDA(c, cudaStreamSynchronize(c->stream));
    if (c->out_stream) QMC_CUDA(c, cudaStreamSynchronize(c->out_stream));
    return QMC_OK;
}

extern "C" int qmc_info(const qmc_ctx *c, qmc_info_t *out)
{
    if (!c || !out) return QMC_E_ARG;
    out->W = c->W; out->N = c->p.N; out->n_groups = c->p.n_groups; out->mode = c->p.mode;
    out->sweep_threads = c->sweep_plan.threads; out->sweep_ctas_per_sm = c->sweep_plan.ctas_per_sm;
    out->sweep_smem_bytes = c->sweep_plan.smem_bytes; out->sweep_pairs_per_thread = c->sweep_plan.J;
    out->energy_threads = c->energy_plan.threads; out->energy_ctas_per_sm = c->energy_plan.ctas_per_sm;
    out->energy_smem_bytes = c->energy_plan.smem_bytes;
    out->sm_count = c->sm_count;
    out->t = c->t;
    out->kernel_launches = c->launches;
    out->sweep_vector = c->sweep_plan.V; out->sweep_pending = c->sweep_plan.P; out->sweep_tile = c->sweep_plan.K;
    out->energy_variant = c->energy_plan.variant;
    out->sweep_cluster = c->sweep_plan.cluster;
    return QMC_OK;
}

extern "C" int qmc_set_tuning(const char *key, int32_t value)
{
    if (!key) { g_tuning = Tuning{}; return QMC_OK; }
    if (tuning_set(g_tuning, key, value)) return QMC_OK;
    snprintf(g_create_err, 512, "qmc_set_tuning: unknown key '%s'", key);
    return QMC_E_ARG;
}
