/*
 * qmc.h -- C ABI of the B200-native He-4 variational Monte Carlo hot path.
 *
 * Implements the per-walker Metropolis sweep of single-particle moves and the
 * local-energy estimator of "Fast quantum Monte Carlo on a GPU" (arXiv:1312.1282;
 * citations below are PAPER.md line numbers, "Rn" are the readings in DESIGN.md).
 *
 * Conventions
 *  - Plain C, no C++ or torch types.  Every call returns QMC_OK (0) or a negative
 *    qmc_status; nothing aborts or throws.  qmc_last_error() gives a message.
 *  - "device" pointers are CUDA device memory owned by the CALLER (e.g. a torch
 *    tensor's data_ptr()); "host" pointers are ordinary host memory (pinned memory
 *    makes the *_host calls asynchronous copies).  The library never frees them.
 *  - All work is enqueued on the CUDA stream given to qmc_create (a cudaStream_t
 *    passed as void*; NULL = legacy default stream) and is asynchronous with respect
 *    to the host, except qmc_create / qmc_destroy and the *_host calls (which
 *    synchronise the stream before returning).
 *  - Units: Angstrom and Kelvin.  Coordinates are SoA per walker: xyz[w][c][i],
 *    c = 0,1,2, i = 0..N-1, i.e. [W][3][N] doubles, wrapped into [0, L].
 *  - Walkers are independent Markov chains (l.169); walker w of this context has
 *    global id walker_id_base + w, which keys its random stream, so a shard of a
 *    larger run reproduces exactly the walkers it owns.
 */
#ifndef QMC_B200_H
#define QMC_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qmc_ctx qmc_ctx;   /* opaque; owned by the library */

typedef enum {
    QMC_OK = 0,
    QMC_E_ARG = -1,        /* bad argument (NULL, N < 2, step >= L/2, ...)                 */
    QMC_E_CAPACITY = -2,   /* N does not fit the mode's per-CTA shared-memory budget        */
    QMC_E_CUDA = -3,       /* a CUDA runtime call failed (message in qmc_last_error)        */
    QMC_E_STATE = -4       /* call order (e.g. sweep before init_walkers/set_positions)     */
} qmc_status;

typedef enum {
    QMC_FP64 = 0,          /* fp64 coordinates and arithmetic throughout                    */
    QMC_FP32C = 1          /* fp32 coordinates + pair arithmetic, fp64 sums (R20)           */
} qmc_mode;

/* Problem statement (l.319 inputs; l.410 run-time fields bulkdimarray, jastrowb, mass).
 * Host memory; copied by qmc_create, the caller keeps ownership. */
typedef struct {
    int32_t        N;                 /* atoms per walker, >= 2                                   */
    int32_t        n_groups;          /* parameter points in this context (>= 1)                  */
    const int32_t *walkers_per_group; /* [n_groups]; W = sum; walkers are numbered group by group */
    const double  *box_L;             /* [n_groups] cubic box edge L (l.460); cutoff is L/2       */
    const double  *jastrow_b;         /* [n_groups] b of Eq.(9) l.155                             */
    double         hbar2_over_2m;     /* K*A^2                                                    */
    double         aziz[9];           /* HFD-B(HE) l.131: eps, rm, A, alpha, beta, c6, c8, c10, D  */
    int32_t        mode;              /* qmc_mode                                                 */
    uint32_t       walker_id_base;    /* global id of this context's walker 0                     */
    double         jitter;            /* half-width of the initial lattice jitter (R13)           */
} qmc_params;

/* Bytes of device memory the walker state of `p` needs (coordinates, per-particle pair
 * sums S_i, counters).  0 on invalid parameters. */
size_t qmc_state_bytes(const qmc_params *p);

/* Create a context.  d_state: caller-owned device buffer of >= qmc_state_bytes(p) bytes,
 * 256-byte aligned, which must outlive the context; or NULL to let the library allocate
 * (cudaMalloc) and free it.  Validates parameters, precomputes per-group constants.
 * Errors: QMC_E_ARG, QMC_E_CAPACITY (e.g. N = 10000 in QMC_FP64), QMC_E_CUDA. */
int qmc_create(const qmc_params *p, void *cuda_stream, void *d_state, size_t state_bytes, qmc_ctx **out);
int qmc_destroy(qmc_ctx *c);

/* Jittered FCC start (R13), pair sums S_i built, counters and sweep index t set to 0. */
int qmc_init_walkers(qmc_ctx *c, uint64_t seed);

/* n_sweeps Metropolis sweeps of every walker (Eq.(5) l.123, Eq.(7) l.146, l.325-331): for each
 * sweep t, for s = 0..N-1: trial r_s + delta with delta uniform in [-step,step]^3 from
 * Philox4x32-10(counter (s,t,walker id,0), key seed); accept iff 2*Delta > log(xi); on accept
 * commit the wrapped position and update the running pair sums.  steps: HOST array [n_groups]
 * (one step per parameter point), 0 < step < L/2.  Successive calls continue t:
 * sweep(a); sweep(b) == sweep(a+b). */
int qmc_sweep(qmc_ctx *c, int32_t n_sweeps, const double *steps);

/* Proposal of the following qmc_sweep calls.  kind 0 (default): particles in order,
 * displacement uniform in [-step,step]^3 (BASELINE.json's reading, R7).  kind 1: the paper's own
 * (l.144, l.325, l.347-349): each of the N moves of a sweep picks a random particle,
 * s = floor(A0 N / 2^32), and displaces it by step * (z0, z1, z2), z standard normal by Box-Muller from
 * Philox4x32-10 words A = (m,t,walker,2), B = (m,t,walker,3) (m = move index within the sweep); step is then the
 * standard deviation per component and must satisfy 6.77 step < L/2.  The variate map is specified to the bit
 * (DESIGN.md "Proposal 1"), so fp64 trajectories still match the oracle move for move. */
int qmc_set_proposal(qmc_ctx *c, int32_t kind);

/* Local energy of every walker's current configuration (l.113-115, l.129, l.381):
 * d_out: device [W][4] = E_PB, V, T_PB, T_JF, totals in K (divide by N for per-atom).
 * Also rebuilds the running pair sums S_i from scratch (R17). */
int qmc_local_energy(qmc_ctx *c, double *d_out);

/* Pair-distance histogram of every walker's current configuration, the raw data of the pair distribution
 * function g(r) (l.421, l.468): d_hist device [W][nbins] uint32, bin k counts the
 * pairs i < j with minimum-image distance r in [k, k+1) * (L/2)/nbins; pairs with r >= L/2 are not counted.
 * The bin of a pair is specified to the bit, so counts are reproducible exactly.
 * Up to 512 bins the kernel decides most pairs from an fp32 estimate and evaluates the specified fp64 arithmetic only
 * near a bin edge (same counts); more bins take the fp64 arithmetic for every pair.
 * 1 <= nbins <= 8192; QMC_E_CAPACITY if 12 N + 4 nbins + 5 KB exceed one CTA's shared memory (N <= ~18 000). */
int qmc_pair_histogram(qmc_ctx *c, int32_t nbins, uint32_t *d_hist);

/* Acceptance ratio, one of the quantities the paper writes out with every block (l.323, l.381; its file
 * acceptance.dat, l.397-406): d_out: device [W] accepted / attempted moves since qmc_init_walkers /
 * qmc_set_positions. */
int qmc_acceptance(qmc_ctx *c, double *d_out);

/* One whole step with HOST buffers (the paper's block cycle, l.319-343: coordinates in, sweeps, energies and
 * coordinates written out).  Any pointer may be NULL to skip that part.  h_xyz_in [W][3][N] is uploaded first; the
 * running pair sums of the uploaded configuration are either uploaded with it (h_S_in [W][N], the h_S_out of an
 * earlier call for the same coordinates: opaque walker state in the library's own unit, sum_j t(r_ij) with
 * u = c1 t) or, with h_S_in = NULL, rebuilt on the device (one more all-pairs pass); then n_sweeps sweeps; then the
 * local energy -> h_energy [W][4], acceptance -> h_acc [W], coordinates -> h_xyz_out [W][3][N], pair sums ->
 * h_S_out [W][N].  The walkers are processed in chunks on internal streams so that the host<->device copies of one
 * chunk run while another chunk computes (l.175, l.319-323: transfers masked by computation); use pinned host
 * memory.  In and out buffers may be the same.  Synchronises before returning. */
int qmc_step_host(qmc_ctx *c, const double *h_xyz_in, const double *h_S_in, int32_t n_sweeps, const double *steps,
                  double *h_energy, double *h_acc, double *h_xyz_out, double *h_S_out);

/* A run of n_blocks blocks with in-flight write-outs (the paper's load masking, l.175, l.323, §4; SURVEY.md §8(f)
 * NEXT-4).  Block b = sweeps_per_block sweeps + local energy + acceptance; its results go to the HOST arrays
 * h_energy[b][W][4] and h_acc[b][W] (may be NULL) on a second stream while block b+1 computes.  If h_xyz is not
 * NULL, every xyz_every-th block (b+1 a multiple of xyz_every >= 1) also writes the walker coordinates out, to
 * h_xyz[(b+1)/xyz_every - 1][W][3][N] (l.323: "walker coordinates ... acceptance ratio, computed potential and
 * kinetic energies").  h_done[b] (host int32, may be NULL; the caller zeroes it) is set to 1 once everything of
 * block b has landed, so the host can analyse block b while the GPU generates the next ones.  Use pinned host
 * memory.  Returns after ENQUEUEING all blocks; qmc_wait (or polling h_done[n_blocks-1]) tells when everything is
 * there.  The buffers must stay valid until then.  Calls may follow each other without qmc_wait in between. */
int qmc_run_blocks_host(qmc_ctx *c, int32_t n_blocks, int32_t sweeps_per_block, const double *steps,
                        double *h_energy, double *h_acc, int32_t xyz_every, double *h_xyz, int32_t *h_done);

/* qmc_sweep with write-outs issued from INSIDE the running kernel (the paper's mechanism itself, l.175, l.323,
 * l.343, Fig. 2; NEXT-4): the walker stays resident in shared memory for all n_sweeps sweeps of the ONE launch, and
 * after every `every` sweeps (m of Fig. 2) each thread block writes its walker's coordinates to
 * xyz_out[k][w][3][N] (Angstrom, k = 0 .. n_sweeps/every - 1) and its accepted-move count since init /
 * set_positions to n_acc_out[k][w] (may be NULL), makes them visible system-wide, and sets flags[k][w] = 1 (the
 * caller zeroes flags first).  The three buffers must be addressable by the device: device memory, or page-locked
 * host memory mapped into the device address space (cudaHostAlloc / torch pin_memory: then the host sees each
 * write-out while the kernel is still running and can analyse it -- the paper's load masking).  Asynchronous like
 * qmc_sweep; the buffers must stay valid until the stream has finished. */
int qmc_sweep_writeouts(qmc_ctx *c, int32_t n_sweeps, const double *steps, int32_t every,
                        double *xyz_out, uint64_t *n_acc_out, int32_t *flags);
/* Blocks until all work of this context (both streams) has finished. */
int qmc_wait(qmc_ctx *c);

/* Message for the last error of this context (or of the last failed qmc_create if c is NULL).
 * Library-owned, valid until the next call. */
const char *qmc_last_error(const qmc_ctx *c);

/* ---- state access and parity hooks (not on the timed path) -------------------------------- */
int qmc_get_positions(qmc_ctx *c, double *d_xyz);        /* device [W][3][N], exact widening in FP32C */
int qmc_set_positions(qmc_ctx *c, const double *d_xyz);  /* device [W][3][N]; rebuilds S_i, zeroes counters,
                                                            keeps the sweep index t and the seed          */
int qmc_set_seed(qmc_ctx *c, uint64_t seed, uint32_t t); /* random key and sweep index for the next sweep  */
int qmc_get_pair_sums(qmc_ctx *c, double *d_S);          /* device [W][N] running S_i                      */
int qmc_refresh_pair_sums(qmc_ctx *c);                   /* S_i <- sum_{j != i} u(r_ij) from scratch       */
/* Record, for walkers w_begin <= w < w_end, one byte per move (1 = accepted) and the decision
 * margin 2*Delta - log(xi) of the following qmc_sweep calls, starting at move 0 of the buffers:
 * d_dec device [(w_end-w_begin)][moves_capacity] uint8, d_margin same shape double (may be NULL).
 * Pass d_dec = NULL to stop recording. */
int qmc_trace_decisions(qmc_ctx *c, int32_t w_begin, int32_t w_end, uint8_t *d_dec, double *d_margin,
                        int64_t moves_capacity);

/* ---- introspection ------------------------------------------------------------------------ */
typedef struct {
    int32_t W, N, n_groups, mode;
    int32_t sweep_threads, sweep_ctas_per_sm, sweep_smem_bytes, sweep_pairs_per_thread;
    int32_t energy_threads, energy_ctas_per_sm, energy_smem_bytes;
    int32_t sm_count;
    uint32_t t;                       /* sweeps done since init                        */
    uint64_t kernel_launches;         /* kernels this context has launched so far      */
    int32_t sweep_vector;             /* particles per shared-memory vector access (V) */
    int32_t sweep_pending;            /* 1: running sums held as fp32 hi + lo (R20)    */
    int32_t sweep_tile;               /* moves per barrier (K; 1 = one-move kernel)    */
    int32_t energy_variant;           /* 0 ordered pairs, 1 fp64 / 2 fp32c unordered pairs, 3 gridded (large N) */
    int32_t sweep_cluster;            /* thread blocks per walker (1; > 1: cluster kernel, distributed shared memory) */
} qmc_info_t;
int qmc_info(const qmc_ctx *c, qmc_info_t *out);

/* qmc_create with this context's own overrides of the launch heuristics: n_keys (key, value) pairs with the keys listed
 * under qmc_set_tuning below; everything not named is left to the heuristics, and the process-wide defaults of
 * qmc_set_tuning are NOT consulted.  Contexts with different forced shapes can coexist and be created from different
 * threads.  keys / values: host arrays, read during the call only.  QMC_E_ARG for an unknown key. */
int qmc_create_tuned(const qmc_params *p, void *cuda_stream, void *d_state, size_t state_bytes,
                     const char *const *keys, const int32_t *values, int32_t n_keys, qmc_ctx **out);

/* Process-wide DEFAULT of those overrides: copied into a context by qmc_create at creation (later changes do not reach
 * it) and ignored by qmc_create_tuned.  A plain global without a lock -- for single-threaded tuning experiments and
 * tests; use qmc_create_tuned otherwise.  The heuristics themselves (no override) are what bench.py times.  Keys: "sweep_threads", "sweep_per_thread", "sweep_vector",
 * "sweep_pending", "sweep_tile" (1 = one-move kernel, 2 / 4 = tile kernel), "sweep_cluster", "energy_threads",
 * "energy_ordered" (1 = ordered-pair energy kernels), "host_chunks" (walker chunks of qmc_step_host, 1..8).  value: the wanted number, or -1 (0 for the energy keys) for
 * "heuristic".  key == NULL resets everything.  A shape that is not compiled or does not fit N falls back to the
 * heuristic.  Returns QMC_E_ARG for an unknown key. */
int qmc_set_tuning(const char *key, int32_t value);

/* ---- local energy without any allocation --------------------------------------------------------------
 * qmc_local_energy_fp32c_static: the FP32C local energy (same quantities as qmc_local_energy: l.113-115, l.129,
 * l.381; HFD-B(HE) l.131, Eq.(9) l.155, box l.460) of W walkers of N atoms, one parameter point, WITHOUT a
 * qmc_ctx and without allocating anything: no cudaMalloc / cudaFree / cudaHostAlloc, no host heap, no library
 * routine that allocates.
 *
 * Who needs it.  qmc_create reserves device memory with cudaMalloc, and qmc_local_energy's gridded kernel reserves
 * its working arrays with cudaMalloc the first time it runs.  Some hosts of this library cannot do that:
 *  - a process whose device memory is already handed out in full to a pool (a tensor framework's caching allocator,
 *    a job scheduler's per-tenant budget): cudaMalloc then fails with out-of-memory although the pool has room;
 *  - a latency-bound loop (an analysis or steering step between blocks of sweeps, l.319-343): cudaMalloc and
 *    cudaFree may synchronise the whole device and would stall every other stream of the process;
 *  - code that is only given the buffers it may touch (a plugin or callback run by another runtime) and has no
 *    licence to create device memory of its own.
 * Such a caller passes its input and output buffers, and the working memory (fixed-point coordinates, the rebuilt
 * pair sums S_i, per-thread-block partial sums, the parameter tables) is ONE array of QMC_STATIC_SCRATCH_BYTES
 * (5 382 656 bytes, about 5.1 MiB) that is part of the library image: every GPU on which the library's kernels
 * get loaded holds it from then until the process exits, whether this call is ever used or not.
 *
 * Limits: 1 <= W <= QMC_STATIC_MAX_WALKERS, 2 <= N <= QMC_STATIC_MAX_ATOMS and W * (N rounded up to a multiple of
 * 32) <= QMC_STATIC_MAX_SLOTS (e.g. 128 walkers of 1952-2048 atoms, 26 of 10000, 6 of 40960).  Anything larger is
 * refused with QMC_E_CAPACITY and a message that names the three limits; nothing is launched in that case.
 *
 * Arguments.  d_xyz: device [W][3][N] doubles, Angstrom, in [0, L] (the layout of qmc_set_positions; rounded to the
 * FP32C grid of L 2^-23 exactly as qmc_set_positions does).  box_L, jastrow_b, aziz[9], hbar2_over_2m: as in
 * qmc_params (host values; aziz is a host array of 9).  d_out: device [W][4] doubles = E_PB, V, T_PB, T_JF in K, as
 * qmc_local_energy writes them (bit-identical to a QMC_FP32C context of the same W and N running the gridded energy
 * kernel on this GPU).  cuda_stream: a cudaStream_t as void*, NULL = legacy default stream; the four kernels are
 * enqueued there and the call returns without waiting.  err / err_len: optional host buffer that receives the
 * message when the return value is not QMC_OK (there is no context to ask; qmc_last_error does not see this call).
 * The caller owns every buffer; none is kept after the kernels have run.
 *
 * First call on a device.  The first call made while a given device is current looks up the device address of
 * the static array (cudaGetSymbolAddress) and the SM count, and caches both; later calls on that device skip this.
 * Make that first call during set-up, before any stream capture is begun.  The first call for a given
 * (aziz, box_L) also spends a few milliseconds of HOST time on the fp32 amplitude scale (R22); the last pair is
 * remembered.
 *
 * Sharing.  All calls in the process that target the same GPU use the SAME array, from whatever thread or stream.
 * Calls enqueued on one stream follow each other and are safe.  Calls whose kernels can overlap on the GPU
 * (different streams, or different host threads on different streams) overwrite each other's working memory and
 * give wrong energies without any error: order them with events or keep them on one stream.  The array still
 * holds the previous call's data when the next one starts; each call rewrites every word it later reads (tables,
 * coordinates including the padding up to a multiple of 32, pair sums, partial sums), so no clearing is asked of
 * the caller.  Host-side bookkeeping is guarded by a mutex; the call is safe to make from several threads.
 * Errors: QMC_E_ARG (NULL pointer, N < 2, W < 1, box_L <= 0, jastrow_b < 0, r_m <= 0), QMC_E_CAPACITY (above),
 * QMC_E_CUDA (a runtime call or a launch failed; message in err). */
#define QMC_STATIC_MAX_WALKERS   4096
#define QMC_STATIC_MAX_ATOMS     65536
#define QMC_STATIC_MAX_SLOTS     262144
#define QMC_STATIC_SCRATCH_BYTES 5382656
int qmc_local_energy_fp32c_static(const double *d_xyz, int32_t W, int32_t N, double box_L, double jastrow_b,
                                  const double *aziz, double hbar2_over_2m, double *d_out, void *cuda_stream,
                                  char *err, size_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* QMC_B200_H */
