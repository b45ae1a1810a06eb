/*
 * vmc_oracle.c -- plain, slow, fp64 CPU oracle of the He-4 VMC hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may call it.
 * It shares no code, header, table or constant generator with the CUDA path
 * (paper_1312_1282_b200/csrc); the two implement the same written definitions
 * (DESIGN.md "Definitions" + "Readings") independently.
 *
 * Everything is written as the definition reads: sequential loops, one pair at
 * a time, no running sums, no blocking, no reordering.  Units: Angstrom, Kelvin.
 * Compile with -O2 -ffp-contract=off (no FMA contraction: the committed
 * coordinates r_s + delta must round exactly once, see orc_sweep).
 *
 * Citations are PAPER.md line numbers (arxiv 1312.1282) and DESIGN.md readings
 * R1..R21.  Parity pins: tests/test_oracle_pins.py (every function below is
 * pinned there, including the proposal-1 variates and the pair histogram;
 * nothing in this file is "parity unpinned").
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t N;        /* atoms                                              */
    double  L;        /* cubic box edge                    */
    double  b;        /* Jastrow parameter of Eq.(9), l.155                 */
    double  Dk;       /* hbar^2/2m, K*A^2                                   */
    double  aziz[9];  /* eps, rm, A, alpha, beta, c6, c8, c10, D  (R3)      */
    int32_t proposal; /* 0: particles in order, uniform cube (R7); 1: the paper's random particle +
                         Gaussian displacement (l.144, l.325)               */
} orc_sys;

/* ---------------------------------------------------------------------------
 * Philox4x32-10 (Salmon et al. 2011, public algorithm; BASELINE.json names it).
 * One round: (c0,c1,c2,c3) -> (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0));
 * the key is bumped by (W0,W1) between rounds; 10 rounds.
 * ------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += W0; k1 += W1; }
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Exact integer -> double maps (R7/R8): a in (-1,1), xi in (0,1); no rounding. */
static double unit_pm1(uint32_t x) { return ((double)x + 0.5) * (1.0 / 2147483648.0) - 1.0; }
static double unit_01(uint32_t x)  { return ((double)x + 0.5) * (1.0 / 4294967296.0); }

/* Variates of move (particle s, sweep t, walker w): counter (s,t,w,0), key = seed.
 * delta[k] = step * a_k (ONE rounding), xi in (0,1).  DESIGN.md "Randomness". */
void orc_move_variates(uint64_t seed, uint32_t w, uint32_t t, uint32_t s, double step,
                       double delta[3], double *xi)
{
    uint32_t ctr[4] = { s, t, w, 0u };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t x[4];
    orc_philox4x32_10(ctr, key, x);
    for (int k = 0; k < 3; ++k) delta[k] = step * unit_pm1(x[k]);
    *xi = unit_01(x[3]);
}

/* ---------------------------------------------------------------------------
 * Proposal 1 (the paper's own, l.144 "a randomly selected particle", l.325 "Gaussian displacements" made
 * by a Box-Muller kernel, l.347-349): written so that both implementations can reproduce every bit with
 * IEEE +, -, *, /, sqrt alone; no library log / sin / cos.
 *
 *   ln u for u = (2 w + 1) 2^-33, w a 32-bit word: n = 2w + 1 = m 2^e, m in [1,2); m > sqrt2 -> m/2, e+1;
 *   s = (m-1)/(m+1), ln m = 2 s P(s^2), P = sum_{k=0..10} s^2k/(2k+1) by Horner; ln u = ln m + (e-33) ln2.
 *   cos, sin of 2 pi v for v = (w + 0.5) 2^-32: quadrant q = w >> 30, f = ((w & (2^30-1)) + 0.5) 2^-30;
 *   f > 1/2: swap sin and cos of g = 1 - f; x = g pi/2 in (0, pi/4]; Taylor to x^15 / x^16 by Horner in x^2.
 * ------------------------------------------------------------------------- */
static double orc_ln_unit(uint32_t w)
{
    uint64_t n = 2ull * (uint64_t)w + 1ull;
    int e = 0;
    while ((n >> (e + 1)) != 0ull) ++e;                   /* e = floor(log2 n) */
    double m = (double)n / (double)(1ull << e);           /* exact: n < 2^33 */
    if (m > 1.4142135623730951) { m = 0.5 * m; e += 1; }
    const double s = (m - 1.0) / (m + 1.0);
    const double s2 = s * s;
    double P = 1.0 / 21.0;
    for (int k = 9; k >= 0; --k) P = P * s2 + 1.0 / (double)(2 * k + 1);
    const double lnm = (2.0 * s) * P;
    return lnm + (double)(e - 33) * 0.6931471805599453;
}
static void orc_cos_sin_2pi(uint32_t w, double *c, double *s)
{
    const uint32_t q = w >> 30;
    double f = ((double)(w & 0x3FFFFFFFu) + 0.5) * (1.0 / 1073741824.0);
    const int swap = f > 0.5;
    if (swap) f = 1.0 - f;
    const double x = f * 1.5707963267948966;
    const double x2 = x * x;
    double ps = -1.0 / 1307674368000.0;                   /* -1/15! */
    ps = ps * x2 + 1.0 / 6227020800.0;                    /*  1/13! */
    ps = ps * x2 - 1.0 / 39916800.0;
    ps = ps * x2 + 1.0 / 362880.0;
    ps = ps * x2 - 1.0 / 5040.0;
    ps = ps * x2 + 1.0 / 120.0;
    ps = ps * x2 - 1.0 / 6.0;
    ps = ps * x2 + 1.0;
    const double sn = x * ps;
    double pc = 1.0 / 20922789888000.0;                   /*  1/16! */
    pc = pc * x2 - 1.0 / 87178291200.0;                   /* -1/14! */
    pc = pc * x2 + 1.0 / 479001600.0;
    pc = pc * x2 - 1.0 / 3628800.0;
    pc = pc * x2 + 1.0 / 40320.0;
    pc = pc * x2 - 1.0 / 720.0;
    pc = pc * x2 + 1.0 / 24.0;
    pc = pc * x2 - 0.5;
    pc = pc * x2 + 1.0;
    const double c1 = swap ? sn : pc, s1 = swap ? pc : sn;   /* cos, sin of f pi/2 */
    switch (q) {
    case 0:  *c = c1;  *s = s1;  break;
    case 1:  *c = -s1; *s = c1;  break;
    case 2:  *c = -c1; *s = -s1; break;
    default: *c = s1;  *s = -c1; break;
    }
}
/* Box-Muller: two standard normals from two words. */
void orc_normal_pair(uint32_t w1, uint32_t w2, double z[2])
{
    const double R = sqrt(-2.0 * orc_ln_unit(w1));
    double c, s;
    orc_cos_sin_2pi(w2, &c, &s);
    z[0] = R * c;
    z[1] = R * s;
}
/* Variates of move m of sweep t of walker w under proposal 1: words A = Philox(m,t,w,2), B = Philox(m,t,w,3);
 * particle s = floor(A0 N / 2^32); (z0,z1) = BoxMuller(A1, A2), z2 = first of BoxMuller(B0, B1);
 * delta[k] = step * z_k (ONE rounding); xi from A3 as in proposal 0. */
void orc_move_variates_gauss(uint64_t seed, uint32_t w, uint32_t t, uint32_t m, int32_t N, double step,
                             int32_t *s, double delta[3], double *xi)
{
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t ca[4] = { m, t, w, 2u }, cb[4] = { m, t, w, 3u }, A[4], B[4];
    orc_philox4x32_10(ca, key, A);
    orc_philox4x32_10(cb, key, B);
    *s = (int32_t)(((uint64_t)A[0] * (uint64_t)(uint32_t)N) >> 32);
    double z01[2], z23[2];
    orc_normal_pair(A[1], A[2], z01);
    orc_normal_pair(B[0], B[1], z23);
    delta[0] = step * z01[0];
    delta[1] = step * z01[1];
    delta[2] = step * z23[0];
    *xi = unit_01(A[3]);
}

/* ---------------------------------------------------------------------------
 * Pair correlation factor.  Eq.(9) l.155: f(r) = -1/2 (b/r)^5.
 * Eq.(8) l.150 under reading R1: u(r) = f(r) + f(L-r) - 2 f(L/2) for r < L/2,
 * 0 beyond (strict '<', R2).
 * ------------------------------------------------------------------------- */
static double f_sv(double r, double b)   { double q = b / r; return -0.5 * q * q * q * q * q; }
static double df_sv(double r, double b)  { return -5.0 * f_sv(r, b) / r; }          /* f'  = +5/2 b^5 r^-6 */
static double d2f_sv(double r, double b) { return 30.0 * f_sv(r, b) / (r * r); }    /* f'' = -15 b^5 r^-7  */

double orc_u(double r, double L, double b)
{
    double h = 0.5 * L;
    if (!(r < h)) return 0.0;
    return f_sv(r, b) + f_sv(L - r, b) - 2.0 * f_sv(h, b);
}
double orc_du(double r, double L, double b)      /* u'(r)  = f'(r) - f'(L-r) */
{
    double h = 0.5 * L;
    if (!(r < h)) return 0.0;
    return df_sv(r, b) - df_sv(L - r, b);
}
double orc_d2u(double r, double L, double b)     /* u''(r) = f''(r) + f''(L-r) */
{
    double h = 0.5 * L;
    if (!(r < h)) return 0.0;
    return d2f_sv(r, b) + d2f_sv(L - r, b);
}

/* HFD-B(HE) pair potential (l.131; form and constants: R3), in K.
 * V(r) = eps [ A exp(-alpha x + beta x^2) - F(x) (c6/x^6 + c8/x^8 + c10/x^10) ],
 * x = r/rm, F(x) = exp(-(D/x - 1)^2) for x < D, 1 otherwise.  No cutoff here. */
double orc_aziz(double r, const double a[9])
{
    double eps = a[0], rm = a[1], A = a[2], alpha = a[3], beta = a[4];
    double c6 = a[5], c8 = a[6], c10 = a[7], D = a[8];
    double x = r / rm;
    double F = 1.0;
    if (x < D) { double t = D / x - 1.0; F = exp(-t * t); }
    double x2 = x * x, x6 = x2 * x2 * x2, x8 = x6 * x2, x10 = x8 * x2;
    return eps * (A * exp(-alpha * x + beta * x2) - F * (c6 / x6 + c8 / x8 + c10 / x10));
}

/* Minimum-image separation a - b in a cubic box (l.325; R5): per component
 * d -= L * rint(d / L). */
static void min_image(const double a[3], const double b[3], double L, double d[3])
{
    for (int k = 0; k < 3; ++k) {
        double t = a[k] - b[k];
        t -= L * rint(t / L);
        d[k] = t;
    }
}
static double dist(const double a[3], const double b[3], double L)
{
    double d[3];
    min_image(a, b, L, d);
    return sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
}

/* Coordinates are SoA: xyz[0..N) = x, xyz[N..2N) = y, xyz[2N..3N) = z. */
static void get_pos(const double *xyz, int N, int i, double p[3])
{
    p[0] = xyz[i]; p[1] = xyz[N + i]; p[2] = xyz[2 * N + i];
}

/* log psi(X) = sum_{i<j} u(r_ij), Eq.(6) l.136. */
double orc_log_psi(const orc_sys *sys, const double *xyz)
{
    int N = sys->N;
    double sum = 0.0;
    for (int i = 0; i < N; ++i)
        for (int j = i + 1; j < N; ++j) {
            double pi[3], pj[3];
            get_pos(xyz, N, i, pi); get_pos(xyz, N, j, pj);
            sum += orc_u(dist(pi, pj, sys->L), sys->L, sys->b);
        }
    return sum;
}

/* Per-particle pair sums S_i = sum_{j != i} u(r_ij)  (so sum_i S_i = 2 log psi). */
void orc_pair_sums(const orc_sys *sys, const double *xyz, double *S)
{
    int N = sys->N;
    for (int i = 0; i < N; ++i) {
        double pi[3], sum = 0.0;
        get_pos(xyz, N, i, pi);
        for (int j = 0; j < N; ++j) {
            if (j == i) continue;
            double pj[3];
            get_pos(xyz, N, j, pj);
            sum += orc_u(dist(pi, pj, sys->L), sys->L, sys->b);
        }
        S[i] = sum;
    }
}

/* Eq.(7) l.146: Delta = sum_{j != s} [ u(|r_s + delta - r_j|) - u(|r_s - r_j|) ],
 * two plain loops (R17: no running sums here). */
double orc_delta_log_psi(const orc_sys *sys, const double *xyz, int s, const double trial[3])
{
    int N = sys->N;
    double ps[3], sum_new = 0.0, sum_old = 0.0;
    get_pos(xyz, N, s, ps);
    for (int j = 0; j < N; ++j) {
        if (j == s) continue;                       /* R9: exclude by index */
        double pj[3];
        get_pos(xyz, N, j, pj);
        sum_new += orc_u(dist(trial, pj, sys->L), sys->L, sys->b);
    }
    for (int j = 0; j < N; ++j) {
        if (j == s) continue;
        double pj[3];
        get_pos(xyz, N, j, pj);
        sum_old += orc_u(dist(ps, pj, sys->L), sys->L, sys->b);
    }
    return sum_new - sum_old;
}

/* One conditional add/sub keeps stored coordinates in [0,L] (R10). */
static double wrap(double x, double L)
{
    if (x >= L) x -= L;
    if (x < 0.0) x += L;
    return x;
}

/* ---------------------------------------------------------------------------
 * Metropolis sweeps of one walker (Eq.(5) l.123, Eq.(7) l.146, l.325-331; R7, R8).
 * For sweep t = t0 .. t0+n_sweeps-1, for s = 0 .. N-1 in order (proposal 1: N moves of the particle and
 * Gaussian displacement orc_move_variates_gauss draws; |z| <= sqrt(66 ln 2) = 6.77 with 32-bit uniforms, and
 * callers keep 6.77 step < L/2, so one wrap still brings a coordinate back into [0, L]):
 *   trial = r_s + delta;  accept iff 2*Delta > log(xi) (strict);
 *   on accept r_s <- wrap(trial).
 * Optional per-move outputs (index m = (t-t0)*N + s):
 *   dec_out[m]    1 if accepted (as decided here, or as forced)
 *   margin_out[m] 2*Delta - log(xi)   (the quantity whose sign decides)
 * dec_force (optional): decisions to ADOPT instead of the oracle's own (used to
 * resynchronise after an exempt near-tie, R19); margin_out still reports the
 * oracle's own margin for that move.
 * Returns the number of accepted moves.
 * ------------------------------------------------------------------------- */
int64_t orc_sweep(const orc_sys *sys, double *xyz, uint64_t seed, uint32_t w, uint32_t t0,
                  int32_t n_sweeps, double step,
                  uint8_t *dec_out, double *margin_out, const uint8_t *dec_force)
{
    int N = sys->N;
    int64_t n_acc = 0, m = 0;
    for (int32_t it = 0; it < n_sweeps; ++it) {
        uint32_t t = t0 + (uint32_t)it;
        for (int sq = 0; sq < N; ++sq, ++m) {
            double delta[3], xi, ps[3], trial[3];
            int32_t s = sq;
            if (sys->proposal == 1) orc_move_variates_gauss(seed, w, t, (uint32_t)sq, N, step, &s, delta, &xi);
            else                    orc_move_variates(seed, w, t, (uint32_t)sq, step, delta, &xi);
            get_pos(xyz, N, s, ps);
            for (int k = 0; k < 3; ++k) trial[k] = ps[k] + delta[k];
            double Delta = orc_delta_log_psi(sys, xyz, s, trial);
            double margin = 2.0 * Delta - log(xi);
            int accept = margin > 0.0;
            if (dec_force) accept = dec_force[m] != 0;
            if (accept) {
                for (int k = 0; k < 3; ++k) xyz[k * N + s] = wrap(trial[k], sys->L);
                ++n_acc;
            }
            if (dec_out) dec_out[m] = (uint8_t)accept;
            if (margin_out) margin_out[m] = margin;
        }
    }
    return n_acc;
}

/* ---------------------------------------------------------------------------
 * Local energy of one configuration (l.113-115 local value; l.129 Hamiltonian;
 * l.153/l.381 two kinetic estimators, R14).  With log psi = sum_{i<j} u(r_ij):
 *   G_i      = grad_i log psi = sum_{j != i} u'(r_ij) d_ij / r_ij
 *   Lambda_i = lap_i  log psi = sum_{j != i} [ u''(r_ij) + 2 u'(r_ij) / r_ij ]
 *   T_PB = -Dk sum_i (Lambda_i + |G_i|^2)      ( = -Dk sum_i lap_i psi / psi )
 *   T_JF = -(Dk/2) sum_i Lambda_i
 *   V    = sum_{i<j, r<L/2} V_Aziz(r_ij)        (truncated, no shift, no tail: R3)
 * out[0..5] = E_PB = V + T_PB, V, T_PB, T_JF, T_CW = Dk sum |G_i|^2, min |r^2/h^2 - 1|.
 * ------------------------------------------------------------------------- */
void orc_local_energy(const orc_sys *sys, const double *xyz, double out[6])
{
    int N = sys->N;
    double L = sys->L, b = sys->b, h = 0.5 * L;
    double V = 0.0, sumLam = 0.0, sumG2 = 0.0, guard = INFINITY;
    for (int i = 0; i < N; ++i) {
        double pi[3], G[3] = { 0.0, 0.0, 0.0 }, Lam = 0.0;
        get_pos(xyz, N, i, pi);
        for (int j = 0; j < N; ++j) {
            if (j == i) continue;
            double pj[3], d[3];
            get_pos(xyz, N, j, pj);
            min_image(pi, pj, L, d);
            double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            double r = sqrt(r2);
            double g = fabs(r2 / (h * h) - 1.0);
            if (g < guard) guard = g;
            if (!(r < h)) continue;
            double du = orc_du(r, L, b), d2u = orc_d2u(r, L, b);
            for (int k = 0; k < 3; ++k) G[k] += du * d[k] / r;
            Lam += d2u + 2.0 * du / r;
            if (j > i) V += orc_aziz(r, sys->aziz);
        }
        sumLam += Lam;
        sumG2 += G[0] * G[0] + G[1] * G[1] + G[2] * G[2];
    }
    double T_PB = -sys->Dk * (sumLam + sumG2);
    double T_JF = -0.5 * sys->Dk * sumLam;
    out[0] = V + T_PB; out[1] = V; out[2] = T_PB; out[3] = T_JF;
    out[4] = sys->Dk * sumG2; out[5] = guard;
}

/* grad_i log psi and lap_i log psi for every particle (pinned against finite
 * differences of orc_log_psi in the tests). G is [3][N], Lam is [N]. */
void orc_grad_lap(const orc_sys *sys, const double *xyz, double *G, double *Lam)
{
    int N = sys->N;
    double L = sys->L, b = sys->b, h = 0.5 * L;
    for (int i = 0; i < N; ++i) {
        double pi[3], g[3] = { 0.0, 0.0, 0.0 }, lam = 0.0;
        get_pos(xyz, N, i, pi);
        for (int j = 0; j < N; ++j) {
            if (j == i) continue;
            double pj[3], d[3];
            get_pos(xyz, N, j, pj);
            min_image(pi, pj, L, d);
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            if (!(r < h)) continue;
            double du = orc_du(r, L, b), d2u = orc_d2u(r, L, b);
            for (int k = 0; k < 3; ++k) g[k] += du * d[k] / r;
            lam += d2u + 2.0 * du / r;
        }
        G[i] = g[0]; G[N + i] = g[1]; G[2 * N + i] = g[2];
        Lam[i] = lam;
    }
}

/* ---------------------------------------------------------------------------
 * Initial walker (R13): FCC lattice with k = smallest integer with 4 k^3 >= N,
 * a = L/k, sites ordered (ix, iy, iz, basis) basis fastest, basis offsets
 * {000, 1/2 1/2 0, 1/2 0 1/2, 0 1/2 1/2}; particle i takes site floor(i*M/N),
 * M = 4 k^3; coordinate c is ((i_c + o_c) * a) + JIT * a_c with a_c in (-1,1)
 * from Philox counter (i, 0, w, 1); then wrap.
 * ------------------------------------------------------------------------- */
void orc_init_walker(const orc_sys *sys, uint64_t seed, uint32_t w, double jitter, double *xyz)
{
    int N = sys->N;
    int64_t k = 1;
    while (4 * k * k * k < N) ++k;
    int64_t M = 4 * k * k * k;
    double a = sys->L / (double)k;
    static const double off[4][3] = { {0,0,0}, {0.5,0.5,0}, {0.5,0,0.5}, {0,0.5,0.5} };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    for (int i = 0; i < N; ++i) {
        int64_t site = ((int64_t)i * M) / N;
        int bas = (int)(site % 4);
        int64_t cell = site / 4;
        int64_t iz = cell % k, iy = (cell / k) % k, ix = cell / (k * k);
        double idx[3] = { (double)ix, (double)iy, (double)iz };
        uint32_t ctr[4] = { (uint32_t)i, 0u, w, 1u }, x[4];
        orc_philox4x32_10(ctr, key, x);
        for (int c = 0; c < 3; ++c) {
            double lattice = (idx[c] + off[bas][c]) * a;
            double jit = jitter * unit_pm1(x[c]);
            xyz[c * N + i] = wrap(lattice + jit, sys->L);
        }
    }
}

/* ---------------------------------------------------------------------------
 * Trivial many-walker wrappers (one OS thread per walker through OpenMP when
 * compiled with -fopenmp; walkers are independent chains, l.169).  Walker v of
 * the batch has global id w0 + v and state xyz + v*3*N.
 * ------------------------------------------------------------------------- */
void orc_init_walkers(const orc_sys *sys, uint64_t seed, uint32_t w0, int32_t W, double jitter, double *xyz)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int v = 0; v < W; ++v)
        orc_init_walker(sys, seed, w0 + (uint32_t)v, jitter, xyz + (size_t)v * 3 * sys->N);
}

void orc_sweep_walkers(const orc_sys *sys, double *xyz, uint64_t seed, uint32_t w0, int32_t W,
                       uint32_t t0, int32_t n_sweeps, double step,
                       uint8_t *dec_out, double *margin_out, const uint8_t *dec_force, int64_t *n_acc)
{
    size_t moves = (size_t)n_sweeps * sys->N;
#pragma omp parallel for schedule(dynamic, 1)
    for (int v = 0; v < W; ++v) {
        int64_t a = orc_sweep(sys, xyz + (size_t)v * 3 * sys->N, seed, w0 + (uint32_t)v, t0, n_sweeps, step,
                              dec_out ? dec_out + v * moves : NULL,
                              margin_out ? margin_out + v * moves : NULL,
                              dec_force ? dec_force + v * moves : NULL);
        if (n_acc) n_acc[v] = a;
    }
}

void orc_local_energy_walkers(const orc_sys *sys, const double *xyz, int32_t W, double *out /*[W][6]*/)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int v = 0; v < W; ++v)
        orc_local_energy(sys, xyz + (size_t)v * 3 * sys->N, out + (size_t)v * 6);
}

int32_t orc_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    n = omp_get_max_threads();
#endif
    return n;
}

/* ---------------------------------------------------------------------------
 * Pair distribution function (the paper's second observable, l.421, l.468): histogram of the
 * minimum-image pair distances of ONE configuration.  Bins of width h / nbins on [0, h), h = L/2
 * (the cutoff of l.460).  For every pair i < j with r < h: k = (int)(r * inv_dr), inv_dr = nbins / h;
 * k = nbins (r within rounding of h) is counted in the last bin.  DESIGN.md "Observables".
 * ------------------------------------------------------------------------- */
void orc_pair_histogram(const orc_sys *sys, const double *xyz, int nbins, uint32_t *hist)
{
    const int N = sys->N;
    const double h = 0.5 * sys->L;
    const double inv_dr = (double)nbins / h;
    for (int k = 0; k < nbins; ++k) hist[k] = 0u;
    for (int i = 0; i < N; ++i) {
        double pi[3];
        get_pos(xyz, N, i, pi);
        for (int j = i + 1; j < N; ++j) {
            double pj[3];
            get_pos(xyz, N, j, pj);
            const double r = dist(pi, pj, sys->L);
            if (r < h) {
                int k = (int)(r * inv_dr);
                if (k >= nbins) k = nbins - 1;
                hist[k] += 1u;
            }
        }
    }
}
