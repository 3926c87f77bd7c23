/*
 * oracle/cos_oracle.c -- plain, slow, obviously-correct CPU oracle for the CoS hot path of
 * arxiv/paper_2501_00675 (Sturt & Kozik, "Exploiting Parallelism for Fast Feynman Diagrammatics").
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, link or call this file.  It shares no code, header, table or
 * helper with paper_2501_00675_b200/ (the CUDA path) and neither includes the other.
 *
 * Contents (each function cites the passage it follows; P:<line> = /root/reference/PAPER.md):
 *   oracle_build_G          G assembly from a tabulated G0(x,tau)      (BASELINE.json configs; R8, R9, R7)
 *   oracle_eval / _f80      propagation -> combine -> connected reduction (R1, R5, R6, R10)
 *   oracle_minors           Z[S] of one species for every subset S     (pinned against LU minors in tests)
 *   oracle_bruteforce       the plain definition: every pair of permutations, connectivity tested
 *                           explicitly ("all O(n!) terms", R3)      -- pins oracle_eval for n <= 7
 *   oracle_abs_sum          conditioning number numerator (R5)
 *
 * Pins (tests/test_oracle_*.py, all run without a GPU): brute force n<=5 (and a pure-Python
 * enumerator written separately), connected-pair counts 1,3,26,426,11064, all = prod(-u) det Gup det Gdn
 * via numpy.linalg, Z[S] = (-1)^|S| det W[S,S] via numpy.linalg for every S, closed forms at n=1,2,
 * rank-1 and identity special cases, block-diagonal => 0, relabelling/transpose/diagonal-similarity
 * invariances, exp/log consistency over set partitions.  No function here is "parity unpinned".
 *
 * Build:  gcc -O2 -std=c11 -ffp-contract=off -fopenmp -shared -fPIC cos_oracle.c -o liboracle.so -lm
 * (-ffp-contract=off: every product and sum below is rounded separately except the one fma() that
 *  reading R8 writes explicitly.)
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define REAL double
#define FN(name) name##_f64
#include "cos_oracle_core.inc"
#undef REAL
#undef FN

#define REAL long double
#define FN(name) name##_f80
#include "cos_oracle_core.inc"
#undef REAL
#undef FN

/* ------------------------------------------------------------------------------------------
 * G assembly (§8(a) a1; BASELINE.json configs: "G0(x,tau) is tabulated ... with 512 tau-points and
 * linear interpolation; spin-up and spin-down G are n x n FP64").  Readings R7, R8, R9:
 *   G_s[b][i][j] = G0_s( (x_i - x_j) mod L , tau_i - tau_j )
 *   table T_s[dx][dy][k] holds G0_s at tau_k = k*beta/(ntau-1), k = 0..ntau-1 (0+ and beta- ends)
 *   dtau > 0 :  lerp(T, dtau);   dtau <= 0 (i != j): -lerp(T, dtau + beta)   (antiperiodicity)
 *   lerp: u = dtau*(ntau-1)/beta, k = min(floor(u), ntau-2), value = fma(u-k, T[k+1]-T[k], T[k])
 *   i == j: g_diag (equal-time diagonal, R7)
 * xy: [batch][n][2] int32 lattice sites; tau: [batch][n]; Gup,Gdn: [batch][n][n] row-major.
 * Tup and Tdn may be the same table; Gdn may be NULL (then only Gup is written).
 */
static double lerp_table(const double *T, int ntau, double beta, double dtau)
{
    const double u = dtau * (double)(ntau - 1) / beta;
    int k = (int)floor(u);
    if (k > ntau - 2) k = ntau - 2;
    if (k < 0) k = 0;
    return fma(u - (double)k, T[k + 1] - T[k], T[k]);
}

void oracle_build_G(int n, long long batch, const int *xy, const double *tau,
                    const double *Tup, const double *Tdn, int Lx, int Ly, int ntau, double beta,
                    double g_diag, double *Gup, double *Gdn)
{
    for (long long b = 0; b < batch; ++b)
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < n; ++j) {
                const size_t o = ((size_t)b * n + i) * n + j;
                if (i == j) {
                    Gup[o] = g_diag;
                    if (Gdn) Gdn[o] = g_diag;
                    continue;
                }
                const int *pi = xy + ((size_t)b * n + i) * 2, *pj = xy + ((size_t)b * n + j) * 2;
                int dx = (pi[0] - pj[0]) % Lx; if (dx < 0) dx += Lx;
                int dy = (pi[1] - pj[1]) % Ly; if (dy < 0) dy += Ly;
                double dtau = tau[(size_t)b * n + i] - tau[(size_t)b * n + j];
                double sign = 1.0;
                if (dtau <= 0.0) { dtau += beta; sign = -1.0; }      /* R9: dtau == 0 is 0- */
                const size_t row = ((size_t)dx * Ly + dy) * (size_t)ntau;
                Gup[o] = sign * lerp_table(Tup + row, ntau, beta, dtau);
                if (Gdn) Gdn[o] = sign * lerp_table(Tdn + row, ntau, beta, dtau);
            }
}

/* ------------------------------------------------------------------------------------------
 * Batch evaluation.  Gup,Gdn: [batch][n][n] (may alias); u: NULL or [batch][n]; U used when u NULL.
 * out_all, out_connected: [batch] (either may be NULL).  threads <= 0: all OpenMP threads.
 * Returns the number of threads used.
 */
int oracle_eval_lw(int n, long long batch, const double *Gup, const double *Gdn, const double *u, double U,
                   double loop_weight, double *out_all, double *out_connected, int threads)
{
    int used = 1;
#ifdef _OPENMP
    if (threads <= 0) threads = omp_get_max_threads();
    used = threads;
#pragma omp parallel num_threads(threads)
#endif
    {
        double *work = (double *)malloc(sizeof(double) * work_reals_f64(n));
        double ubuf[32];
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (long long b = 0; b < batch; ++b) {
            for (int a = 0; a < n; ++a) ubuf[a] = u ? u[(size_t)b * n + a] : U;
            double all, conn;
            eval_one_f64(n, Gup + (size_t)b * n * n, Gdn + (size_t)b * n * n, ubuf, -loop_weight, work, &all, &conn);
            if (out_all) out_all[b] = all;
            if (out_connected) out_connected[b] = conn;
        }
        free(work);
    }
    return used;
}

/* The paper's own weight: -1 per closed fermion loop, i.e. loop_weight = 1. */
int oracle_eval(int n, long long batch, const double *Gup, const double *Gdn,
                const double *u, double U, double *out_all, double *out_connected, int threads)
{
    return oracle_eval_lw(n, batch, Gup, Gdn, u, U, 1.0, out_all, out_connected, threads);
}

/* Same, every accumulator in long double; results rounded to double on output ("truth" mode). */
int oracle_eval_lw_f80(int n, long long batch, const double *Gup, const double *Gdn, const double *u, double U,
                       double loop_weight, double *out_all, double *out_connected, int threads)
{
    int used = 1;
#ifdef _OPENMP
    if (threads <= 0) threads = omp_get_max_threads();
    used = threads;
#pragma omp parallel num_threads(threads)
#endif
    {
        long double *work = (long double *)malloc(sizeof(long double) * work_reals_f80(n));
        double ubuf[32];
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (long long b = 0; b < batch; ++b) {
            for (int a = 0; a < n; ++a) ubuf[a] = u ? u[(size_t)b * n + a] : U;
            long double all, conn;
            eval_one_f80(n, Gup + (size_t)b * n * n, Gdn + (size_t)b * n * n, ubuf, -loop_weight, work, &all, &conn);
            if (out_all) out_all[b] = (double)all;
            if (out_connected) out_connected[b] = (double)conn;
        }
        free(work);
    }
    return used;
}

int oracle_eval_f80(int n, long long batch, const double *Gup, const double *Gdn,
                    const double *u, double U, double *out_all, double *out_connected, int threads)
{
    return oracle_eval_lw_f80(n, batch, Gup, Gdn, u, U, 1.0, out_all, out_connected, threads);
}

/* Z[S] for every subset S of one n x n matrix W (step 1 alone) with loop factor -loop_weight.  Z: [2^n]. */
void oracle_minors_lw(int n, const double *W, double loop_weight, double *Z)
{
    double *A = (double *)malloc(sizeof(double) * ((size_t)n << n));
    propagate_f64(n, W, -loop_weight, Z, A);
    free(A);
}

void oracle_minors(int n, const double *W, double *Z) { oracle_minors_lw(n, W, 1.0, Z); }

/* Half-vertex formulation (cos_oracle_core.inc: eval_one_halfvertex).  W: [batch][2n'][2n'], V: [batch][n']. */
int oracle_eval_halfvertex(int np, long long batch, const double *W, const double *V, double loop_weight,
                           double *out_all, double *out_connected, int threads)
{
    const int m = 2 * np;
    int used = 1;
#ifdef _OPENMP
    if (threads <= 0) threads = omp_get_max_threads();
    used = threads;
#pragma omp parallel num_threads(threads)
#endif
    {
        double *work = (double *)malloc(sizeof(double) * work_reals_f64(m));
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (long long b = 0; b < batch; ++b) {
            double all, conn;
            eval_one_halfvertex_f64(np, W + (size_t)b * m * m, V + (size_t)b * np, -loop_weight, work, &all, &conn);
            if (out_all) out_all[b] = all;
            if (out_connected) out_connected[b] = conn;
        }
        free(work);
    }
    return used;
}

/* D[S] and C[S] for every subset of one configuration (steps 1-3), for the exp/log pin. */
void oracle_DC(int n, const double *Gup, const double *Gdn, const double *u, double *D, double *C)
{
    const size_t N = (size_t)1 << n;
    double *A = (double *)malloc(sizeof(double) * (N * n + 2 * N));
    double *Zup = A + N * n, *Zdn = Zup + N;
    propagate_f64(n, Gup, -1.0, Zup, A);
    propagate_f64(n, Gdn, -1.0, Zdn, A);
    combine_f64(n, Zup, Zdn, u, D);
    reduce_connected_f64(n, D, C);
    free(A);
}

/* |.|-sum of every term with all signs dropped, one configuration (R5 conditioning numerator). */
double oracle_abs_sum(int n, const double *Gup, const double *Gdn, const double *u, double *abs_all)
{
    long double *work = (long double *)malloc(sizeof(long double) * work_reals_f80(n));
    long double aa = 0;
    const long double r = abs_sum_one_f80(n, Gup, Gdn, u, work, &aa);
    if (abs_all) *abs_all = (double)aa;
    free(work);
    return (double)r;
}

/* Batch form: abs_conn[b], abs_all[b] for every configuration (u NULL -> U).  Error-bound scales:
 * |fl(connected) - connected| <~ c * eps * abs_conn, |fl(all) - all| <~ c * eps * abs_all. */
void oracle_abs_sums(int n, long long batch, const double *Gup, const double *Gdn, const double *u,
                     double U, double *abs_conn, double *abs_all, int threads)
{
#ifdef _OPENMP
    if (threads <= 0) threads = omp_get_max_threads();
#pragma omp parallel for num_threads(threads) schedule(static)
#endif
    for (long long b = 0; b < batch; ++b) {
        double ubuf[32];
        for (int a = 0; a < n; ++a) ubuf[a] = u ? u[(size_t)b * n + a] : U;
        abs_conn[b] = oracle_abs_sum(n, Gup + (size_t)b * n * n, Gdn + (size_t)b * n * n, ubuf, abs_all + b);
    }
}

/* ------------------------------------------------------------------------------------------
 * The plain definition, one configuration, n <= 8 (SURVEY §8(c) "Plain definition"):
 *   all       = prod_a(-u_a) * sum_{sigma_up, sigma_dn in S_n} (-1)^{cyc(sigma_up)+cyc(sigma_dn)}
 *                              prod_i Gup[i][sigma_up(i)] * Gdn[i][sigma_dn(i)]
 *   connected = the same sum restricted to pairs for which the graph on {0..n-1} with edges
 *               {i, sigma_up(i)} and {i, sigma_dn(i)} is connected
 *   ("all O(n!) terms"; "-1 ... closing a fermion loop"; R3: (n!)^2 pairs for two species)
 * n_connected returns the number of connected pairs (must be 1, 3, 26, 426, 11064 for n = 1..5).
 * Returns 0, or -1 if n is out of range.
 */
static int next_permutation_int(int *p, int n)
{
    int i = n - 2;
    while (i >= 0 && p[i] > p[i + 1]) --i;
    if (i < 0) return 0;
    int j = n - 1;
    while (p[j] < p[i]) --j;
    int t = p[i]; p[i] = p[j]; p[j] = t;
    for (int a = i + 1, b = n - 1; a < b; ++a, --b) { t = p[a]; p[a] = p[b]; p[b] = t; }
    return 1;
}

static int uf_find(int *parent, int x)
{
    while (parent[x] != x) x = parent[x];
    return x;
}

int oracle_bruteforce_lw(int n, const double *Gup, const double *Gdn, const double *u, double loop_weight,
                         double *out_all, double *out_connected, long long *n_connected)
{
    if (n < 1 || n > 8) return -1;
    int fact = 1;
    for (int i = 2; i <= n; ++i) fact *= i;
    int *perm = (int *)malloc(sizeof(int) * (size_t)fact * n);
    double *tu = (double *)malloc(sizeof(double) * (size_t)fact * 2), *td = tu + fact;

    int p[8];
    for (int i = 0; i < n; ++i) p[i] = i;
    int idx = 0;
    do {                                              /* every permutation, its cycle count, its product */
        memcpy(perm + (size_t)idx * n, p, sizeof(int) * n);
        int seen[8] = {0}, cyc = 0;
        for (int i = 0; i < n; ++i) {
            if (seen[i]) continue;
            ++cyc;
            for (int j = i; !seen[j]; j = p[j]) seen[j] = 1;
        }
        double pu = 1.0, pd = 1.0;
        for (int i = 0; i < n; ++i) { pu *= Gup[i * n + p[i]]; pd *= Gdn[i * n + p[i]]; }
        double sg = 1.0;                               /* (-loop_weight)^{number of closed fermion loops}; */
        for (int c = 0; c < cyc; ++c) sg *= -loop_weight;   /* loop_weight = 1: the paper's -1 per loop */
        tu[idx] = sg * pu;
        td[idx] = sg * pd;
        ++idx;
    } while (next_permutation_int(p, n));

    double w = 1.0;
    for (int a = 0; a < n; ++a) w *= -u[a];

    long double sum_all = 0, sum_conn = 0;
    long long cnt = 0;
    for (int a = 0; a < fact; ++a)
        for (int b = 0; b < fact; ++b) {
            const double term = tu[a] * td[b];
            sum_all += term;
            int parent[8];
            for (int i = 0; i < n; ++i) parent[i] = i;
            const int *pa = perm + (size_t)a * n, *pb = perm + (size_t)b * n;
            int comps = n;
            for (int i = 0; i < n; ++i) {
                int r0 = uf_find(parent, i), r1 = uf_find(parent, pa[i]);
                if (r0 != r1) { parent[r0] = r1; --comps; }
                r0 = uf_find(parent, i); r1 = uf_find(parent, pb[i]);
                if (r0 != r1) { parent[r0] = r1; --comps; }
            }
            if (comps == 1) { sum_conn += term; ++cnt; }
        }
    if (out_all) *out_all = (double)((long double)w * sum_all);
    if (out_connected) *out_connected = (double)((long double)w * sum_conn);
    if (n_connected) *n_connected = cnt;
    free(perm);
    free(tu);
    return 0;
}

int oracle_bruteforce(int n, const double *Gup, const double *Gdn, const double *u,
                      double *out_all, double *out_connected, long long *n_connected)
{
    return oracle_bruteforce_lw(n, Gup, Gdn, u, 1.0, out_all, out_connected, n_connected);
}

/* Plain definition of the half-vertex formulation (cos_oracle_core.inc: eval_one_halfvertex): every permutation
 * of the m = 2n' half-vertices, (-loop_weight)^cycles, connectivity of the interaction-line graph tested with
 * union-find.  n' <= 4 (8! = 40320 permutations).  n_connected: number of connected permutations. */
int oracle_bruteforce_halfvertex(int np, const double *W, const double *V, double loop_weight,
                                 double *out_all, double *out_connected, long long *n_connected)
{
    if (np < 1 || np > 4) return -1;
    const int m = 2 * np;
    int p[8];
    for (int i = 0; i < m; ++i) p[i] = i;
    long double sum_all = 0, sum_conn = 0;
    long long cnt = 0;
    do {
        int seen[8] = {0}, cyc = 0;
        for (int i = 0; i < m; ++i) {
            if (seen[i]) continue;
            ++cyc;
            for (int j = i; !seen[j]; j = p[j]) seen[j] = 1;
        }
        double term = 1.0;
        for (int c = 0; c < cyc; ++c) term *= -loop_weight;
        for (int i = 0; i < m; ++i) term *= W[i * m + p[i]];
        sum_all += term;
        int parent[4], comps = np;
        for (int k = 0; k < np; ++k) parent[k] = k;
        for (int i = 0; i < m; ++i) {
            const int r0 = uf_find(parent, i / 2), r1 = uf_find(parent, p[i] / 2);
            if (r0 != r1) { parent[r0] = r1; --comps; }
        }
        if (comps == 1) { sum_conn += term; ++cnt; }
    } while (next_permutation_int(p, m));
    long double w = 1;
    for (int k = 0; k < np; ++k) w *= -(long double)V[k];
    if (out_all) *out_all = (double)(w * sum_all);
    if (out_connected) *out_connected = (double)(w * sum_conn);
    if (n_connected) *n_connected = cnt;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Monte Carlo over the vertex coordinates (reading R19).
 * P:47 "The integration over the vertex coordinates can then be performed by stochastic (Monte Carlo) sampling";
 * P:137 "one needs to handle proposal and acceptance of configurations ... readily implemented in device-sided
 * code".  The paper gives no update scheme; reading R19 fixes the plainest one: independent Metropolis walkers
 * ("many Markov chain walkers"), configuration weight |connected(x)|, one update per step:
 *   draw (r0, r1, r2, r3) = philox4x32_10(counter = (step, 0, walker_lo, walker_hi), key = (seed_lo, seed_hi))
 *   and  (s0, s1, s2, s3) = philox4x32_10(counter = (step, 1, walker_lo, walker_hi), same key);
 *   vertex k = r0 mod n moves to site (r1 mod Lx, r2 mod Ly) and time beta * u53(s0, s1);
 *   accept iff u53(s2, s3) * |w_old| < |w_new|   (symmetric proposal: min(1, |w_new| / |w_old|));
 *   u53(a, b) = (((uint64)a << 21) ^ ((uint64)b >> 11)) * 2^-53 in [0, 1).
 * philox4x32_10 is the counter-based generator of Salmon et al. (SC'11), restated here from its definition.
 */
typedef unsigned int u32;
typedef unsigned long long u64;

void oracle_philox4x32_10(const u32 ctr[4], const u32 key[2], u32 out[4])
{
    u32 c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        const u64 p0 = (u64)0xD2511F53u * c0, p1 = (u64)0xCD9E8D57u * c2;
        const u32 n0 = (u32)(p1 >> 32) ^ c1 ^ k0, n1 = (u32)p1;
        const u32 n2 = (u32)(p0 >> 32) ^ c3 ^ k1, n3 = (u32)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;          /* Weyl key schedule */
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

double oracle_u53(u32 a, u32 b)
{
    const u64 x = ((u64)a << 21) ^ ((u64)b >> 11);
    return (double)x * (1.0 / 9007199254740992.0);
}

/* xy [walkers][n][2], tau [walkers][n]: state, in/out.  weight [walkers]: connected value of the current
 * configuration (out).  accept_hist: NULL or [steps][walkers] (1 = accepted).  margin: NULL or [steps][walkers],
 * (|w_new| - r |w_old|) / max(|w_new|, |w_old|): a decision with |margin| below the parity tolerance is a tie that
 * another FP64 evaluation order may take the other way.  accepted [walkers], sign_sum [walkers] (sum over the
 * steps of sign(w) of the configuration held AFTER the step): out.  One table for both species (G_up = G_dn). */
void oracle_mc_run(int n, long long walkers, int steps, u64 seed, int *xy, double *tau,
                   const double *table, int Lx, int Ly, int ntau, double beta, double g_diag, double U,
                   double loop_weight, double *weight, unsigned char *accept_hist, double *margin,
                   long long *accepted, double *sign_sum, int threads)
{
#ifdef _OPENMP
    if (threads <= 0) threads = omp_get_max_threads();
#pragma omp parallel for num_threads(threads) schedule(static)
#endif
    for (long long w = 0; w < walkers; ++w) {
        double *work = (double *)malloc(sizeof(double) * (work_reals_f64(n) + 2 * (size_t)n * n));
        double *G = work + work_reals_f64(n);
        int pxy[2 * 32];
        double ptau[32], ubuf[32];
        for (int a = 0; a < n; ++a) ubuf[a] = U;
        int *sx = xy + (size_t)w * n * 2;
        double *st = tau + (size_t)w * n;
        double all, wold;
        oracle_build_G(n, 1, sx, st, table, table, Lx, Ly, ntau, beta, g_diag, G, NULL);
        eval_one_f64(n, G, G, ubuf, -loop_weight, work, &all, &wold);
        long long acc = 0;
        double ss = 0.0;
        const u32 key[2] = {(u32)seed, (u32)(seed >> 32)};
        for (int step = 0; step < steps; ++step) {
            u32 r[4], s[4];
            const u32 c0[4] = {(u32)step, 0u, (u32)w, (u32)((u64)w >> 32)};
            const u32 c1[4] = {(u32)step, 1u, (u32)w, (u32)((u64)w >> 32)};
            oracle_philox4x32_10(c0, key, r);
            oracle_philox4x32_10(c1, key, s);
            memcpy(pxy, sx, sizeof(int) * 2 * n);
            memcpy(ptau, st, sizeof(double) * n);
            const int k = (int)(r[0] % (u32)n);
            pxy[2 * k] = (int)(r[1] % (u32)Lx);
            pxy[2 * k + 1] = (int)(r[2] % (u32)Ly);
            ptau[k] = beta * oracle_u53(s[0], s[1]);
            double wnew;
            oracle_build_G(n, 1, pxy, ptau, table, table, Lx, Ly, ntau, beta, g_diag, G, NULL);
            eval_one_f64(n, G, G, ubuf, -loop_weight, work, &all, &wnew);
            const double rr = oracle_u53(s[2], s[3]);
            const int ok = rr * fabs(wold) < fabs(wnew);
            if (margin) {
                const double big = fabs(wold) > fabs(wnew) ? fabs(wold) : fabs(wnew);
                margin[(size_t)step * walkers + w] = big > 0 ? (fabs(wnew) - rr * fabs(wold)) / big : 0.0;
            }
            if (ok) {
                memcpy(sx, pxy, sizeof(int) * 2 * n);
                memcpy(st, ptau, sizeof(double) * n);
                wold = wnew;
                ++acc;
            }
            if (accept_hist) accept_hist[(size_t)step * walkers + w] = (unsigned char)ok;
            ss += (wold > 0) - (wold < 0);
        }
        weight[w] = wold;
        if (accepted) accepted[w] = acc;
        if (sign_sum) sign_sum[w] = ss;
        free(work);
    }
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
