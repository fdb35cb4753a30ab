/*
 * hmc_oracle.c -- CPU ORACLE for the orbit step of the Henon Monte Carlo method
 * (arXiv 1206.5878, Pattabiraman et al.; cited below as PAPER.md:LINE).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow,
 * single-threaded restatement of what the hot path computes, written from the
 * paper, so that the CUDA library can be checked against it star by star.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.  It shares no code, header, table or
 * constant generator with paper_1206_5878_b200/csrc/.
 *
 * Build:  gcc -O2 -ffp-contract=off -fPIC -shared hmc_oracle.c -o libhmc_oracle.so -lm
 * (-ffp-contract=off: no fused multiply-add, every +,-,*,/,sqrt below is one
 *  correctly rounded IEEE-754 binary64 operation, evaluated in the order the
 *  parentheses state -- DESIGN.md "Readings" R2.)
 * The same source built with -fopenmp (libhmc_oracle_omp.so) runs the per-star loops of S3,
 * S4 and the energy correction on all host cores: every star is
 * independent of the others and the random numbers are counter-based, so the results are
 * bit-identical to the single-threaded build (tests check it); the sort and the running
 * sums stay serial.  Without -fopenmp the pragmas are ignored.
 *
 * Numbering.  The paper numbers the radius-sorted stars 1..N.
 * Arrays here are 0-based: array element a holds node j = a+1.  Sentinel nodes
 * (R4): node 0 at r = 0 and node N+1 at r = +inf with Phi_{N+1} = 0
 * (Eq. 2).  "Shell j" is the interval [r_j, r_{j+1}], j = 0..N.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"):
 *   philox      : Random123 known-answer vectors (tests/golden/philox4x32_10_kat.txt)
 *   sort        : numpy stable argsort / lexsort; adversarial keys
 *   potential   : O(N^2) shell-theorem brute force in exact rational arithmetic,
 *                 Eq. 2-5 recursion, hand cases, Plummer closed form (statistical)
 *   turning pts : linear-scan brute force, Q(root)=0 with Phi from brute force,
 *                 Kepler closed form, circular orbit
 *   sampling    : energy identity, KS vs Kepler time-weighted CDF, closed-form
 *                 acceptance rate, order independence
 *   diagnostics : exact rational pair sums for T and W, numpy searchsorted for the
 *                 Lagrange radii, two-star hand case, Plummer closed forms, scaling laws
 *   energy corr.: exact invariance of T + W over a corrected step (pair-sum symmetry
 *                 of the shell potential), identity when the potential does not change,
 *                 v_r/v_t preserved, ten-step drift against the uncorrected run
 * No function in this file is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* per-star status bits (same numeric values as include/hmc.h, restated) */
#define ST_UNBOUND    1u   /* E >= 0 (or not a number): no turning points, no draw   */
#define ST_RADIAL     2u   /* J^2 == 0: pericentre is r = 0, no draw                 */
#define ST_DEGENERATE 4u   /* closed-form root not defined (C >= 0 in outer shell)   */
#define ST_CIRCULAR   8u   /* r_max - r_min <= 0 or end slopes of wrong sign         */
#define ST_MAXTRIES   16u  /* rejection loop hit T_MAX                               */
#define ST_CLIPPED    32u  /* some trial had g > F (density clipped; informational)  */

#ifndef T_MAX              /* a test-only build with -DT_MAX=3u exercises the exhaustion branch of S4 */
#define T_MAX 4096u        /* DESIGN.md R7 */
#endif
#define C_F   1.2          /* DESIGN.md R7 */

/* ------------------------------------------------------------------------ */
/* Philox4x32-10 (Salmon et al. 2011, "Parallel random numbers: as easy as  */
/* 1, 2, 3").  Replaces the paper's per-thread Tausworthe streams           */
/* so that a star's draws depend only on           */
/* (seed, step, star id) -- DESIGN.md R9; the paper's own reproducibility   */
/* test needed the same stream->star mapping on both sides.  */
/* ------------------------------------------------------------------------ */
void hmc_ref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------------ */
/* S1.  Sort stars by radial distance (step 6).               */
/* The paper uses Quicksort and does not say how ties are ordered; the      */
/* reading (R1) is the unique order by the pair (r_i, i).         */
/* perm[k] = original index of the k-th smallest radius.                    */
/* ------------------------------------------------------------------------ */
typedef struct { double r; uint32_t i; } key_index;

static int cmp_key_index(const void *pa, const void *pb)
{
    const key_index *a = (const key_index *)pa, *b = (const key_index *)pb;
    if (a->r < b->r) return -1;
    if (a->r > b->r) return 1;
    if (a->i < b->i) return -1;
    if (a->i > b->i) return 1;
    return 0;
}

/* what this build is: T_MAX and whether the per-star loops are threaded */
uint32_t hmc_ref_t_max(void) { return T_MAX; }
int hmc_ref_openmp(void)
{
#ifdef _OPENMP
    return 1;
#else
    return 0;
#endif
}

int hmc_ref_sort_by_radius(uint64_t n, const double *r_in, double *r_sorted, uint32_t *perm,
                           int ncols, const double *const *cols_in, double *const *cols_out,
                           const uint32_t *id_in, uint32_t *id_out)
{
    if (n == 0) return 0;
    key_index *a = (key_index *)malloc(n * sizeof(key_index));
    if (!a) return -1;
    for (uint64_t i = 0; i < n; ++i) { a[i].r = r_in[i]; a[i].i = (uint32_t)i; }
    qsort(a, n, sizeof(key_index), cmp_key_index);   /* Quicksort */
    for (uint64_t k = 0; k < n; ++k) {
        perm[k] = a[k].i;
        r_sorted[k] = a[k].r;
    }
    for (int c = 0; c < ncols; ++c) {
#pragma omp parallel for schedule(static)
        for (uint64_t k = 0; k < n; ++k) cols_out[c][k] = cols_in[c][perm[k]];
    }
    if (id_in && id_out) {
#pragma omp parallel for schedule(static)
        for (uint64_t k = 0; k < n; ++k) id_out[k] = id_in[perm[k]];
    }
    free(a);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* S2.  Potential at the star positions (Eq. 1 at r = r_k): */
/*   Phi_k = -G ( M_k / r_k  +  S_k ),                                      */
/*   M_k = sum_{i<=k} m_i ,   S_k = sum_{i>k} m_i / r_i .                   */
/* Eq. 2-5 is the same quantity as a recursion; tests check both.           */
/* Precision (R1p): the paper says only "double precision"        */
/* (PAPER.md:326).  M_k and S_k are defined here as the EXACT sums of the   */
/* binary64 terms m_i and fl(m_i / r_i), rounded once to binary64; the      */
/* running sums are therefore carried in binary128 (113-bit significand,    */
/* error ~N*2^-113, far below half an ulp of binary64 except with           */
/* probability ~N*2^-33 per run).  Phi_k is then three binary64 operations. */
/* ------------------------------------------------------------------------ */
int hmc_ref_potential(uint64_t n, double G, const double *r, const double *m,
                      double *phi, double *m_cum)
{
    __float128 acc = 0;
    for (uint64_t a = 0; a < n; ++a) {            /* Eq. 3 taken prefix by prefix */
        acc += (__float128)m[a];
        m_cum[a] = (double)acc;
    }
    acc = 0;                                      /* S_N = 0 <=> Phi_{N+1} = 0, Eq. 2 */
    for (uint64_t a = n; a-- > 0;) {
        double S = (double)acc;
        phi[a] = -(G * (m_cum[a] / r[a] + S));    /* Eq. 1 at r = r_k */
        double t = m[a] / r[a];
        acc += (__float128)t;
    }
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Table access with sentinels, paper numbering j = 0..N+1.                 */
/* ------------------------------------------------------------------------ */
typedef struct {
    uint64_t n;
    double G;
    const double *r, *phi, *mc;   /* 0-based arrays of length n */
} table;

/* Sign test of Q(r_j) = 2E - 2Phi_j - J^2/r_j^2 (Eq. 12) at a
 * table node: returns 1 when Q_j < 0.  Written division-free by multiplying
 * with r_j^2 > 0 (R2): Q_j < 0  <=>  2 (E - Phi_j) r_j^2 < J^2.
 * Node 0 (r = 0): Q = -inf for J > 0.  Node N+1 (r = inf, Phi = 0): Q = 2E < 0
 * for a bound star.  Both sentinels therefore answer "negative". */
static int q_negative(const table *T, uint64_t j, double E, double J2)
{
    if (j == 0 || j == T->n + 1) return 1;
    double rj = T->r[j - 1];
    return 2.0 * ((E - T->phi[j - 1]) * (rj * rj)) < J2;
}

/* Coefficients of Q inside shell j, as a function of u = 1/r:
 *   Phi(u) = Phi_j - G M_j (u - u_j)  (Eq. 1 == Eq. 6 anchored at node j, R3)
 *   Q(u)   = 2 C + 2 B u - J^2 u^2,  B = G M_j,  C = (E - Phi_j) - B u_j.
 * Shell 0 (inside the innermost star): Phi == Phi_1, so B = 0, C = E - Phi_1. */
static void shell_coeff(const table *T, uint64_t j, double E, double *B, double *C)
{
    if (j == 0) {
        *B = 0.0;
        *C = E - T->phi[0];
    } else {
        double b = T->G * T->mc[j - 1];
        *B = b;
        *C = (E - T->phi[j - 1]) - b * (1.0 / T->r[j - 1]);
    }
}

/* ------------------------------------------------------------------------ */
/* S3.  Pericentre and apocentre.                        */
/* For star k (node k): E = Phi_k + (v_r^2 + v_t^2)/2  (Eq. 16,             */
/* PAPER.md:202), J = r_k v_t.  "We need to determine k such that           */
/* Q(r_k) < 0 < Q(r_k+1).  We use the bisection method":     */
/*   k_min = the node j in [0, k-1]  with Q_j < 0 <= Q_{j+1}  (pericentre)  */
/*   k_max = the node j in [k, N]    with Q_j >= 0 > Q_{j+1}  (apocentre)   */
/* The star's own node is taken as Q >= 0 without being evaluated           */
/* (Q(r_k) = v_r^2, R5).  Then "Phi, and thus Q, can be computed  */
/* analytically in that interval, and so can r_min and r_max"               */
/* (PAPER.md:124): the roots of the quadratic in u of shell_coeff().        */
/* Stars are selected as array index first + i*stride, i < count; outputs   */
/* are compact arrays of length count.                                      */
/* ------------------------------------------------------------------------ */
int hmc_ref_orbit_turning_points(uint64_t n, double G,
        const double *r, const double *v_r, const double *v_t,
        const double *phi, const double *m_cum,
        uint64_t first, uint64_t stride, uint64_t count,
        double *E_out, double *J_out, double *r_min_out, double *r_max_out,
        uint32_t *k_min_out, uint32_t *k_max_out, uint8_t *status_out)
{
    table T = { n, G, r, phi, m_cum };
#pragma omp parallel for schedule(dynamic, 4096)
    for (uint64_t i = 0; i < count; ++i) {
        uint64_t a = first + i * stride;        /* array index           */
        uint64_t k = a + 1;                     /* node number, 1..N     */
        double E = phi[a] + 0.5 * (v_r[a] * v_r[a] + v_t[a] * v_t[a]);   /* Eq. 16 */
        double J = r[a] * v_t[a];
        double J2 = J * J;
        E_out[i] = E; J_out[i] = J;
        unsigned st = 0;
        if (!(E < 0.0)) st |= ST_UNBOUND;
        if (J2 == 0.0) st |= ST_RADIAL;
        if (st) {
            r_min_out[i] = (st & ST_RADIAL) ? 0.0 : r[a];
            r_max_out[i] = (st & ST_UNBOUND) ? INFINITY : r[a];
            k_min_out[i] = (uint32_t)(k - 1); k_max_out[i] = (uint32_t)k;
            status_out[i] = (uint8_t)st;
            continue;
        }
        /* bisection for the pericentre bracket: Q_lo < 0, Q_hi >= 0 */
        uint64_t lo = 0, hi = k;
        while (hi - lo > 1) {
            uint64_t mid = lo + (hi - lo) / 2;
            if (q_negative(&T, mid, E, J2)) lo = mid; else hi = mid;
        }
        uint64_t kmin = lo;
        /* bisection for the apocentre bracket: Q_lo >= 0, Q_hi < 0 */
        lo = k; hi = n + 1;
        while (hi - lo > 1) {
            uint64_t mid = lo + (hi - lo) / 2;
            if (q_negative(&T, mid, E, J2)) hi = mid; else lo = mid;
        }
        uint64_t kmax = lo;

        double B, C, D;
        shell_coeff(&T, kmin, E, &B, &C);
        D = B * B + 2.0 * (J2 * C);
        if (D < 0.0) D = 0.0;
        double rmin = J2 / (B + sqrt(D));                 /* larger-u root  */
        shell_coeff(&T, kmax, E, &B, &C);
        D = B * B + 2.0 * (J2 * C);
        if (D < 0.0) D = 0.0;
        double rmax;
        if (C < 0.0) rmax = (B + sqrt(D)) / (-2.0 * C);   /* smaller-u root, via the product of roots */
        else { rmax = INFINITY; st |= ST_DEGENERATE; }
        r_min_out[i] = rmin; r_max_out[i] = rmax;
        k_min_out[i] = (uint32_t)kmin; k_max_out[i] = (uint32_t)kmax;
        status_out[i] = (uint8_t)st;
    }
    return 0;
}

/* "To get the potential Phi(r) at any other radius, one first finds k such
 * that r_k <= r <= r_{k+1}": j = #{ i : r_i <= x } by bisection,
 * restricted to the orbit's own bracket [k_min, k_max]. */
static uint64_t shell_of(const table *T, double x, uint64_t kmin, uint64_t kmax)
{
    uint64_t lo = kmin, hi = kmax + 1;   /* answer in [kmin, kmax]; invariant r_lo <= x < r_hi (by clamping) */
    while (hi - lo > 1) {
        uint64_t mid = lo + (hi - lo) / 2;          /* node mid, 1..N */
        if (T->r[mid - 1] <= x) lo = mid; else hi = mid;
    }
    return lo;
}

/* Eq. 6 in the anchored form of DESIGN.md R3. */
static double phi_in_shell(const table *T, uint64_t j, double x)
{
    if (j == 0) return T->phi[0];
    return T->phi[j - 1] - (T->G * T->mc[j - 1]) * (1.0 / x - 1.0 / T->r[j - 1]);
}

/* ------------------------------------------------------------------------ */
/* S4.  New radial position: von Neumann rejection with  */
/* density f(r) ~ 1/|v_r|, v_r = sqrt(Q(r)) (Eq. 13).  The paper's Eq. 14-15 */
/* draw r_0 uniformly and compare F X' with f(r_0); "a slightly modified    */
/* version of the method is used, since f(r) = 1/|v_r| becomes infinite at  */
/* both ends", details deferred to Joshi et al. (2000).      */
/* Reading DESIGN.md R7 (Henon's change of variable):                       */
/*   s = 2X - 1,  r_0 = (r_min+r_max)/2 + (Delta/4)(3s - s^3)               */
/*   g(s) = f(r_0) dr/ds = (3/4) Delta (1 - s^2) / sqrt(Q(r_0))  (bounded)  */
/*   F = C_F max( sqrt(3 Delta / Q'(r_min)), sqrt(-3 Delta / Q'(r_max)) )   */
/*   accept iff Q(r_0) > 0 and F X' < g.                                    */
/* Random numbers: trial t of star `id` at step `step` uses                 */
/* Philox4x32-10(counter = (id, 0, step, t), key = (seed_lo, seed_hi)):     */
/* X from words 0,1 and X' from words 2,3 (53 bits each); the sign of the   */
/* new v_r from bit 0 of word 3 (R8, R9).                         */
/* All per-star arrays are compact, length count.                           */
/* counters[0] += total trials (if counters != NULL).                       */
/* ------------------------------------------------------------------------ */
int hmc_ref_sample_new_radius(uint64_t n, double G, uint64_t seed, uint32_t step,
        const double *r, const double *phi, const double *m_cum,
        uint64_t count,
        const double *r_self, const double *v_r_self, const double *v_t_self,
        const double *E_in, const double *J_in, const double *r_min_in, const double *r_max_in,
        const uint32_t *k_min_in, const uint32_t *k_max_in, const uint32_t *id,
        const uint8_t *status_in,
        double *r_new, double *v_r_new, double *v_t_new, uint16_t *n_try, uint8_t *status_out,
        uint64_t *counters)
{
    table T = { n, G, r, phi, m_cum };
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    const double two_m53 = 1.0 / 9007199254740992.0;
    uint64_t total_trials = 0;
#pragma omp parallel for schedule(dynamic, 4096) reduction(+ : total_trials)
    for (uint64_t i = 0; i < count; ++i) {
        unsigned st = status_in[i];
        r_new[i] = r_self[i]; v_r_new[i] = v_r_self[i]; v_t_new[i] = v_t_self[i];
        if (n_try) n_try[i] = 0;
        if (st & (ST_UNBOUND | ST_RADIAL | ST_DEGENERATE)) { status_out[i] = (uint8_t)st; continue; }
        double E = E_in[i], J = J_in[i], J2 = J * J;
        double rmin = r_min_in[i], rmax = r_max_in[i];
        uint64_t kmin = k_min_in[i], kmax = k_max_in[i];
        double delta = rmax - rmin;
        if (!(delta > 0.0)) { status_out[i] = (uint8_t)(st | ST_CIRCULAR); continue; }
        /* end slopes Q'(r) = 2 J^2 / r^3 - 2 G M_j / r^2 inside the bracketing shells */
        double Bmin = (kmin == 0) ? 0.0 : G * m_cum[kmin - 1];
        double Bmax = (kmax == 0) ? 0.0 : G * m_cum[kmax - 1];
        double q1 = (2.0 * (J2 / rmin - Bmin)) / (rmin * rmin);
        double q2 = (2.0 * (J2 / rmax - Bmax)) / (rmax * rmax);
        if (!(q1 > 0.0) || !(q2 < 0.0)) { status_out[i] = (uint8_t)(st | ST_CIRCULAR); continue; }
        double F = C_F * fmax(sqrt((3.0 * delta) / q1), sqrt((3.0 * delta) / (-q2)));
        double mid = 0.5 * (rmin + rmax);
        double quarter = 0.25 * delta, three_q = 0.75 * delta;
        int accepted = 0, have_good = 0;
        double good_r = 0, good_Q = 0; uint32_t good_w3 = 0;
        uint32_t t;
        for (t = 0; t < T_MAX; ++t) {
            uint32_t ctr[4] = { id[i], 0u, step, t }, w[4];
            hmc_ref_philox4x32_10(ctr, key, w);
            double X  = (double)((((uint64_t)w[0] << 32) | w[1]) >> 11) * two_m53;
            double Xp = (double)((((uint64_t)w[2] << 32) | w[3]) >> 11) * two_m53;
            double s = 2.0 * X - 1.0;
            double r0 = mid + quarter * (3.0 * s - (s * s) * s);       /* replaces Eq. 14 */
            uint64_t j = shell_of(&T, r0, kmin, kmax);
            double phi0 = phi_in_shell(&T, j, r0);                      /* Eq. 6 */
            double Q0 = 2.0 * (E - phi0) - J2 / (r0 * r0);              /* Eq. 12 */
            if (Q0 > 0.0) {
                double g = (three_q * (1.0 - s * s)) / sqrt(Q0);
                have_good = 1; good_r = r0; good_Q = Q0; good_w3 = w[3];
                if (g > F) st |= ST_CLIPPED;
                if (F * Xp < g) { accepted = 1; break; }                /* Eq. 15 with f -> g */
            }
        }
        uint32_t used = accepted ? t + 1 : T_MAX;
        total_trials += used;
        if (!accepted) st |= ST_MAXTRIES;
        if (have_good) {
            r_new[i] = good_r;
            v_t_new[i] = J / good_r;
            double vr = sqrt(good_Q);                                   /* v_r = Q^(1/2) */
            v_r_new[i] = (good_w3 & 1u) ? -vr : vr;
        }
        if (n_try) n_try[i] = (uint16_t)used;
        status_out[i] = (uint8_t)st;
    }
    if (counters) counters[0] += total_trials;
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Diagnostics on the radius-sorted arrays ("half-mass radius   */
/* ... that control program termination"; :346 Eq. 20; :354 total energy).   */
/* SURVEY.md 8(f) item 4.  Readings (R15-R17):                    */
/*  - kinetic energy T = sum_k m_k * (0.5 * (v_r^2 + v_t^2)), potential     */
/*    energy W = sum_k 0.5 * (m_k * Phi_k) (Phi_k of Eq. 1 contains the      */
/*    star's own term, as the paper's potential does); each term is the     */
/*    binary64 value of the expression written, the SUM is exact, rounded   */
/*    once (binary128 accumulator, as for Eq. 3-5);                          */
/*  - E_tot = T + W, virial ratio = (2 T) / |W|;                            */
/*  - Lagrange radius of mass fraction f: r_k of the first star k with      */
/*    M_k >= f * M_N (binary64 product); half-mass radius r_h = f = 1/2;    */
/*  - t_rh = 0.138 N / ln(0.1 N) * (r_h^3 / (G M_N))^(1/2), Eq. 20.         */
/* out: [0] M_N, [1] T, [2] W, [3] E_tot, [4] virial ratio, [5] r_h,        */
/*      [6] t_rh, [7 .. 7 + nfrac) Lagrange radii of fractions[].           */
/* ------------------------------------------------------------------------ */
static double lagrange_radius(uint64_t n, const double *r, const double *m_cum, double f)
{
    double target = f * m_cum[n - 1];
    uint64_t k = 0;
    while (k + 1 < n && !(m_cum[k] >= target)) ++k;      /* first k with M_k >= target, else the last star */
    return r[k];
}

int hmc_ref_diagnostics(uint64_t n, double G, const double *r, const double *v_r, const double *v_t,
                        const double *m, const double *phi, const double *m_cum,
                        int nfrac, const double *fractions, double *out)
{
    if (n == 0) return -2;
    __float128 accT = 0, accW = 0;
    for (uint64_t a = 0; a < n; ++a) {
        double t = m[a] * (0.5 * (v_r[a] * v_r[a] + v_t[a] * v_t[a]));
        double w = 0.5 * (m[a] * phi[a]);
        accT += (__float128)t;
        accW += (__float128)w;
    }
    double M = m_cum[n - 1], T = (double)accT, W = (double)accW;
    double rh = lagrange_radius(n, r, m_cum, 0.5);
    out[0] = M;
    out[1] = T;
    out[2] = W;
    out[3] = T + W;
    out[4] = (2.0 * T) / fabs(W);
    out[5] = rh;
    out[6] = ((0.138 * (double)n) / log(0.1 * (double)n)) * sqrt(((rh * rh) * rh) / (G * M));
    for (int i = 0; i < nfrac; ++i) out[7 + i] = lagrange_radius(n, r, m_cum, fractions[i]);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Energy correction for the time-varying potential ("corrections */
/* are made to the kinetic energy of each particle that account for the fact  */
/* that the new orbit has been calculated in the old potential ... adjusting   */
/* the stellar velocities according to the mechanical work done on the stellar */
/* orbit by the time varying potential ... such that the ratio v_r/v_t is      */
/* preserved"; formula deferred to Stodolkiewicz 1982 / Fregeau & Rasio 2007,  */
/* not in the paper's text).  SURVEY.md 8(f) item 2.  Reading DESIGN.md R18:   */
/* dE/dt = dPhi/dt along the orbit, integrated over the step by the mean of    */
/* the potential change at the two positions known, the old and the new one:   */
/*   dE = 1/2 [ (Phi'(r_old) - Phi(r_old)) + (Phi'(r_new) - Phi(r_new)) ]      */
/* Phi = potential the orbit was drawn in (previous step), Phi' = potential of */
/* the new configuration.  With the shell potential this makes the total       */
/* energy T + W exactly invariant: sum_i m_i Phi'(r_old,i) and                 */
/* sum_i m_i Phi(r_new,i) are the same double sum over pairs.                  */
/* Arrays are in the NEW radius-sorted order, star k at node k:                */
/*   r, phi, m_cum  the new table (Phi'(r_new) of star k is phi[k]);            */
/*   E_old          the star's energy in the old potential (S3's E);            */
/*   r_old, p_old   its previous radius and Phi(r_old) (the old table at its    */
/*                  own node), carried through the sort;                        */
/*   v_r, v_t       the velocities S4 gave it.                                  */
/* Phi(r_new) is taken from the draw's energy identity, Phi(r_new) = E_old - K, */
/* K = (v_r^2 + v_t^2)/2; Phi'(r_old) by Eq. 6 (anchored, R3) in the new table. */
/* New kinetic energy K' = (E_old + dE) - Phi'(r_new); both velocity components */
/* are scaled by sqrt(K'/K).  K' <= 0 or K <= 0: flag ST_NOKINETIC, unchanged.  */
/* ------------------------------------------------------------------------ */
#define ST_NOKINETIC 64u

int hmc_ref_energy_correction(uint64_t n, double G, const double *r, const double *phi, const double *m_cum,
                              const double *E_old, const double *r_old, const double *p_old,
                              const double *v_r, const double *v_t,
                              double *v_r_out, double *v_t_out, uint8_t *status_out)
{
    table T = { n, G, r, phi, m_cum };
#pragma omp parallel for schedule(dynamic, 4096)
    for (uint64_t a = 0; a < n; ++a) {
        double vr = v_r[a], vt = v_t[a];
        double K = 0.5 * (vr * vr + vt * vt);
        double pn = E_old[a] - K;                                /* Phi(r_new) */
        uint64_t j = shell_of(&T, r_old[a], 0, n);
        double po2 = phi_in_shell(&T, j, r_old[a]);              /* Phi'(r_old) */
        double dE = 0.5 * ((po2 - p_old[a]) + (phi[a] - pn));
        double Kp = (E_old[a] + dE) - phi[a];
        unsigned st = 0;
        if (Kp > 0.0 && K > 0.0) {
            double lam = sqrt(Kp / K);
            vr = lam * vr; vt = lam * vt;
        } else st |= ST_NOKINETIC;
        v_r_out[a] = vr; v_t_out[a] = vt; status_out[a] = (uint8_t)st;
    }
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Relaxation timestep and two-body relaxation on neighbour pairs           */
/* (Eq. 7 at :87; bins of 20 at :194).  SURVEY.md 8(f) 3.  */
/*                                                                          */
/* Eq. 7:  T_rel = (theta_max / (pi/2)) (pi/32) <v_rel>^3                   */
/*                 / ( ln(gamma N) G^2 n <(M_1 + M_2)^2> ).                 */
/* "Instead of using sliding averages for each star, we choose radial bins  */
/* containing a fixed number of stars ... a bin size of 20"; */
/* "the minimum is taken as the value of the global relaxation timestep"    */
/* (:108).  Readings (R19):                                       */
/*  - bin b = sorted stars 20b .. 20b+19; the n mod 20 stars left over join */
/*    the last bin; n < 20: one bin.                                        */
/*  - pairs are the neighbours (2j, 2j+1) of the sorted order ("pairs of    */
/*    neighboring stars", :177), which never straddle a bin; an odd last    */
/*    star has no partner.                                                  */
/*  - v_rel of a pair: its transverse velocities make an unknown angle,     */
/*    uniform in [0, 2 pi); the timestep takes the rms over that angle,     */
/*    v_rel = sqrt((v_r1 - v_r2)^2 + v_t1^2 + v_t2^2); < > is the mean over */
/*    the bin's pairs, summed in pair order.                                */
/*  - n: the shell between the last star of the previous bin (r = 0 for the */
/*    first bin) and the last star of this bin holds exactly the bin's      */
/*    stars: n = count / ((4 pi / 3) (r_out^3 - r_in^3)).                   */
/*  - ln(gamma N) is passed in (the caller evaluates the logarithm once).   */
/*  - a bin without a pair, with zero volume, or with zero mass: no         */
/*    constraint, T = +inf (zero volume: n = inf gives T = 0, kept).        */
/* ------------------------------------------------------------------------ */
#define BIN 20u
#define FOUR_PI_3 4.1887902047863909846   /* 4 pi / 3 */
#define PI_OVER_2 1.5707963267948966192
#define PI_OVER_32 0.098174770424681038702
#define TWO_PI 6.2831853071795864769

static uint64_t n_bins(uint64_t n) { return n < BIN ? (n ? 1 : 0) : n / BIN; }

/* number density of bin b (count / volume of its shell) */
static double bin_density(uint64_t n, const double *r, uint64_t b)
{
    uint64_t nb = n_bins(n);
    uint64_t first = b * BIN, last = (b + 1 == nb) ? n - 1 : first + BIN - 1;
    double r_in = b ? r[first - 1] : 0.0, r_out = r[last];
    double vol = FOUR_PI_3 * ((r_out * r_out) * r_out - (r_in * r_in) * r_in);
    return (double)(last - first + 1) / vol;
}

int hmc_ref_relaxation_timestep(uint64_t n, double G, double ln_gamma_n, double theta_max,
                                const double *r, const double *v_r, const double *v_t, const double *m,
                                double *t_rel_bin, double *t_rel_min)
{
    uint64_t nb = n_bins(n);
    double tmin = INFINITY;
    for (uint64_t b = 0; b < nb; ++b) {
        uint64_t first = b * BIN, last = (b + 1 == nb) ? n - 1 : first + BIN - 1;
        double sv = 0.0, sm = 0.0;
        uint64_t pairs = 0;
        for (uint64_t a = first; a + 1 <= last; a += 2) {
            double dvr = v_r[a] - v_r[a + 1];
            double w = sqrt(dvr * dvr + v_t[a] * v_t[a] + v_t[a + 1] * v_t[a + 1]);
            double M = m[a] + m[a + 1];
            sv += w; sm += M * M;
            ++pairs;
        }
        double T = INFINITY;
        if (pairs) {
            double vmean = sv / (double)pairs, m2mean = sm / (double)pairs;
            double dens = bin_density(n, r, b);
            double den = ((ln_gamma_n * (G * G)) * dens) * m2mean;
            if (den > 0.0) T = (((theta_max / PI_OVER_2) * PI_OVER_32) * ((vmean * vmean) * vmean)) / den;
        }
        if (t_rel_bin) t_rel_bin[b] = T;
        if (T < tmin) tmin = T;
    }
    *t_rel_min = tmin;
    return 0;
}

/* ------------------------------------------------------------------------ */
/* "Two-body relaxation is applied based on an analytic expression for a    */
/* representative encounter between two nearest-neighbor stars"             */
/* (PAPER.md:110); the expression is deferred to Joshi et al. (2000) and is  */
/* not in the text.  Reading DESIGN.md R20 (Henon's scheme):                */
/*  - the pair (1, 2) = sorted stars (2j, 2j+1); in a local frame with z    */
/*    radial, v_1 = (v_t1, 0, v_r1), v_2 = (v_t2 cos phi, v_t2 sin phi,     */
/*    v_r2), phi uniform;  w = v_1 - v_2,  V = (m_1 v_1 + m_2 v_2) / M,     */
/*    M = m_1 + m_2;                                                        */
/*  - one encounter deflects w by the angle beta that the many distant      */
/*    encounters of the step dt add up to: the mean square deflection       */
/*    behind Eq. 7, <beta^2> = 8 pi G^2 n M^2 ln(gamma N) dt / w^3 (Eq. 7   */
/*    is this set to (pi/2) theta_max), carried by sin^2(beta/2) =          */
/*    2 pi G^2 M^2 n ln(gamma N) dt / w^3, capped at 1;                     */
/*  - w' = w cos beta + |w| sin beta (e_1 cos psi + e_2 sin psi), psi       */
/*    uniform, e_1 = (w_y, -w_x, 0)/w_p, e_2 = (w_x w_z, w_y w_z, -w_p^2) /  */
/*    (w_p |w|), w_p = (w_x^2 + w_y^2)^(1/2) (w along z: e_1 = x, e_2 = y); */
/*  - v_1' = V + (m_2/M) w',  v_2' = V - (m_1/M) w': the pair's momentum    */
/*    and kinetic energy are conserved;  v_r' = z,  v_t' = (x^2+y^2)^(1/2). */
/*  - unit vectors (cos, sin) without trigonometric functions (which are    */
/*    not correctly rounded): (a, b) uniform in the unit disc by rejection, */
/*    then (cos, sin) = ((a^2 - b^2)/s, 2ab/s), s = a^2 + b^2 -- the        */
/*    doubled angle of a uniform point is uniform.  Draw t of the pair      */
/*    uses Philox4x32-10(counter = (id of star 1, 1, step, t)); phi takes   */
/*    the first accepted draw, psi the next accepted one (at most 64 draws, */
/*    then (1, 0)).                                                         */
/*  n is the pair's bin density as in the timestep.                          */
/* ------------------------------------------------------------------------ */
static void unit_vector(uint32_t id, uint32_t step, const uint32_t key[2], uint32_t *t, double *c, double *s_out)
{
    const double two_m53 = 1.0 / 9007199254740992.0;
    while (*t < 64u) {
        uint32_t ctr[4] = { id, 1u, step, *t }, w[4];
        ++*t;
        hmc_ref_philox4x32_10(ctr, key, w);
        double a = 2.0 * ((double)((((uint64_t)w[0] << 32) | w[1]) >> 11) * two_m53) - 1.0;
        double b = 2.0 * ((double)((((uint64_t)w[2] << 32) | w[3]) >> 11) * two_m53) - 1.0;
        double s = a * a + b * b;
        if (s > 0.0 && s < 1.0) { *c = (a * a - b * b) / s; *s_out = (2.0 * (a * b)) / s; return; }
    }
    *c = 1.0; *s_out = 0.0;
}

int hmc_ref_two_body_relaxation(uint64_t n, double G, double ln_gamma_n, double dt, uint64_t seed, uint32_t step,
                                const double *r, const double *v_r, const double *v_t, const double *m,
                                const uint32_t *id, double *v_r_out, double *v_t_out)
{
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint64_t nb = n_bins(n);
#pragma omp parallel for schedule(dynamic, 4096)
    for (uint64_t j = 0; j < (n + 1) / 2; ++j) {
        uint64_t a = 2 * j, b = a + 1;
        if (b >= n) { v_r_out[a] = v_r[a]; v_t_out[a] = v_t[a]; continue; }      /* odd star out */
        uint64_t bin = a / BIN; if (bin >= nb) bin = nb - 1;
        double dens = bin_density(n, r, bin);
        double m1 = m[a], m2 = m[b], M = m1 + m2;
        uint32_t t = 0;
        double cphi, sphi, cpsi, spsi;
        unit_vector(id[a], step, key, &t, &cphi, &sphi);
        unit_vector(id[a], step, key, &t, &cpsi, &spsi);
        double x1 = v_t[a], z1 = v_r[a];
        double x2 = v_t[b] * cphi, y2 = v_t[b] * sphi, z2 = v_r[b];
        double wx = x1 - x2, wy = 0.0 - y2, wz = z1 - z2;
        double wp2 = wx * wx + wy * wy, w2 = wp2 + wz * wz, wn = sqrt(w2);
        if (!(wn > 0.0) || !(M > 0.0)) {
            v_r_out[a] = v_r[a]; v_t_out[a] = v_t[a]; v_r_out[b] = v_r[b]; v_t_out[b] = v_t[b];
            continue;
        }
        double S = (((((TWO_PI * (G * G)) * (M * M)) * dens) * ln_gamma_n) * dt) / (w2 * wn);
        /* DESIGN.md R20a: no encounter where the expression has no value -- S is NaN (a zero-volume bin, density  */
        /* infinite, with dt = 0: what T_rel's minimum gives when such a bin exists) or dt is not finite (no bin   */
        /* holds a pair, T_rel = +inf).  Otherwise a step of zero length would turn every such pair head-on.       */
        if (S != S || !(dt < INFINITY)) S = 0.0;
        if (!(S < 1.0)) S = 1.0;
        if (!(S > 0.0)) S = 0.0;
        double cb = 1.0 - 2.0 * S, sb = 2.0 * sqrt(S * (1.0 - S));
        double wp = sqrt(wp2);
        double e1x, e1y, e1z, e2x, e2y, e2z;
        if (wp > 0.0) {
            e1x = wy / wp; e1y = (0.0 - wx) / wp; e1z = 0.0;
            double q = wp * wn;
            e2x = (wx * wz) / q; e2y = (wy * wz) / q; e2z = (0.0 - wp2) / q;
        } else { e1x = 1.0; e1y = 0.0; e1z = 0.0; e2x = 0.0; e2y = 1.0; e2z = 0.0; }
        double k = wn * sb;
        double nx = wx * cb + k * (e1x * cpsi + e2x * spsi);
        double ny = wy * cb + k * (e1y * cpsi + e2y * spsi);
        double nz = wz * cb + k * (e1z * cpsi + e2z * spsi);
        double Vx = (m1 * x1 + m2 * x2) / M, Vy = (m2 * y2) / M, Vz = (m1 * z1 + m2 * z2) / M;
        double f1 = m2 / M, f2 = m1 / M;
        double ax = Vx + f1 * nx, ay = Vy + f1 * ny, az = Vz + f1 * nz;
        double bx = Vx - f2 * nx, by = Vy - f2 * ny, bz = Vz - f2 * nz;
        v_r_out[a] = az; v_t_out[a] = sqrt(ax * ax + ay * ay);
        v_r_out[b] = bz; v_t_out[b] = sqrt(bx * bx + by * by);
    }
    return 0;
}
