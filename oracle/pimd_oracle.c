/*
 * oracle/pimd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-translation-unit CPU restatement of the force evaluation
 * of bosonic / xi-particle path integral molecular dynamics exactly as
 * arXiv 2404.02628 writes it (cited below as PAPER.md:<line>, Eq. <n>).
 * It shares no code, header, table or constant generator with the CUDA path
 * under paper_2404_02628_b200/csrc/ and neither includes the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * Conventions
 *   units hbar = m = k_B = 1.
 *   x[j][l][c]  bead j (0..P-1 <-> paper's 1..P), particle l (0..N-1 <-> 1..N),
 *               coordinate c (0..d-1);  flat index ((j*N)+l)*d+c.
 *   k_s = m omega_P^2 = P / beta^2   (omega_P = sqrt(P)/(beta hbar)).
 *   Every potential term of H enters the sampled weight as U/P (Eq. 4).
 *   The pair potential is v(r) = g exp(-r^2/s^2) (BASELINE.json north_star; the
 *   paper's Eq. 20 prefactor g_paper/(pi s^2) maps to g here; reading R4).
 *
 * Precision: FP64 inputs/outputs.  Sums that add many terms (chains of spring
 * energies, the log-sum-exp sums) are carried in long double so the oracle's
 * own rounding is well below the 1e-9 parity tolerance at N = 1e4.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"):
 *   E^{[u,v]}      literal Eq. 7 triple loop written in the test            PINNED
 *   V_B            2^{N-1} composition sum, relabel-averaged N! sum,
 *                  identical-ring closed form, xi=0 closed form, L_N = M_1  PINNED
 *   Pr             row sums = column sums = 1, xi=0 identity                PINNED
 *   forces         central finite differences of the potential, sum F = 0,
 *                  two-particle closed form, Newton's third law             PINNED
 *   estimators     d(beta V_B)/d beta by finite differences, virial vs
 *                  primitive ensemble agreement, exact ideal-gas energy     PINNED
 *   orc_step       NVE reversibility / energy drift, <v^2> = 1/beta,
 *                  ensemble energy vs exact; Nose-Hoover chain (nhc_half):
 *                  reversibility under (v, v_xi) -> (-v, -v_xi) and the
 *                  conserved extended energy to O(dt^2)                     PINNED
 *                  The parameter CHOICES the paper leaves open (chain length
 *                  4, Q = beta/P, gamma = 1; R10) have no reference
 *                  to be checked against:                                   PARITY UNPINNED (parameters only)
 *   orc_philox_normal  Philox4x32-10 known-answer vector (Random123 KAT)    PINNED
 *   orc_stream_*   (O(N) memory) brute-force finite differences at small N,
 *                  identical-ring closed form at N = 3000                   PINNED
 *   orc_*_species  product of two composition sums, finite differences      PINNED
 *   pair potential kind 1: finite differences, two-particle closed form     PINNED
 *   orc_pair_histogram  numpy histogram of brute-force distances            PINNED
 *   orc_conditioning    = 1 for xi >= 0; N = 2 closed form for xi < 0       PINNED
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_OK 0
#define ORC_EINVAL -1
#define ORC_ENOMEM -2
#define ORC_ENODE -4 /* e^{-beta V} summed to exactly zero (xi<0 node) */

#define IDX(j, l, c) ((((size_t)(j)) * (size_t)N + (size_t)(l)) * (size_t)d + (size_t)(c))

static double sqdist(const double *a, const double *b, int d)
{
    double r2 = 0.0;
    for (int c = 0; c < d; ++c) {
        double t = a[c] - b[c];
        r2 += t * t;
    }
    return r2;
}

/* 1/2 m omega_P^2 (r_l^P - r_lp^1)^2 : the spring that ties the last bead of
 * particle l to the first bead of particle lp (the terms of Eq. 7 with j = P,
 * PAPER.md:73-76). */
static double closing(const double *x, int N, int P, int d, double ks, int l, int lp)
{
    return 0.5 * ks * sqdist(&x[IDX(P - 1, l, 0)], &x[IDX(0, lp, 0)], d);
}

/* Eq. 9: E_int^{(v)} = 1/2 m omega_P^2 sum_{j=1}^{P-1} (r_v^{j+1}-r_v^j)^2 */
int orc_eint(const double *x, int N, int P, int d, double beta, double *Eint)
{
    if (N < 1 || P < 2 || d < 1 || !(beta > 0)) return ORC_EINVAL;
    const double ks = (double)P / (beta * beta);
    for (int v = 0; v < N; ++v) {
        long double acc = 0.0L;
        for (int j = 0; j + 1 < P; ++j)
            acc += (long double)sqdist(&x[IDX(j + 1, v, 0)], &x[IDX(j, v, 0)], d);
        Eint[v] = (double)(0.5L * ks * acc);
    }
    return ORC_OK;
}

/* Eq. 7 for one (u,v), 1-based, literally: double sum over
 * l = u..v and j = 1..P with r_l^{P+1} = r_{l+1}^1 unless l = v where
 * r_v^{P+1} = r_u^1.  O((v-u+1) P).  Used for small-N cross checks. */
double orc_cycle_energy_eq7(const double *x, int N, int P, int d, double beta, int u, int v)
{
    const double ks = (double)P / (beta * beta);
    long double acc = 0.0L;
    for (int l = u; l <= v; ++l) {
        for (int j = 1; j <= P; ++j) {
            const double *a = &x[IDX(j - 1, l - 1, 0)];
            const double *b;
            if (j < P)
                b = &x[IDX(j, l - 1, 0)];
            else if (l < v)
                b = &x[IDX(0, l, 0)]; /* r_{l+1}^1 */
            else
                b = &x[IDX(0, u - 1, 0)]; /* r_u^1 closes the ring */
            acc += (long double)sqdist(b, a, d);
        }
    }
    return (double)(0.5L * ks * acc);
}

/* All E^{[u,v]}, 1 <= u <= v <= N, stored at E[(u-1)*N + (v-1)] (upper
 * triangle; the rest is left untouched).  This is Eq. 7 with the shared
 * partial sums written once: for fixed v walk u = v, v-1, .., 1 and keep
 *   chain(u..v) = sum_{l=u}^{v} E_int^{(l)} + sum_{l=u}^{v-1} C(l,l+1),
 *   E^{[u,v]}  = chain(u..v) + C(v,u).
 * Additions only, O(N^2 + NP) as PAPER.md:97 states for Eq. 8-10. */
int orc_cycle_energies(const double *x, int N, int P, int d, double beta, long double *E)
{
    if (N < 1 || P < 2 || d < 1 || !(beta > 0)) return ORC_EINVAL;
    const double ks = (double)P / (beta * beta);
    double *Eint = (double *)malloc(sizeof(double) * (size_t)N);
    if (!Eint) return ORC_ENOMEM;
    orc_eint(x, N, P, d, beta, Eint);
    for (int v = 0; v < N; ++v) {
        long double chain = 0.0L;
        for (int u = v; u >= 0; --u) {
            chain += (long double)Eint[u];
            if (u < v) chain += (long double)closing(x, N, P, d, ks, u, u + 1);
            E[(size_t)u * N + v] = chain + (long double)closing(x, N, P, d, ks, v, u);
        }
    }
    free(Eint);
    return ORC_OK;
}

/* Eq. 8 and the iteration Eq. 10, literally, in
 * double.  Same storage as orc_cycle_energies.  Kept to show that the
 * regrouped Eq. 7 above and the paper's iterative update agree. */
int orc_cycle_energies_eq10(const double *x, int N, int P, int d, double beta, double *E)
{
    if (N < 1 || P < 2 || d < 1 || !(beta > 0)) return ORC_EINVAL;
    const double ks = (double)P / (beta * beta);
    double *Eint = (double *)malloc(sizeof(double) * (size_t)N);
    if (!Eint) return ORC_ENOMEM;
    orc_eint(x, N, P, d, beta, Eint);
    for (int v = 0; v < N; ++v) {
        E[(size_t)v * N + v] = Eint[v] + closing(x, N, P, d, ks, v, v); /* Eq. 8 */
        for (int u = v - 1; u >= 0; --u) {                                /* Eq. 10 */
            E[(size_t)u * N + v] = E[(size_t)(u + 1) * N + v]
                                   - closing(x, N, P, d, ks, v, u + 1)
                                   + closing(x, N, P, d, ks, u, u + 1)
                                   + closing(x, N, P, d, ks, v, u)
                                   + Eint[u];
        }
    }
    free(Eint);
    return ORC_OK;
}

/* signed log-sum-exp of n terms: sum_i sg[i] exp(t[i]) = (*sgn) exp(return) */
static int signed_lse(const long double *t, const int *sg, int n, long double *out, int *sgn)
{
    long double m = -INFINITY;
    for (int i = 0; i < n; ++i)
        if (t[i] > m) m = t[i];
    if (!(m > -INFINITY)) return ORC_ENODE;
    long double sum = 0.0L;
    for (int i = 0; i < n; ++i) sum += (long double)sg[i] * (long double)exp((double)(t[i] - m));
    if (sum == 0.0L || !isfinite((double)sum)) return ORC_ENODE;
    *sgn = sum > 0 ? 1 : -1;
    *out = m + logl(fabsl(sum));
    return ORC_OK;
}

/* Eq. 6, n = 1..N, base V^{[1,0]} = 0 (reading R3):
 *   e^{-beta V^{[1,n]}} = (1/n) sum_{k=1}^{n} xi^{k-1} e^{-beta (E^{[n-k+1,n]} + V^{[1,n-k]})}
 * L[n] = -beta V^{[1,n]} (log of the magnitude), sg[n] its sign; L, sg have N+1
 * entries.  xi = 0 keeps only k = 1 (0^0 = 1). */
int orc_forward(const long double *E, int N, double beta, double xi, long double *L, int *sg)
{
    const long double lam = (xi != 0.0) ? logl(fabsl((long double)xi)) : 0.0L;
    const int sx = xi < 0 ? -1 : 1;
    long double *t = (long double *)malloc(sizeof(long double) * (size_t)N);
    int *s = (int *)malloc(sizeof(int) * (size_t)N);
    if (!t || !s) { free(t); free(s); return ORC_ENOMEM; }
    L[0] = 0.0L;
    sg[0] = 1;
    int rc = ORC_OK;
    for (int n = 1; n <= N && rc == ORC_OK; ++n) {
        int cnt = 0;
        for (int k = 1; k <= n; ++k) {
            if (xi == 0.0 && k > 1) break;
            const int u = n - k + 1;
            t[cnt] = (long double)(k - 1) * lam - (long double)beta * E[(size_t)(u - 1) * N + (n - 1)] + L[n - k];
            s[cnt] = (((k - 1) & 1) ? sx : 1) * sg[n - k];
            ++cnt;
        }
        long double lse;
        int sgn;
        rc = signed_lse(t, s, cnt, &lse, &sgn);
        if (rc == ORC_OK) {
            L[n] = -logl((long double)n) + lse;
            sg[n] = sgn;
        }
    }
    free(t);
    free(s);
    return rc;
}

/* Eq. 11, u = N..1:
 *   e^{-beta V^{[u,N]}} = sum_{l=u}^{N} xi^{l-u} (1/l) e^{-beta (E^{[u,l]} + V^{[l+1,N]})}
 * with the empty-range base V^{[N+1,N]} = 0 (the printed "V^{[N,N]} = 0",
 * PAPER.md:105, contradicts Eq. 11 at u = N; reading R2).
 * M[u] = -beta V^{[u,N]}, u = 1..N+1 (M[0] unused); M, sg have N+2 entries. */
int orc_backward(const long double *E, int N, double beta, double xi, long double *M, int *sg)
{
    const long double lam = (xi != 0.0) ? logl(fabsl((long double)xi)) : 0.0L;
    const int sx = xi < 0 ? -1 : 1;
    long double *t = (long double *)malloc(sizeof(long double) * (size_t)N);
    int *s = (int *)malloc(sizeof(int) * (size_t)N);
    if (!t || !s) { free(t); free(s); return ORC_ENOMEM; }
    M[0] = 0.0L;
    sg[0] = 1;
    M[N + 1] = 0.0L;
    sg[N + 1] = 1;
    int rc = ORC_OK;
    for (int u = N; u >= 1 && rc == ORC_OK; --u) {
        int cnt = 0;
        for (int l = u; l <= N; ++l) {
            if (xi == 0.0 && l > u) break;
            t[cnt] = (long double)(l - u) * lam - logl((long double)l)
                     - (long double)beta * E[(size_t)(u - 1) * N + (l - 1)] + M[l + 1];
            s[cnt] = (((l - u) & 1) ? sx : 1) * sg[l + 1];
            ++cnt;
        }
        long double lse;
        int sgn;
        rc = signed_lse(t, s, cnt, &lse, &sgn);
        if (rc == ORC_OK) {
            M[u] = lse;
            sg[u] = sgn;
        }
    }
    free(t);
    free(s);
    return rc;
}

/* Eq. 12-14.  Pr[(l-1)*N + (lp-1)] = Pr[G(l) = lp],
 * 1 <= l, lp <= N.  For xi < 0 these are signed quasi-probabilities
 * (reading R7); rows and columns still sum to 1. */
int orc_probabilities(const long double *E, const long double *L, const int *sgL,
                      const long double *M, const int *sgM, int N, double beta, double xi, double *Pr)
{
    const long double lam = (xi != 0.0) ? logl(fabsl((long double)xi)) : 0.0L;
    const int sx = xi < 0 ? -1 : 1;
    for (int l = 1; l <= N; ++l) {
        for (int lp = 1; lp <= N; ++lp) {
            double p = 0.0; /* Eq. 14 */
            if (lp <= l) {  /* Eq. 12 */
                if (!(xi == 0.0 && lp < l)) {
                    long double e = (long double)(l - lp) * lam - logl((long double)l) + L[lp - 1]
                                    - (long double)beta * E[(size_t)(lp - 1) * N + (l - 1)] + M[l + 1] - L[N];
                    int s = (((l - lp) & 1) ? sx : 1) * sgL[lp - 1] * sgM[l + 1] * sgL[N];
                    p = (double)s * exp((double)e);
                }
            } else if (lp == l + 1) { /* Eq. 13 */
                long double e = L[l] + M[l + 1] - L[N];
                int s = sgL[l] * sgM[l + 1] * sgL[N];
                p = 1.0 - (double)s * exp((double)e);
            }
            Pr[(size_t)(l - 1) * N + (lp - 1)] = p;
        }
    }
    return ORC_OK;
}

/* Eq. 15, 16, 17, literally: F = -grad V_xi^{[1,N]}.
 * F is overwritten (layout of x). */
int orc_exchange_forces(const double *x, const double *Pr, int N, int P, int d, double beta, double *F)
{
    const double ks = (double)P / (beta * beta);
    memset(F, 0, sizeof(double) * (size_t)N * P * d);
    /* interior beads, Eq. 17 */
    for (int j = 1; j + 1 < P; ++j)
        for (int l = 0; l < N; ++l)
            for (int c = 0; c < d; ++c)
                F[IDX(j, l, c)] = -ks * (2.0 * x[IDX(j, l, c)] - x[IDX(j + 1, l, c)] - x[IDX(j - 1, l, c)]);
    for (int l = 0; l < N; ++l) {
        for (int c = 0; c < d; ++c) {
            long double f1 = 0.0L, fP = 0.0L;
            for (int lp = 0; lp < N; ++lp) {
                /* Eq. 15: bead 1 of l, weight Pr[G(lp) = l] */
                f1 -= (long double)Pr[(size_t)lp * N + l] * ks
                      * (2.0 * x[IDX(0, l, c)] - x[IDX(1, l, c)] - x[IDX(P - 1, lp, c)]);
                /* Eq. 16: bead P of l, weight Pr[G(l) = lp] */
                fP -= (long double)Pr[(size_t)l * N + lp] * ks
                      * (2.0 * x[IDX(P - 1, l, c)] - x[IDX(P - 2, l, c)] - x[IDX(0, lp, c)]);
            }
            /* P == 2: bead 1 and bead P are different beads, both exterior; += keeps both */
            F[IDX(0, l, c)] += (double)f1;
            F[IDX(P - 1, l, c)] += (double)fP;
        }
    }
    return ORC_OK;
}

/* The pair potential v(r) of Eq. 18 (PAPER.md:142-144 leaves V generic; Eq. 20, is the Gaussian
 * instance), as a function of r^2:
 *   kind 0 (default)  v = g exp(-r^2/s^2)
 *   kind 1            v = g / sqrt(r^2 + s^2)          (soft Coulomb)
 * *v = v(r), *fw = -(1/r) dv/dr (force on l from i is fw (r_l - r_i)), *vir = v + (r/2) dv/dr (virial estimator term). */
static int g_pair_kind = 0;
void orc_set_pair_potential(int kind) { g_pair_kind = kind; }

static void pair_v(double r2, double g, double s, double *v, double *fw, double *vir)
{
    if (g_pair_kind == 0) {
        const double is2 = 1.0 / (s * s);
        const double e = g * exp(-r2 * is2);
        *v = e;
        *fw = 2.0 * is2 * e;
        *vir = (1.0 - r2 * is2) * e;
    } else {
        const double q = r2 + s * s;
        const double rq = sqrt(q);
        *v = g / rq;
        *fw = g / (q * rq);
        *vir = *v - 0.5 * r2 * *fw;
    }
}

/* -(1/P) grad U for U = sum_j [ sum_l 1/2 omega^2 |r_l^j|^2 + sum_{i<l} v(|r_l^j-r_i^j|) ], v = g e^{-r^2/s^2} by default
 * (Eq. 4, Eq. 18 :142, Eq. 19 :158, Eq. 20 :193).  Added into F.
 * Returns Ubar = U/P through *ubar if not NULL. */
int orc_external_forces(const double *x, int N, int P, int d, double omega, double g, double s,
                        double *F, double *ubar_trap, double *ubar_pair)
{
    const double invP = 1.0 / (double)P;
    long double ut = 0.0L, up = 0.0L;
    for (int j = 0; j < P; ++j) {
        for (int l = 0; l < N; ++l) {
            const double *rl = &x[IDX(j, l, 0)];
            double r2 = 0.0;
            for (int c = 0; c < d; ++c) {
                r2 += rl[c] * rl[c];
                F[IDX(j, l, c)] += -invP * omega * omega * rl[c];
            }
            ut += 0.5L * omega * omega * r2;
        }
    }
    if (g != 0.0) {
#pragma omp parallel for schedule(static) reduction(+ : up)
        for (int jl = 0; jl < P * N; ++jl) {
            const int j = jl / N, l = jl % N;
            const double *rl = &x[IDX(j, l, 0)];
            double acc[3] = {0.0, 0.0, 0.0};
            for (int i = 0; i < N; ++i) {
                if (i == l) continue;
                const double *ri = &x[IDX(j, i, 0)];
                double e, fw, vir;
                pair_v(sqdist(rl, ri, d), g, s, &e, &fw, &vir);
                for (int c = 0; c < d; ++c) acc[c] += fw * (rl[c] - ri[c]);
                if (i < l) up += e;
            }
            for (int c = 0; c < d; ++c) F[IDX(j, l, c)] += invP * acc[c];
        }
    }
    if (ubar_trap) *ubar_trap = (double)(ut * invP);
    if (ubar_pair) *ubar_pair = (double)(up * invP);
    return ORC_OK;
}

/* Pair + trap force on the single bead (j,l) only: what the full-size parity
 * tests sample (same formulas as orc_external_forces). */
int orc_external_force_on(const double *x, int N, int P, int d, double omega, double g, double s,
                          int j, int l, double *f)
{
    const double invP = 1.0 / (double)P;
    const double *rl = &x[IDX(j, l, 0)];
    long double acc[3] = {0.0L, 0.0L, 0.0L};
    for (int i = 0; i < N; ++i) {
        if (i == l) continue;
        const double *ri = &x[IDX(j, i, 0)];
        double e, fw, vir;
        pair_v(sqdist(rl, ri, d), g, s, &e, &fw, &vir);
        for (int c = 0; c < d; ++c) acc[c] += fw * (rl[c] - ri[c]);
    }
    for (int c = 0; c < d; ++c) f[c] = invP * (double)acc[c] - invP * omega * omega * rl[c];
    return ORC_OK;
}

typedef struct {
    long double *E;
    long double *L, *M;
    int *sgL, *sgM;
    double *Pr;
} orc_ws;

static void ws_free(orc_ws *w)
{
    free(w->E); free(w->L); free(w->M); free(w->sgL); free(w->sgM); free(w->Pr);
}

static int ws_alloc(orc_ws *w, int N, int need_pr)
{
    memset(w, 0, sizeof(*w));
    w->E = (long double *)malloc(sizeof(long double) * (size_t)N * N);
    w->L = (long double *)malloc(sizeof(long double) * (size_t)(N + 2));
    w->M = (long double *)malloc(sizeof(long double) * (size_t)(N + 2));
    w->sgL = (int *)malloc(sizeof(int) * (size_t)(N + 2));
    w->sgM = (int *)malloc(sizeof(int) * (size_t)(N + 2));
    if (need_pr) w->Pr = (double *)malloc(sizeof(double) * (size_t)N * N);
    if (!w->E || !w->L || !w->M || !w->sgL || !w->sgM || (need_pr && !w->Pr)) {
        ws_free(w);
        return ORC_ENOMEM;
    }
    return ORC_OK;
}

/* V_xi^{[1,n]} for n = 0..N (vb_table, N+1 doubles, may be NULL) and the sign
 * table of e^{-beta V}; returns V_xi^{[1,N]} in *vb. */
int orc_vb(const double *x, int N, int P, int d, double beta, double xi, double *vb, int *sign,
           double *vb_table, double *vback_table)
{
    orc_ws w;
    int rc = ws_alloc(&w, N, 0);
    if (rc) return rc;
    rc = orc_cycle_energies(x, N, P, d, beta, w.E);
    if (!rc) rc = orc_forward(w.E, N, beta, xi, w.L, w.sgL);
    if (!rc && vback_table) rc = orc_backward(w.E, N, beta, xi, w.M, w.sgM);
    if (!rc) {
        *vb = (double)(-w.L[N] / (long double)beta);
        if (sign) *sign = w.sgL[N];
        if (vb_table)
            for (int n = 0; n <= N; ++n) vb_table[n] = (double)(-w.L[n] / (long double)beta);
        if (vback_table)
            for (int u = 1; u <= N + 1; ++u) vback_table[u] = (double)(-w.M[u] / (long double)beta);
    }
    ws_free(&w);
    return rc;
}

/* Full connection-probability matrix (N x N) for a configuration. */
int orc_pr_matrix(const double *x, int N, int P, int d, double beta, double xi, double *Pr)
{
    orc_ws w;
    int rc = ws_alloc(&w, N, 0);
    if (rc) return rc;
    rc = orc_cycle_energies(x, N, P, d, beta, w.E);
    if (!rc) rc = orc_forward(w.E, N, beta, xi, w.L, w.sgL);
    if (!rc) rc = orc_backward(w.E, N, beta, xi, w.M, w.sgM);
    if (!rc) rc = orc_probabilities(w.E, w.L, w.sgL, w.M, w.sgM, N, beta, xi, Pr);
    ws_free(&w);
    return rc;
}

/* The whole force evaluation of one MD step: F = -grad( V_xi^{[1,N]} + U/P ),
 * V_B = V_xi^{[1,N]} and the sign of e^{-beta V}.  include_external = 0 gives
 * the exchange/spring part alone. */
int orc_forces(const double *x, int N, int P, int d, double beta, double omega, double g, double s,
               double xi, int include_external, double *F, double *vb, int *sign)
{
    if (N < 1 || P < 2 || d < 1 || d > 3 || !(beta > 0) || !(s > 0)) return ORC_EINVAL;
    orc_ws w;
    int rc = ws_alloc(&w, N, 1);
    if (rc) return rc;
    rc = orc_cycle_energies(x, N, P, d, beta, w.E);
    if (!rc) rc = orc_forward(w.E, N, beta, xi, w.L, w.sgL);
    if (!rc) rc = orc_backward(w.E, N, beta, xi, w.M, w.sgM);
    if (!rc) rc = orc_probabilities(w.E, w.L, w.sgL, w.M, w.sgM, N, beta, xi, w.Pr);
    if (!rc) rc = orc_exchange_forces(x, w.Pr, N, P, d, beta, F);
    if (!rc && include_external) rc = orc_external_forces(x, N, P, d, omega, g, s, F, NULL, NULL);
    if (!rc) {
        if (vb) *vb = (double)(-w.L[N] / (long double)beta);
        if (sign) *sign = w.sgL[N];
    }
    ws_free(&w);
    return rc;
}

/* Sampled potential Phi = V_xi^{[1,N]} + U/P of Eq. 4; used by
 * the finite-difference pins and the NVE energy-conservation pin. */
int orc_potential(const double *x, int N, int P, int d, double beta, double omega, double g, double s,
                  double xi, double *phi)
{
    double vb, ut = 0.0, up = 0.0;
    int sign;
    int rc = orc_vb(x, N, P, d, beta, xi, &vb, &sign, NULL, NULL);
    if (rc) return rc;
    double *F = (double *)calloc((size_t)N * P * d, sizeof(double));
    if (!F) return ORC_ENOMEM;
    orc_external_forces(x, N, P, d, omega, g, s, F, &ut, &up);
    free(F);
    *phi = vb + ut + up;
    return ORC_OK;
}

/* Estimators for one configuration (readings R9, R15).
 *  E_prim = P d N/(2 beta) + eps^{(N)} + Ubar,  eps^{(n)} = d(beta V^{[1,n]})/d beta:
 *      eps^{(n)} = sum_k w_k (eps^{(n-k)} - E^{[n-k+1,n]}) / sum_k w_k,
 *      w_k = xi^{k-1} e^{-beta (E^{[n-k+1,n]} + V^{[1,n-k]})}   (from Eq. 6 with E ~ beta^-2)
 *  E_vir  = Ubar + 1/2 sum r . grad Ubar
 *         = (1/P) sum_j [ sum_l omega^2 |r|^2 + sum_{i<l} (v + r v'/2)(r) ],  (1 - r^2/s^2) g e^{-r^2/s^2} for the Gaussian
 *  hist[b] = number of beads with |r| in bin b of [0,rmax) (raw counts, nbins doubles);
 *  the density is hist / (N P shell volume), the harness normalises. */
int orc_estimators(const double *x, int N, int P, int d, double beta, double omega, double g, double s,
                   double xi, double *e_prim, double *e_vir, double *hist, int nbins, double rmax)
{
    orc_ws w;
    int rc = ws_alloc(&w, N, 0);
    if (rc) return rc;
    rc = orc_cycle_energies(x, N, P, d, beta, w.E);
    if (!rc) rc = orc_forward(w.E, N, beta, xi, w.L, w.sgL);
    if (rc) { ws_free(&w); return rc; }
    const long double lam = (xi != 0.0) ? logl(fabsl((long double)xi)) : 0.0L;
    const int sx = xi < 0 ? -1 : 1;
    long double *eps = (long double *)malloc(sizeof(long double) * (size_t)(N + 1));
    if (!eps) { ws_free(&w); return ORC_ENOMEM; }
    eps[0] = 0.0L;
    for (int n = 1; n <= N; ++n) {
        long double m = -INFINITY;
        for (int k = 1; k <= n; ++k) {
            if (xi == 0.0 && k > 1) break;
            long double t = (long double)(k - 1) * lam - (long double)beta * w.E[(size_t)(n - k) * N + (n - 1)] + w.L[n - k];
            if (t > m) m = t;
        }
        long double num = 0.0L, den = 0.0L;
        for (int k = 1; k <= n; ++k) {
            if (xi == 0.0 && k > 1) break;
            long double Ek = w.E[(size_t)(n - k) * N + (n - 1)];
            long double t = (long double)(k - 1) * lam - (long double)beta * Ek + w.L[n - k];
            long double wk = (long double)((((k - 1) & 1) ? sx : 1) * w.sgL[n - k]) * (long double)exp((double)(t - m));
            num += wk * (eps[n - k] - Ek);
            den += wk;
        }
        eps[n] = num / den;
    }
    const long double epsN = eps[N];
    free(eps);
    ws_free(&w);

    long double ut = 0.0L, up = 0.0L, vir_pair = 0.0L;
    for (int b = 0; b < nbins; ++b) hist[b] = 0.0;
    for (int j = 0; j < P; ++j) {
        for (int l = 0; l < N; ++l) {
            const double *rl = &x[IDX(j, l, 0)];
            double r2 = 0.0;
            for (int c = 0; c < d; ++c) r2 += rl[c] * rl[c];
            ut += 0.5L * omega * omega * r2;
            if (nbins > 0) {
                double r = sqrt(r2);
                if (r < rmax) {
                    int b = (int)(r / rmax * nbins);
                    if (b >= nbins) b = nbins - 1;
                    hist[b] += 1.0;
                }
            }
            if (g != 0.0) {
                for (int i = 0; i < l; ++i) {
                    double e, fw, vir;
                    pair_v(sqdist(rl, &x[IDX(j, i, 0)], d), g, s, &e, &fw, &vir);
                    up += e;
                    vir_pair += vir;
                }
            }
        }
    }
    const long double invP = 1.0L / P;
    *e_prim = (double)((long double)P * d * N / (2.0L * beta) + epsN + (ut + up) * invP);
    *e_vir = (double)((2.0L * ut + vir_pair) * invP);
    return ORC_OK;
}

/* ------------------------------------------------------------------------
 * Counter-based Gaussian generator (DESIGN.md section "Random numbers").
 * Philox4x32-10 (Salmon et al., SC'11), counter = (dof_lo, dof_hi, step_lo,
 * step_hi), key = (seed_lo, seed_hi).  Words (w0,w1) -> u1, (w2,w3) -> u2,
 * u = ((w_a * 2^32 + w_b) >> 11 + 0.5) * 2^-53 in (0,1); Box-Muller:
 *   z0 = sqrt(-2 ln u1) cos(2 pi u2),  z1 = sqrt(-2 ln u1) sin(2 pi u2).
 * z0 feeds the thermostat half-step that opens MD step `step`, z1 the one
 * that closes it.
 * ---------------------------------------------------------------------- */
static void philox4x32_10(uint32_t c[4], uint32_t k0, uint32_t k1)
{
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c[0];
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c[2];
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
}

void orc_philox_raw(uint64_t seed, uint64_t dof, uint64_t step, uint32_t out[4])
{
    uint32_t c[4] = {(uint32_t)dof, (uint32_t)(dof >> 32), (uint32_t)step, (uint32_t)(step >> 32)};
    philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
    memcpy(out, c, sizeof(c));
}

void orc_philox_normal(uint64_t seed, uint64_t dof, uint64_t step, double z[2])
{
    uint32_t c[4];
    orc_philox_raw(seed, dof, step, c);
    const uint64_t a = ((uint64_t)c[0] << 32) | c[1];
    const uint64_t b = ((uint64_t)c[2] << 32) | c[3];
    const double u1 = ((double)(a >> 11) + 0.5) * 0x1.0p-53;
    const double u2 = ((double)(b >> 11) + 0.5) * 0x1.0p-53;
    const double r = sqrt(-2.0 * log(u1));
    const double th = 6.283185307179586476925286766559 * u2;
    z[0] = r * cos(th);
    z[1] = r * sin(th);
}

/* ------------------------------------------------------------------------
 * Dynamics (reading R10; PAPER.md:175 names "massive Nose-Hoover
 * chains" but gives no parameters).  One MD step, masses 1, target T = 1/beta:
 *   thermostat half-step (dt/2) ; v += dt/2 F ; x += dt v ; F = F(x) ;
 *   v += dt/2 F ; thermostat half-step (dt/2)
 * thermostat 0: none (NVE).
 * thermostat 1: Langevin (OBABO): v <- c1 v + c2 z, c1 = exp(-gamma dt/2),
 *               c2 = sqrt((1 - c1^2)/beta), z from orc_philox_normal.
 * thermostat 2: massive Nose-Hoover chains, one chain of length M = 4 per
 *               degree of freedom, Q_k = 1/(beta omega_P^2) = beta/P, the
 *               Martyna-Tuckerman-Klein half-step update (one Suzuki-Yoshida
 *               weight, one sub-step).  nhc holds M doubles per DOF, layout
 *               nhc[k][dof].
 * F must hold the forces of x on entry and holds those of the new x on exit.
 * ---------------------------------------------------------------------- */
#define ORC_NHC_M 4

static void nhc_half(double *v, double *nhc, size_t ndof, double dt_half, double beta, double Q)
{
    const double kT = 1.0 / beta;
    const double h = dt_half;
    for (size_t i = 0; i < ndof; ++i) {
        double vx[ORC_NHC_M];
        for (int k = 0; k < ORC_NHC_M; ++k) vx[k] = nhc[(size_t)k * ndof + i];
        double vi = v[i];
        double G;
        G = (Q * vx[ORC_NHC_M - 2] * vx[ORC_NHC_M - 2] - kT) / Q;
        vx[ORC_NHC_M - 1] += 0.5 * h * G;
        for (int k = ORC_NHC_M - 2; k >= 0; --k) {
            const double a = exp(-0.25 * h * vx[k + 1]);
            G = (k == 0) ? (vi * vi - kT) / Q : (Q * vx[k - 1] * vx[k - 1] - kT) / Q;
            vx[k] = (vx[k] * a + 0.5 * h * G) * a;
        }
        vi *= exp(-h * vx[0]);
        for (int k = 0; k <= ORC_NHC_M - 2; ++k) {
            const double a = exp(-0.25 * h * vx[k + 1]);
            G = (k == 0) ? (vi * vi - kT) / Q : (Q * vx[k - 1] * vx[k - 1] - kT) / Q;
            vx[k] = (vx[k] * a + 0.5 * h * G) * a;
        }
        G = (Q * vx[ORC_NHC_M - 2] * vx[ORC_NHC_M - 2] - kT) / Q;
        vx[ORC_NHC_M - 1] += 0.5 * h * G;
        v[i] = vi;
        for (int k = 0; k < ORC_NHC_M; ++k) nhc[(size_t)k * ndof + i] = vx[k];
    }
}

int orc_step(double *x, double *v, double *F, double *nhc, int N, int P, int d, double beta, double omega,
             double g, double s, double xi, double dt, int thermostat, double gamma, uint64_t seed,
             uint64_t step0, int nsteps)
{
    const size_t ndof = (size_t)N * P * d;
    const double c1 = exp(-gamma * dt * 0.5);
    const double c2 = sqrt((1.0 - c1 * c1) / beta);
    const double Q = beta / (double)P;
    for (int it = 0; it < nsteps; ++it) {
        const uint64_t step = step0 + (uint64_t)it;
        if (thermostat == 1) {
            for (size_t i = 0; i < ndof; ++i) {
                double z[2];
                orc_philox_normal(seed, i, step, z);
                v[i] = c1 * v[i] + c2 * z[0];
            }
        } else if (thermostat == 2) {
            nhc_half(v, nhc, ndof, 0.5 * dt, beta, Q);
        }
        for (size_t i = 0; i < ndof; ++i) v[i] += 0.5 * dt * F[i];
        for (size_t i = 0; i < ndof; ++i) x[i] += dt * v[i];
        int rc = orc_forces(x, N, P, d, beta, omega, g, s, xi, 1, F, NULL, NULL);
        if (rc) return rc;
        for (size_t i = 0; i < ndof; ++i) v[i] += 0.5 * dt * F[i];
        if (thermostat == 1) {
            for (size_t i = 0; i < ndof; ++i) {
                double z[2];
                orc_philox_normal(seed, i, step, z);
                v[i] = c1 * v[i] + c2 * z[1];
            }
        } else if (thermostat == 2) {
            nhc_half(v, nhc, ndof, 0.5 * dt, beta, Q);
        }
    }
    return ORC_OK;
}

/* double-precision copy of orc_cycle_energies for callers without long double */
int orc_cycle_energies_d(const double *x, int N, int P, int d, double beta, double *E)
{
    long double *El = (long double *)malloc(sizeof(long double) * (size_t)N * N);
    if (!El) return ORC_ENOMEM;
    int rc = orc_cycle_energies(x, N, P, d, beta, El);
    if (!rc)
        for (int u = 0; u < N; ++u)
            for (int v = 0; v < N; ++v) E[(size_t)u * N + v] = (v >= u) ? (double)El[(size_t)u * N + v] : 0.0;
    free(El);
    return rc;
}

/* ------------------------------------------------------------------------
 * Conditioning of the signed sums (reading R7; xi < 0 lies outside the
 * paper's stated domain).  kappa = the largest ratio
 * sum|terms| / |sum terms| met in Eq. 6 (every n), in Eq. 11 (every u), and in
 * the row and column sums of the quasi-probabilities of Eq. 12-14 (which are 1,
 * so there it is sum |Pr|).  For xi >= 0 every term is positive and kappa = 1.
 * The parity tolerance of a signed case is 1e-9 * kappa.
 * ---------------------------------------------------------------------- */
int orc_conditioning(const double *x, int N, int P, int d, double beta, double xi, double *kappa)
{
    orc_ws w;
    int rc = ws_alloc(&w, N, 1);
    if (rc) return rc;
    rc = orc_cycle_energies(x, N, P, d, beta, w.E);
    if (!rc) rc = orc_forward(w.E, N, beta, xi, w.L, w.sgL);
    if (!rc) rc = orc_backward(w.E, N, beta, xi, w.M, w.sgM);
    if (!rc) rc = orc_probabilities(w.E, w.L, w.sgL, w.M, w.sgM, N, beta, xi, w.Pr);
    if (rc) { ws_free(&w); return rc; }
    const long double lam = (xi != 0.0) ? logl(fabsl((long double)xi)) : 0.0L;
    long double k = 1.0L;
    for (int n = 1; n <= N; ++n) { /* Eq. 6: sum_k |term_k| / |sum| = sum_k exp(t_k - ln n - L_n) */
        long double a = 0.0L;
        for (int kk = 1; kk <= n; ++kk) {
            if (xi == 0.0 && kk > 1) break;
            a += expl((long double)(kk - 1) * lam - (long double)beta * w.E[(size_t)(n - kk) * N + (n - 1)] + w.L[n - kk]
                      - logl((long double)n) - w.L[n]);
        }
        if (a > k) k = a;
    }
    for (int u = N; u >= 1; --u) { /* Eq. 11 */
        long double a = 0.0L;
        for (int l = u; l <= N; ++l) {
            if (xi == 0.0 && l > u) break;
            a += expl((long double)(l - u) * lam - logl((long double)l) - (long double)beta * w.E[(size_t)(u - 1) * N + (l - 1)]
                      + w.M[l + 1] - w.M[u]);
        }
        if (a > k) k = a;
    }
    for (int l = 0; l < N; ++l) {
        long double r = 0.0L, c = 0.0L;
        for (int m = 0; m < N; ++m) {
            r += fabsl((long double)w.Pr[(size_t)l * N + m]);
            c += fabsl((long double)w.Pr[(size_t)m * N + l]);
        }
        if (r > k) k = r;
        if (c > k) k = c;
    }
    *kappa = (double)k;
    ws_free(&w);
    return ORC_OK;
}

/* ------------------------------------------------------------------------
 * Several species ("the spin unpolarized case"): particles
 * [0, counts[0]) are species 0, the next counts[1] species 1, ...  Exchange acts
 * within a species only, so V_xi = sum_s V_xi^{[range s]} (each by Eq. 6 on that
 * species' particles alone); the trap and the pair potential act on all
 * particles (Eq. 4, 18).  vb = sum over species, sign = product.
 * ---------------------------------------------------------------------- */
static double *sub_config(const double *x, int N, int P, int d, int l0, int n)
{
    double *xs = (double *)malloc(sizeof(double) * (size_t)n * P * d);
    if (!xs) return NULL;
    for (int j = 0; j < P; ++j)
        for (int l = 0; l < n; ++l)
            for (int c = 0; c < d; ++c) xs[(((size_t)j * n) + l) * d + c] = x[IDX(j, l0 + l, c)];
    return xs;
}

int orc_forces_species(const double *x, int N, int P, int d, double beta, double omega, double g, double s, double xi,
                       int nspecies, const int *counts, double *F, double *vb, int *sign)
{
    int l0 = 0, sg = 1;
    long double v = 0.0L;
    memset(F, 0, sizeof(double) * (size_t)N * P * d);
    for (int sp = 0; sp < nspecies; ++sp) {
        const int n = counts[sp];
        double *xs = sub_config(x, N, P, d, l0, n);
        double *Fs = (double *)malloc(sizeof(double) * (size_t)n * P * d);
        if (!xs || !Fs) { free(xs); free(Fs); return ORC_ENOMEM; }
        double vs;
        int ss;
        int rc = orc_forces(xs, n, P, d, beta, omega, g, s, xi, 0, Fs, &vs, &ss);
        if (!rc)
            for (int j = 0; j < P; ++j)
                for (int l = 0; l < n; ++l)
                    for (int c = 0; c < d; ++c) F[IDX(j, l0 + l, c)] = Fs[(((size_t)j * n) + l) * d + c];
        free(xs);
        free(Fs);
        if (rc) return rc;
        v += vs;
        sg *= ss;
        l0 += n;
    }
    if (l0 != N) return ORC_EINVAL;
    int rc = orc_external_forces(x, N, P, d, omega, g, s, F, NULL, NULL);
    if (vb) *vb = (double)v;
    if (sign) *sign = sg;
    return rc;
}

/* estimators with species: eps = d(beta V_xi)/d beta adds over species; the bead sums run over all particles.
 * orc_estimators(x) = P d N/(2 beta) + eps + Ubar, so eps_s = orc_estimators(species s alone, omega = g = 0) - P d n_s/(2 beta). */
int orc_estimators_species(const double *x, int N, int P, int d, double beta, double omega, double g, double s, double xi,
                           int nspecies, const int *counts, double *e_prim, double *e_vir, double *hist, int nbins, double rmax)
{
    int l0 = 0;
    long double eps = 0.0L;
    for (int sp = 0; sp < nspecies; ++sp) {
        const int n = counts[sp];
        double *xs = sub_config(x, N, P, d, l0, n);
        if (!xs) return ORC_ENOMEM;
        double ep, ev;
        int rc = orc_estimators(xs, n, P, d, beta, 0.0, 0.0, s, xi, &ep, &ev, NULL, 0, 1.0);
        free(xs);
        if (rc) return rc;
        eps += (long double)ep - (long double)P * d * n / (2.0L * beta);
        l0 += n;
    }
    if (l0 != N) return ORC_EINVAL;
    /* the bead sums (Ubar, virial, histogram) of all particles: xi = 0 makes the exchange part of this call trivial and its
     * eps (distinguishable rings) is taken out again */
    double ep0, ev0, epd, evd;
    int rc = orc_estimators(x, N, P, d, beta, omega, g, s, 0.0, &ep0, &ev0, hist, nbins, rmax);
    if (!rc) rc = orc_estimators(x, N, P, d, beta, 0.0, 0.0, s, 0.0, &epd, &evd, NULL, 0, 1.0);
    if (rc) return rc;
    *e_prim = (double)((long double)ep0 - (long double)epd + (long double)P * d * N / (2.0L * beta) + eps);
    *e_vir = ev0;
    return ORC_OK;
}

/* Pair-distance histogram (pair-correlation estimator): counts of |r_l^j - r_i^j|, i < l, over all bead indices j
 * (the pairs Eq. 18, couples) in nbins equal bins on [0, rmax); raw counts. */
int orc_pair_histogram(const double *x, int N, int P, int d, double *hist, int nbins, double rmax)
{
    for (int b = 0; b < nbins; ++b) hist[b] = 0.0;
    for (int j = 0; j < P; ++j)
        for (int l = 0; l < N; ++l)
            for (int i = 0; i < l; ++i) {
                const double r = sqrt(sqdist(&x[IDX(j, l, 0)], &x[IDX(j, i, 0)], d));
                if (r < rmax) {
                    int b = (int)(r / rmax * nbins);
                    if (b >= nbins) b = nbins - 1;
                    hist[b] += 1.0;
                }
            }
    return ORC_OK;
}

/* ------------------------------------------------------------------------
 * The same definitions with O(N) memory, for sizes whose N x N matrices do not
 * fit (N = 4e4: 25.6 GB as long double): E^{[u,v]} is regenerated from Eq. 7's
 * shared partial sums whenever Eq. 6 / Eq. 11 / Eq. 12 ask for it, nothing else
 * changes.  For fixed v the walk u = v..1 is the one of orc_cycle_energies; for
 * fixed u the walk v = u..N adds the same terms in the opposite order.
 * ---------------------------------------------------------------------- */
static void energies_to_v(const double *x, int N, int P, int d, double ks, const double *Eint, int v, long double *col)
{
    long double chain = 0.0L; /* col[u] = E^{[u+1,v+1]} (0-based u <= v) */
    for (int u = v; u >= 0; --u) {
        chain += (long double)Eint[u];
        if (u < v) chain += (long double)closing(x, N, P, d, ks, u, u + 1);
        col[u] = chain + (long double)closing(x, N, P, d, ks, v, u);
    }
}

static void energies_from_u(const double *x, int N, int P, int d, double ks, const double *Eint, int u, long double *row)
{
    long double chain = 0.0L; /* row[v] = E^{[u+1,v+1]} (0-based v >= u) */
    for (int v = u; v < N; ++v) {
        chain += (long double)Eint[v];
        if (v > u) chain += (long double)closing(x, N, P, d, ks, v - 1, v);
        row[v] = chain + (long double)closing(x, N, P, d, ks, v, u);
    }
}

/* Eq. 6 and Eq. 11 with regenerated energies: L[0..N], sgL, M[1..N+1] (M[0] unused), sgM; arrays of N+2. */
int orc_stream_tables(const double *x, int N, int P, int d, double beta, double xi, long double *L, int *sgL,
                      long double *M, int *sgM)
{
    if (N < 1 || P < 2 || d < 1 || !(beta > 0)) return ORC_EINVAL;
    const double ks = (double)P / (beta * beta);
    const long double lam = (xi != 0.0) ? logl(fabsl((long double)xi)) : 0.0L;
    const int sx = xi < 0 ? -1 : 1;
    double *Eint = (double *)malloc(sizeof(double) * (size_t)N);
    long double *e = (long double *)malloc(sizeof(long double) * (size_t)N);
    long double *t = (long double *)malloc(sizeof(long double) * (size_t)N);
    int *s = (int *)malloc(sizeof(int) * (size_t)N);
    if (!Eint || !e || !t || !s) { free(Eint); free(e); free(t); free(s); return ORC_ENOMEM; }
    orc_eint(x, N, P, d, beta, Eint);
    int rc = ORC_OK;
    L[0] = 0.0L;
    sgL[0] = 1;
    for (int n = 1; n <= N && rc == ORC_OK; ++n) { /* Eq. 6 */
        energies_to_v(x, N, P, d, ks, Eint, n - 1, e);
        int cnt = 0;
        for (int k = 1; k <= n; ++k) {
            if (xi == 0.0 && k > 1) break;
            const int u = n - k + 1;
            t[cnt] = (long double)(k - 1) * lam - (long double)beta * e[u - 1] + L[n - k];
            s[cnt] = (((k - 1) & 1) ? sx : 1) * sgL[n - k];
            ++cnt;
        }
        long double lse;
        int sgn;
        rc = signed_lse(t, s, cnt, &lse, &sgn);
        if (rc == ORC_OK) { L[n] = -logl((long double)n) + lse; sgL[n] = sgn; }
    }
    M[0] = 0.0L; sgM[0] = 1;
    M[N + 1] = 0.0L; sgM[N + 1] = 1;
    for (int u = N; u >= 1 && rc == ORC_OK; --u) { /* Eq. 11 */
        energies_from_u(x, N, P, d, ks, Eint, u - 1, e);
        int cnt = 0;
        for (int l = u; l <= N; ++l) {
            if (xi == 0.0 && l > u) break;
            t[cnt] = (long double)(l - u) * lam - logl((long double)l) - (long double)beta * e[l - 1] + M[l + 1];
            s[cnt] = (((l - u) & 1) ? sx : 1) * sgM[l + 1];
            ++cnt;
        }
        long double lse;
        int sgn;
        rc = signed_lse(t, s, cnt, &lse, &sgn);
        if (rc == ORC_OK) { M[u] = lse; sgM[u] = sgn; }
    }
    free(Eint); free(e); free(t); free(s);
    return rc;
}

/* Total force F = -grad(V_xi + U/P) on every bead of the nl selected particles ls[] (0-based), Fsel[k][j][c], from
 * Eq. 12-17 with regenerated energies; also V_B, its sign and (if not NULL) the tables V^{[1,n]}, n = 0..N, and
 * V^{[u,N]}, u = 1..N+1 (index u; N+2 entries). */
int orc_stream_forces_on(const double *x, int N, int P, int d, double beta, double omega, double g, double s, double xi,
                         const int *ls, int nl, double *Fsel, double *vb, int *sign, double *vfwd, double *vbwd)
{
    if (N < 1 || P < 2 || d < 1 || d > 3 || !(beta > 0) || !(s > 0)) return ORC_EINVAL;
    const double ks = (double)P / (beta * beta);
    const long double lam = (xi != 0.0) ? logl(fabsl((long double)xi)) : 0.0L;
    const int sx = xi < 0 ? -1 : 1;
    long double *L = (long double *)malloc(sizeof(long double) * (size_t)(N + 2));
    long double *M = (long double *)malloc(sizeof(long double) * (size_t)(N + 2));
    int *sgL = (int *)malloc(sizeof(int) * (size_t)(N + 2)), *sgM = (int *)malloc(sizeof(int) * (size_t)(N + 2));
    double *Eint = (double *)malloc(sizeof(double) * (size_t)N);
    long double *e = (long double *)malloc(sizeof(long double) * (size_t)N);
    double *pr = (double *)malloc(sizeof(double) * (size_t)N);
    int rc = (!L || !M || !sgL || !sgM || !Eint || !e || !pr) ? ORC_ENOMEM : ORC_OK;
    if (!rc) rc = orc_stream_tables(x, N, P, d, beta, xi, L, sgL, M, sgM);
    if (!rc) {
        orc_eint(x, N, P, d, beta, Eint);
        if (vb) *vb = (double)(-L[N] / (long double)beta);
        if (sign) *sign = sgL[N];
        if (vfwd) for (int n = 0; n <= N; ++n) vfwd[n] = (double)(-L[n] / (long double)beta);
        if (vbwd) { vbwd[0] = 0.0; for (int u = 1; u <= N + 1; ++u) vbwd[u] = (double)(-M[u] / (long double)beta); }
    }
    for (int k = 0; k < nl && !rc; ++k) {
        const int l = ls[k] + 1; /* 1-based, as in the paper */
        double *F = Fsel + (size_t)k * P * d;
        memset(F, 0, sizeof(double) * (size_t)P * d);
        for (int j = 1; j + 1 < P; ++j) /* Eq. 17 */
            for (int c = 0; c < d; ++c)
                F[j * d + c] = -ks * (2.0 * x[IDX(j, l - 1, c)] - x[IDX(j + 1, l - 1, c)] - x[IDX(j - 1, l - 1, c)]);
        /* Eq. 16: bead P of l, weights Pr[G(l) = lp] -- Eq. 12 for lp <= l (energies E^{[lp,l]}), Eq. 13 for lp = l+1 */
        energies_to_v(x, N, P, d, ks, Eint, l - 1, e);
        for (int lp = 1; lp <= N; ++lp) {
            double p = 0.0;
            if (lp <= l) {
                if (!(xi == 0.0 && lp < l)) {
                    long double ex = (long double)(l - lp) * lam - logl((long double)l) + L[lp - 1] - (long double)beta * e[lp - 1] + M[l + 1] - L[N];
                    p = (double)((((l - lp) & 1) ? sx : 1) * sgL[lp - 1] * sgM[l + 1] * sgL[N]) * exp((double)ex);
                }
            } else if (lp == l + 1) {
                p = 1.0 - (double)(sgL[l] * sgM[l + 1] * sgL[N]) * exp((double)(L[l] + M[l + 1] - L[N]));
            }
            pr[lp - 1] = p;
        }
        for (int c = 0; c < d; ++c) {
            long double fP = 0.0L;
            for (int lp = 0; lp < N; ++lp)
                fP -= (long double)pr[lp] * ks * (2.0 * x[IDX(P - 1, l - 1, c)] - x[IDX(P - 2, l - 1, c)] - x[IDX(0, lp, c)]);
            F[(P - 1) * d + c] += (double)fP;
        }
        /* Eq. 15: bead 1 of l, weights Pr[G(lp) = l] -- Eq. 12 for lp >= l (energies E^{[l,lp]}), Eq. 13 for lp = l-1 */
        energies_from_u(x, N, P, d, ks, Eint, l - 1, e);
        for (int lp = 1; lp <= N; ++lp) {
            double p = 0.0;
            if (lp >= l) {
                if (!(xi == 0.0 && lp > l)) {
                    long double ex = (long double)(lp - l) * lam - logl((long double)lp) + L[l - 1] - (long double)beta * e[lp - 1] + M[lp + 1] - L[N];
                    p = (double)((((lp - l) & 1) ? sx : 1) * sgL[l - 1] * sgM[lp + 1] * sgL[N]) * exp((double)ex);
                }
            } else if (lp == l - 1) {
                p = 1.0 - (double)(sgL[lp] * sgM[lp + 1] * sgL[N]) * exp((double)(L[lp] + M[lp + 1] - L[N]));
            }
            pr[lp - 1] = p;
        }
        for (int c = 0; c < d; ++c) {
            long double f1 = 0.0L;
            for (int lp = 0; lp < N; ++lp)
                f1 -= (long double)pr[lp] * ks * (2.0 * x[IDX(0, l - 1, c)] - x[IDX(1, l - 1, c)] - x[IDX(P - 1, lp, c)]);
            F[c] += (double)f1;
        }
        for (int j = 0; j < P; ++j) { /* -(1/P) grad U */
            double fe[3];
            orc_external_force_on(x, N, P, d, omega, g, s, j, l - 1, fe);
            for (int c = 0; c < d; ++c) F[j * d + c] += fe[c];
        }
    }
    free(L); free(M); free(sgL); free(sgM); free(Eint); free(e); free(pr);
    return rc;
}
