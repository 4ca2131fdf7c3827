/*
 * qarray_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, single-threaded, obviously-correct CPU implementation (C11, fp64) of the per-pixel ground-state charge
 * search of the constant capacitance model, written from the paper (arXiv 2404.04994, /root/reference/PAPER.md; "Lnnn"
 * below is a PAPER.md line) and from the readings R1..R12 listed in DESIGN.md.  It defines correctness for the CUDA
 * path in paper_2404_04994_b200/csrc/ and shares NO code, header, table or helper with it.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * What it computes, per gate-voltage vector ("pixel"):
 *   1. N_c = C_gd V_g                                   Eq. (6) L90           (fixed fma order, reading R1)
 *   2. continuous minimum x: open x = N_c (L88-L92); closed Eq. (7) L102 / (D7) L660-L663; if any x_i < 0 the
 *      constrained convex QP of Eq. (8) L110-L119 (with the 1/2 restored) solved EXACTLY by a textbook primal
 *      active-set method and certified by its KKT conditions (reading R3)
 *   3. candidate set: default = all 2^n floor/ceil roundings (L127); thresholded = Eq. (9), closed doubling rule
 *      L141 (reading R5); brute force = {0..n_max}^n (L13); closed arrays keep sum N = N_hat (L127, L159)
 *   4. energy of every candidate FROM THE DEFINITION E(N) = 1/2 (N - N_c)^T M (N - N_c), M = c_dd^-1
 *      (Eq. (C1)/(C2) L607-L613, (H2) L748; equals Eq. (4) L45 + 1/2 N_c^T M N_c) -- O(n^2) per candidate, no Gray
 *      code, no incremental update, no blocking
 *   5. argmin (Eq. (5)), ties -> lexicographically smallest N (reading R6); also the second-best energy
 *   6. charge-sensor dots (L149, Eq. (3); reading R8)
 *   7. thermal broadening: the soft arg min of Eq. (10) L157 over the same candidate set (qo_thermal; reading R13)
 *   8. charge-sensor response profile, noise and gradient (qo_sensor_response; L149, L464; reading R14)
 *
 * Pins (tests/test_oracle_*.py): P0..P13 of DESIGN.md (P13: Eq. (10) -- Fermi function of a single dot, kT -> 0 and
 * kT -> infinity limits, Eq. (4)-energy numpy sums on tiny arrays, sum <N> = N_hat).  Functions with no pin independent of the oracle itself:
 *   - qo_sensor's potential values on random arrays                           : "parity unpinned" beyond the
 *     single-sensor closed form tested in tests/test_oracle_pins.py (rounding of s, V_s = [M (N - N_c)]_s)
 *   - thresholded-vs-default agreement RATE on config 5                       : parity unpinned (statistic only)
 *   - qo_sensor_response: the paper gives neither formula nor parameter for the response profile and the noise
 *     (L149), so WHICH profile / noise model is right is "parity unpinned"; what reading R14 fixes is pinned (profile
 *     closed forms, SplitMix64 test vector, moments / spectrum / jump statistics of the noise, numpy.gradient)
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fPIC -shared [-fopenmp]   (oracle/build.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define QO_MAXN 16
#define QO_MAXG 64

#define QO_ALG_DEFAULT 0
#define QO_ALG_THRESHOLDED 1
#define QO_ALG_BRUTE 2

#define QO_FLAG_QP 1        /* analytic minimum had a negative component; QP solved        */
#define QO_FLAG_WIDENED 2   /* never set: the widened set of an earlier reading R5 is unreachable (R5) */
#define QO_FLAG_QP_FAIL 4   /* KKT certificate not met / iteration cap (must never happen) */
#define QO_FLAG_EMPTY 8     /* no admissible candidate (closed brute force with n*n_max < N_hat) */

typedef struct {
    int n, g;
    double C[QO_MAXN * QO_MAXN];    /* c_dd, Maxwell format                       */
    double Cgd[QO_MAXN * QO_MAXG];  /* gate -> dot couplings, row-major [n][g]    */
    double M[QO_MAXN * QO_MAXN];    /* c_dd^-1                                    */
    double C1[QO_MAXN];             /* c_dd 1                                     */
    double oneC1;                   /* 1^T c_dd 1                                 */
    double EC;                      /* "charging energy" 1/2 min_i M_ii (|e| = 1) */
} qo_model;

/* ------------------------------------------------------------------------------------------------------------------ */
/* dense SPD helpers (Cholesky); k <= QO_MAXN                                                                          */

static int chol_factor(const double *A, int k, double *L)
{ /* A = L L^T, lower triangular L, row-major k x k; returns 0 or 1 if not positive definite */
    for (int i = 0; i < k; i++) {
        for (int j = 0; j <= i; j++) {
            double s = A[i * k + j];
            for (int q = 0; q < j; q++) s -= L[i * k + q] * L[j * k + q];
            if (i == j) {
                if (!(s > 0.0)) return 1;
                L[i * k + i] = sqrt(s);
            } else {
                L[i * k + j] = s / L[j * k + j];
            }
        }
        for (int j = i + 1; j < k; j++) L[i * k + j] = 0.0;
    }
    return 0;
}

static void chol_solve(const double *L, int k, const double *b, double *x)
{
    double y[QO_MAXN];
    for (int i = 0; i < k; i++) {
        double s = b[i];
        for (int q = 0; q < i; q++) s -= L[i * k + q] * y[q];
        y[i] = s / L[i * k + i];
    }
    for (int i = k - 1; i >= 0; i--) {
        double s = y[i];
        for (int q = i + 1; q < k; q++) s -= L[q * k + i] * x[q];
        x[i] = s / L[i * k + i];
    }
}

/* ------------------------------------------------------------------------------------------------------------------ */
/* model: validation (L204: shape, symmetric, positive definite) and M = c_dd^-1 (L41)                                 */

int qo_model_init(qo_model *m, const double *C_dd, const double *C_gd, int n, int g)
{
    if (!m || !C_dd || !C_gd || n < 1 || n > QO_MAXN || g < 1 || g > QO_MAXG) return 1;
    memset(m, 0, sizeof(*m));
    m->n = n;
    m->g = g;
    double amax = 0.0;
    for (int i = 0; i < n * n; i++) {
        if (!isfinite(C_dd[i])) return 1;
        if (fabs(C_dd[i]) > amax) amax = fabs(C_dd[i]);
    }
    for (int i = 0; i < n * g; i++)
        if (!isfinite(C_gd[i])) return 1;
    for (int i = 0; i < n; i++)
        for (int j = 0; j < i; j++)
            if (fabs(C_dd[i * n + j] - C_dd[j * n + i]) > 1e-12 * amax) return 2;
    memcpy(m->C, C_dd, sizeof(double) * n * n);
    memcpy(m->Cgd, C_gd, sizeof(double) * n * g);
    double L[QO_MAXN * QO_MAXN];
    if (chol_factor(m->C, n, L)) return 3;
    for (int j = 0; j < n; j++) { /* column j of the inverse */
        double e[QO_MAXN] = {0}, col[QO_MAXN];
        e[j] = 1.0;
        chol_solve(L, n, e, col);
        for (int i = 0; i < n; i++) m->M[i * n + j] = col[i];
    }
    /* c_dd 1 and 1^T c_dd 1 for Eq. (7): plain left-to-right sums (reading R1) */
    double tot = 0.0;
    for (int i = 0; i < n; i++) {
        double s = 0.0;
        for (int j = 0; j < n; j++) s = s + m->C[i * n + j];
        m->C1[i] = s;
        tot = tot + s;
    }
    m->oneC1 = tot;
    double mn = m->M[0];
    for (int i = 1; i < n; i++)
        if (m->M[i * n + i] < mn) mn = m->M[i * n + i];
    m->EC = 0.5 * mn;
    return 0;
}

/* N_c = C_gd V_g, Eq. (6) L90.  Reading R1: acc = 0; acc = fma(C_gd[i,k], V[k], acc), k ascending. */
void qo_nc(const qo_model *m, const double *Vg, double *Nc)
{
    for (int i = 0; i < m->n; i++) {
        double acc = 0.0;
        for (int k = 0; k < m->g; k++) acc = fma(m->Cgd[i * m->g + k], Vg[k], acc);
        Nc[i] = acc;
    }
}

/* E(N) = 1/2 (N - N_c)^T M (N - N_c), Eq. (C1)/(C2) L607-L613, straight from the definition. */
double qo_energy(const qo_model *m, const double *Nc, const int32_t *N)
{
    int n = m->n;
    double d[QO_MAXN];
    for (int i = 0; i < n; i++) d[i] = (double)N[i] - Nc[i];
    double E = 0.0;
    for (int i = 0; i < n; i++) {
        double row = 0.0;
        for (int j = 0; j < n; j++) row += m->M[i * n + j] * d[j];
        E += d[i] * row;
    }
    return 0.5 * E;
}

/* Eq. (4) L45 as printed: F = 1/2 Q^T M Q - (M C_gd V_g)^T Q  (constant terms dropped). Used by the pin tests only. */
double qo_free_energy_eq4(const qo_model *m, const double *Nc, const int32_t *N)
{
    int n = m->n;
    double quad = 0.0, lin = 0.0;
    for (int i = 0; i < n; i++) {
        double row = 0.0, mv = 0.0;
        for (int j = 0; j < n; j++) {
            row += m->M[i * n + j] * (double)N[j];
            mv += m->M[i * n + j] * Nc[j];
        }
        quad += (double)N[i] * row;
        lin += mv * (double)N[i];
    }
    return 0.5 * quad - lin;
}

/* ------------------------------------------------------------------------------------------------------------------ */
/* Exact QP (reading R3): minimise 1/2 (x - c)^T M (x - c)  s.t. x >= 0 [and 1^T x = N_hat]                            */
/* Textbook primal active-set method for a strictly convex QP (Nocedal & Wright, Numerical Optimization, Alg. 16.3):   */
/* working set W of active bounds; solve the equality-constrained QP on the free set; step until a bound blocks; when   */
/* the step is zero drop the bound with the most negative multiplier; stop when all multipliers are non-negative.      */

/* equality-constrained minimiser with x_W = 0: M_FF x_F = (M c)_F + lambda 1_F, closed: sum_F x_F = N_hat */
static int eqp_solve(const qo_model *m, const double *c, const int *W, int closed, double Nhat, double *xh, double *lambda)
{
    int n = m->n, F[QO_MAXN], k = 0;
    for (int i = 0; i < n; i++) {
        xh[i] = 0.0;
        if (!W[i]) F[k++] = i;
    }
    *lambda = 0.0;
    if (k == 0) return 0;
    double A[QO_MAXN * QO_MAXN], L[QO_MAXN * QO_MAXN], rhs[QO_MAXN], u[QO_MAXN], w[QO_MAXN], one[QO_MAXN];
    for (int a = 0; a < k; a++) {
        for (int b = 0; b < k; b++) A[a * k + b] = m->M[F[a] * n + F[b]];
        double s = 0.0;
        for (int j = 0; j < n; j++) s += m->M[F[a] * n + j] * c[j];
        rhs[a] = s;
        one[a] = 1.0;
    }
    if (chol_factor(A, k, L)) return 1;
    chol_solve(L, k, rhs, u);
    if (closed) {
        chol_solve(L, k, one, w);
        double su = 0.0, sw = 0.0;
        for (int a = 0; a < k; a++) {
            su += u[a];
            sw += w[a];
        }
        *lambda = (Nhat - su) / sw;
        for (int a = 0; a < k; a++) u[a] += *lambda * w[a];
        if (k == 1) u[0] = Nhat; /* reading R3: a single free dot carries the whole charge, exactly (1^T x = N_hat) */
    }
    for (int a = 0; a < k; a++) xh[F[a]] = u[a];
    return 0;
}

/* returns number of active-set iterations (>= 1), or -1 on failure; *kkt = largest KKT violation (scaled) */
int qo_qp(const qo_model *m, const double *c, int closed, double Nhat, double *x, double *kkt)
{
    int n = m->n, W[QO_MAXN];
    double xh[QO_MAXN], lambda = 0.0;
    double scale = 1.0;
    for (int i = 0; i < n; i++)
        if (fabs(c[i]) > scale) scale = fabs(c[i]);
    if (closed && fabs(Nhat) > scale) scale = fabs(Nhat);
    *kkt = 0.0;
    if (closed && Nhat <= 0.0) { /* only feasible point */
        for (int i = 0; i < n; i++) x[i] = 0.0;
        return (Nhat == 0.0) ? 1 : -1;
    }
    for (int i = 0; i < n; i++) { /* feasible start */
        if (closed) {
            x[i] = Nhat / (double)n;
            W[i] = 0;
        } else {
            x[i] = c[i] > 0.0 ? c[i] : 0.0;
            W[i] = !(c[i] > 0.0);
        }
    }
    const double tol = 1e-13 * scale;
    int it, done = 0;
    for (it = 1; it <= 50 * n + 50; it++) {
        if (eqp_solve(m, c, W, closed, Nhat, xh, &lambda)) return -1;
        double pmax = 0.0;
        for (int i = 0; i < n; i++)
            if (fabs(xh[i] - x[i]) > pmax) pmax = fabs(xh[i] - x[i]);
        if (pmax <= tol) {
            for (int i = 0; i < n; i++) x[i] = xh[i]; /* x is now exactly the EQP solution, x_W = 0 */
            int worst = -1;
            double rmin = -1e-12 * scale;
            for (int i = 0; i < n; i++) {
                if (!W[i]) continue;
                double r = -lambda;
                for (int j = 0; j < n; j++) r += m->M[i * n + j] * (x[j] - c[j]);
                if (r < rmin) {
                    rmin = r;
                    worst = i;
                }
            }
            if (worst < 0) {
                done = 1;
                break;
            }
            W[worst] = 0;
            continue;
        }
        double alpha = 1.0;
        int block = -1;
        for (int i = 0; i < n; i++) {
            if (W[i]) continue;
            double p = xh[i] - x[i];
            if (p < 0.0) {
                double a = x[i] / (-p);
                if (a < alpha) {
                    alpha = a;
                    block = i;
                }
            }
        }
        if (block < 0) {
            for (int i = 0; i < n; i++) x[i] = xh[i];
        } else {
            for (int i = 0; i < n; i++)
                if (!W[i]) x[i] += alpha * (xh[i] - x[i]);
            x[block] = 0.0;
            W[block] = 1;
        }
    }
    /* KKT certificate: x >= 0, x_W = 0, r = M (x - c) - lambda 1, r_F = 0, r_W >= 0, closed: sum x = N_hat */
    double viol = 0.0, sum = 0.0;
    for (int i = 0; i < n; i++) {
        double r = -lambda;
        for (int j = 0; j < n; j++) r += m->M[i * n + j] * (x[j] - c[j]);
        sum += x[i];
        if (x[i] < 0.0 && -x[i] > viol) viol = -x[i];
        if (W[i]) {
            if (x[i] != 0.0 && fabs(x[i]) > viol) viol = fabs(x[i]);
            if (r < 0.0 && -r > viol) viol = -r;
        } else if (fabs(r) > viol) {
            viol = fabs(r);
        }
    }
    if (closed && fabs(sum - Nhat) > viol) viol = fabs(sum - Nhat);
    *kkt = viol / scale;
    if (!done || *kkt > 1e-9) return -1;
    return it;
}

/* continuous minimum (step 2).  returns flags (QO_FLAG_QP, QO_FLAG_QP_FAIL) */
int qo_continuous_min(const qo_model *m, const double *Nc, int closed, int N_hat, double *x)
{
    int n = m->n, neg = 0;
    if (!closed) {
        for (int i = 0; i < n; i++) x[i] = Nc[i]; /* Eq. (6) */
    } else {                                      /* Eq. (7), reading R1 for the order */
        double s = 0.0;
        for (int i = 0; i < n; i++) s = s + Nc[i];
        double lam = ((double)N_hat - s) / m->oneC1;
        for (int i = 0; i < n; i++) x[i] = fma(lam, m->C1[i], Nc[i]);
    }
    for (int i = 0; i < n; i++)
        if (x[i] < 0.0) neg = 1;
    if (!neg) return 0; /* L82: accept the analytic solution */
    double kkt;
    int it = qo_qp(m, Nc, closed, (double)N_hat, x, &kkt); /* L106 */
    return QO_FLAG_QP | (it < 0 ? QO_FLAG_QP_FAIL : 0);
}

/* ------------------------------------------------------------------------------------------------------------------ */
/* candidate ranges (step 3): dot i may take base[i] .. base[i] + cnt[i] - 1                                            */

static void ranges_floor_ceil(int n, const double *x, double t, int thresholded, int32_t *base, int32_t *cnt)
{
    for (int i = 0; i < n; i++) {
        double fl = floor(x[i]);
        double frac = x[i] - fl;
        int32_t lo = fl > 0.0 ? (int32_t)fl : 0; /* lo = max(0, floor x), reading R4 */
        if (!thresholded || fabs(frac - 0.5) <= t * 0.5) { /* Eq. (9), "<=" as printed (R10) */
            base[i] = lo;
            cnt[i] = 2; /* lo and lo + 1: always two distinct values (R4) */
        } else {
            base[i] = frac < 0.5 ? lo : lo + 1; /* L133: round to the closest */
            cnt[i] = 1;
        }
    }
}

static int closed_nonempty(int n, const int32_t *base, const int32_t *cnt, int N_hat)
{
    int64_t smin = 0, smax = 0;
    for (int i = 0; i < n; i++) {
        smin += base[i];
        smax += base[i] + cnt[i] - 1;
    }
    return smin <= N_hat && N_hat <= smax; /* contiguous ranges: every total in [smin, smax] is reachable */
}

typedef struct {
    int32_t N[QO_MAXN];
    double E, E2;
    int64_t n_scored, n_enum;
} qo_best;

/* steps 4-5: lexicographic enumeration (dot 0 slowest), energy from the definition, strict '<' keeps the first
 * (= lexicographically smallest) among bitwise-equal energies (R6). */
static void enumerate_argmin(const qo_model *m, const double *Nc, const int32_t *base, const int32_t *cnt, int closed,
                             int N_hat, qo_best *out)
{
    int n = m->n;
    int32_t N[QO_MAXN];
    for (int i = 0; i < n; i++) N[i] = base[i];
    out->E = INFINITY;
    out->E2 = INFINITY;
    out->n_scored = 0;
    out->n_enum = 0;
    for (int i = 0; i < n; i++) out->N[i] = -1;
    for (;;) {
        out->n_enum++;
        int ok = 1;
        if (closed) {
            int64_t s = 0;
            for (int i = 0; i < n; i++) s += N[i];
            ok = (s == N_hat);
        }
        if (ok) {
            double e = qo_energy(m, Nc, N);
            out->n_scored++;
            if (e < out->E) {
                out->E2 = out->E;
                out->E = e;
                for (int i = 0; i < n; i++) out->N[i] = N[i];
            } else if (e < out->E2) {
                out->E2 = e;
            }
        }
        int i = n - 1;
        while (i >= 0) {
            if (N[i] < base[i] + cnt[i] - 1) {
                N[i]++;
                break;
            }
            N[i] = base[i];
            i--;
        }
        if (i < 0) break;
    }
}

/* one pixel, all steps.  returns flags. */
int qo_pixel(const qo_model *m, const double *Vg, int closed, int N_hat, int alg, double t, int n_max, int32_t *N,
             double *E, double *E2, double *xcont, int64_t *n_scored, int64_t *n_enum, int32_t *n_doublings)
{
    int n = m->n, flags = 0, doublings = 0;
    double Nc[QO_MAXN], x[QO_MAXN];
    int32_t base[QO_MAXN], cnt[QO_MAXN];
    qo_nc(m, Vg, Nc);
    flags |= qo_continuous_min(m, Nc, closed, N_hat, x);
    if (alg == QO_ALG_BRUTE) {
        for (int i = 0; i < n; i++) {
            base[i] = 0;
            cnt[i] = n_max + 1;
        }
    } else {
        double tt = (alg == QO_ALG_THRESHOLDED) ? t : 1.0;
        ranges_floor_ceil(n, x, tt, alg == QO_ALG_THRESHOLDED, base, cnt);
        if (closed) {
            /* L141 + reading R5: per pixel, t <- min(1, 2t) (t = 0 -> 1) until the kept set is non-empty */
            while (alg == QO_ALG_THRESHOLDED && !closed_nonempty(n, base, cnt, N_hat) && tt < 1.0) {
                tt = (tt > 0.0) ? fmin(1.0, 2.0 * tt) : 1.0;
                doublings++;
                ranges_floor_ceil(n, x, tt, 1, base, cnt);
            }
            /* At t = 1 the kept set is the closed default set, which is never empty for a feasible x (x >= 0,
             * |sum x - N_hat| << 1): sum lo <= sum x and sum (lo + 1) > sum x, so 0 <= N_hat - sum lo <= n
             * (reading R5).  Should it ever be empty the pixel is reported as QO_FLAG_EMPTY below. */
        }
    }
    qo_best b;
    enumerate_argmin(m, Nc, base, cnt, closed, N_hat, &b);
    if (b.n_scored == 0) flags |= QO_FLAG_EMPTY;
    for (int i = 0; i < n; i++) N[i] = b.N[i];
    *E = b.E;
    if (E2) *E2 = b.E2;
    if (xcont)
        for (int i = 0; i < n; i++) xcont[i] = x[i];
    if (n_scored) *n_scored = b.n_scored;
    if (n_enum) *n_enum = b.n_enum;
    if (n_doublings) *n_doublings = doublings;
    return flags;
}

/* ------------------------------------------------------------------------------------------------------------------ */
/* Thermal broadening (section IV.B, Eq. (10)): the arg min of Eq. (5) is replaced by the Boltzmann-weighted   */
/* mean over the SAME candidate set (steps 1-3 above; closed: only sum N = N_hat, L159):                                 */
/*     <N> = sum_N N exp(-F(N)/kT) / sum_N exp(-F(N)/kT)                                                                 */
/* kT > 0 is k_B T in the energy units of E (|e| = 1, R11).  Eq. (4) and the completed square E differ by a per-pixel    */
/* constant, which cancels in the ratio; the weights are formed as exp(-(E - E_min)/kT) (E_min = smallest energy of the  */
/* set) so that the largest weight is exactly 1.  Two plain passes in lexicographic order, energy from the definition.  */
/* Nmean[n] (all -1 if the set is empty), *Emin.  returns flags.                                                         */
int qo_pixel_thermal(const qo_model *m, const double *Vg, int closed, int N_hat, int alg, double t, int n_max, double kT,
                     double *Nmean, double *Emin, int64_t *n_scored)
{
    int n = m->n;
    int32_t Nbest[QO_MAXN];
    double E, E2, x[QO_MAXN];
    int64_t ns = 0, ne = 0;
    int32_t dbl = 0;
    /* steps 1-3 and E_min: exactly the ground-state search (its candidate ranges are recomputed below the same way) */
    int flags = qo_pixel(m, Vg, closed, N_hat, alg, t, n_max, Nbest, &E, &E2, x, &ns, &ne, &dbl);
    if (n_scored) *n_scored = ns;
    *Emin = E;
    if (ns == 0) {
        for (int i = 0; i < n; i++) Nmean[i] = -1.0;
        return flags;
    }
    double Nc[QO_MAXN];
    int32_t base[QO_MAXN], cnt[QO_MAXN];
    qo_nc(m, Vg, Nc);
    if (alg == QO_ALG_BRUTE) {
        for (int i = 0; i < n; i++) {
            base[i] = 0;
            cnt[i] = n_max + 1;
        }
    } else {
        double tt = (alg == QO_ALG_THRESHOLDED) ? t : 1.0;
        ranges_floor_ceil(n, x, tt, alg == QO_ALG_THRESHOLDED, base, cnt);
        if (closed) {
            while (alg == QO_ALG_THRESHOLDED && !closed_nonempty(n, base, cnt, N_hat) && tt < 1.0) {
                tt = (tt > 0.0) ? fmin(1.0, 2.0 * tt) : 1.0;
                ranges_floor_ceil(n, x, tt, 1, base, cnt);
            }
        }
    }
    double Z = 0.0, S[QO_MAXN];
    int32_t N[QO_MAXN];
    for (int i = 0; i < n; i++) {
        S[i] = 0.0;
        N[i] = base[i];
    }
    for (;;) {
        int ok = 1;
        if (closed) {
            int64_t s = 0;
            for (int i = 0; i < n; i++) s += N[i];
            ok = (s == N_hat);
        }
        if (ok) {
            double w = exp(-(qo_energy(m, Nc, N) - E) / kT);
            Z += w;
            for (int i = 0; i < n; i++) S[i] += w * (double)N[i];
        }
        int i = n - 1;
        while (i >= 0) {
            if (N[i] < base[i] + cnt[i] - 1) {
                N[i]++;
                break;
            }
            N[i] = base[i];
            i--;
        }
        if (i < 0) break;
    }
    for (int i = 0; i < n; i++) Nmean[i] = S[i] / Z;
    return flags;
}

int qo_thermal(const qo_model *m, const double *Vg, int64_t P, int closed, int N_hat, int alg, double t, int n_max,
               double kT, double *Nmean, double *Emin, int64_t *n_scored, int32_t *flags)
{
    if (!m || !Vg || !Nmean || !Emin || P < 0 || !(kT > 0.0)) return 1;
    if (alg < 0 || alg > 2) return 1;
    if (alg == QO_ALG_THRESHOLDED && !(t >= 0.0 && t <= 1.0)) return 1;
    if (alg == QO_ALG_BRUTE && n_max < 0) return 1;
    if (closed && N_hat < 0) return 1;
    int n = m->n, g = m->g;
    for (int64_t p = 0; p < P; p++) {
        int f = qo_pixel_thermal(m, Vg + p * g, closed, N_hat, alg, t, n_max, kT, Nmean + p * n, Emin + p,
                                 n_scored ? n_scored + p : 0);
        if (flags) flags[p] = f;
    }
    return 0;
}

/* whole sweep: Vg[P][g] -> N[P][n], E[P], optional E2[P], xcont[P][n], n_scored[P], n_enum[P], flags[P], doublings[P].
 * n_threads <= 1: single thread (the oracle proper).  n_threads > 1: the same function under an OpenMP parallel-for
 * over pixels (only when built with -fopenmp; used for the all-cores CPU baseline in bench.py). */
int qo_ground_state(const qo_model *m, const double *Vg, int64_t P, int closed, int N_hat, int alg, double t, int n_max,
                    int32_t *N, double *E, double *E2, double *xcont, int64_t *n_scored, int64_t *n_enum,
                    int32_t *flags, int32_t *n_doublings, int n_threads)
{
    if (!m || !Vg || !N || !E || P < 0) return 1;
    if (alg < 0 || alg > 2) return 1;
    if (alg == QO_ALG_THRESHOLDED && !(t >= 0.0 && t <= 1.0)) return 1;
    if (alg == QO_ALG_BRUTE && n_max < 0) return 1;
    if (closed && N_hat < 0) return 1;
    int n = m->n, g = m->g;
    (void)n_threads;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 8) num_threads(n_threads > 1 ? n_threads : 1)
#endif
    for (int64_t p = 0; p < P; p++) {
        int f = qo_pixel(m, Vg + p * g, closed, N_hat, alg, t, n_max, N + p * n, E + p, E2 ? E2 + p : 0,
                         xcont ? xcont + p * n : 0, n_scored ? n_scored + p : 0, n_enum ? n_enum + p : 0,
                         n_doublings ? n_doublings + p : 0);
        if (flags) flags[p] = f;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------------ */
/* Charge sensors (L149, Eq. (3)), reading R8.                                                                     */
/* full: the full model (array dots + sensor dots).  sub: the model built from the sub-blocks C[D,D], C_gd[D,:] of the */
/* full Maxwell matrices, D = non-sensor dots in ascending order.  For each pixel:                                     */
/*   a. N_D = ground state of `sub` (all the steps above)                                                              */
/*   b. with N_D fixed, each sensor s independently (the other sensors at their continuous value, d = 0):              */
/*        y = sum_{j in D} M_sj (N_j - N_c,j);  s* = N_c,s - y / M_ss;  c0 = max(0, floor s*);                          */
/*        e(c) = (c - N_c,s) y + 1/2 M_ss (c - N_c,s)^2;   N_s = c0 + 1 if e(c0 + 1) < e(c0) else c0                   */
/*   c. V_s = [M (N - N_c)]_s over the full model with every N_s set  (Eq. (3) with the positive-C_gd convention)      */
/* sgap (optional) returns |e(c0 + 1) - e(c0)| per sensor: the margin of step b's two-way choice, so that the parity   */
/* tests can apply the near-tie rule (margin < 1e-9 E_C) to the sensor columns as they do to the array columns.        */
int qo_sensor(const qo_model *full, const qo_model *sub, const int32_t *sensor_idx, int ns, const double *Vg, int64_t P,
              int closed, int N_hat, int alg, double t, int n_max, int32_t *N /* [P][n_full] */, double *E /* [P] */,
              double *E2, double *Vs /* [P][ns] */, double *sgap /* [P][ns] |e(c0+1) - e(c0)| or NULL */, int32_t *flags)
{
    int n = full->n, g = full->g;
    if (sub->n != n - ns || sub->g != g || ns < 1 || ns >= n) return 1;
    int is_s[QO_MAXN] = {0}, D[QO_MAXN], nd = 0;
    for (int a = 0; a < ns; a++) {
        if (sensor_idx[a] < 0 || sensor_idx[a] >= n || is_s[sensor_idx[a]]) return 1;
        is_s[sensor_idx[a]] = 1;
    }
    for (int i = 0; i < n; i++)
        if (!is_s[i]) D[nd++] = i;
    for (int64_t p = 0; p < P; p++) {
        int32_t ND[QO_MAXN];
        double e, e2;
        int f = qo_pixel(sub, Vg + p * g, closed, N_hat, alg, t, n_max, ND, &e, &e2, 0, 0, 0, 0);
        E[p] = e;
        if (E2) E2[p] = e2;
        if (flags) flags[p] = f;
        double Nc[QO_MAXN], d[QO_MAXN];
        qo_nc(full, Vg + p * g, Nc);
        int32_t *Np = N + p * n;
        for (int i = 0; i < n; i++) d[i] = 0.0;
        for (int a = 0; a < nd; a++) {
            Np[D[a]] = ND[a];
            d[D[a]] = (double)ND[a] - Nc[D[a]];
        }
        for (int a = 0; a < ns; a++) {
            int s = sensor_idx[a];
            double y = 0.0;
            for (int b = 0; b < nd; b++) y += full->M[s * n + D[b]] * d[D[b]];
            double Mss = full->M[s * n + s];
            double sstar = Nc[s] - y / Mss;
            double fl = floor(sstar);
            int32_t c0 = fl > 0.0 ? (int32_t)fl : 0;
            double d0 = (double)c0 - Nc[s], d1 = (double)(c0 + 1) - Nc[s];
            double e0 = d0 * y + 0.5 * Mss * d0 * d0;
            double e1 = d1 * y + 0.5 * Mss * d1 * d1;
            Np[s] = (e1 < e0) ? c0 + 1 : c0;
            if (sgap) sgap[p * ns + a] = fabs(e1 - e0); /* the two-way choice's margin (near-tie rule of the parity tests) */
        }
        for (int a = 0; a < ns; a++) d[sensor_idx[a]] = (double)Np[sensor_idx[a]] - Nc[sensor_idx[a]];
        for (int a = 0; a < ns; a++) {
            int s = sensor_idx[a];
            double v = 0.0;
            for (int j = 0; j < n; j++) v += full->M[s * n + j] * d[j];
            Vs[p * ns + a] = v;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------------ */
/* 8. charge-sensor RESPONSE and noise (L149 last two sentences; reading R14 of DESIGN.md).        */
/* The paper names the ingredients but prints no formula or parameter ("Lorentzian or an approximately Gaussian        */
/* profile in the weak and strong coupling regimes"; "white, 1/f, and sensor jump noise can be added on top"; Fig. 3   */
/* L464 plots the derivative of the sensor signal along the swept gate and, for a qpc, "replaced the Lorentzian shape  */
/* response with a linear function").  Reading R14 fixes every choice; all parameters are the caller's.                */
/*   profile 0 Lorentzian  S = A / (1 + ((V_s - v0)/w)^2)          w = half width at half maximum                       */
/*   profile 1 Gaussian    S = A exp(-(V_s - v0)^2 / (2 w^2))      w = standard deviation                               */
/*   profile 2 linear      S = A (V_s - v0) / w                    (qpc, L464)                                          */
/* Noise is added to S in pixel order p = iy W + ix (the raster is the time axis):                                      */
/*   white   sigma_w z(0, p)                                                                                           */
/*   1/f     (sigma_p / sqrt K) sum_{j<K} z(1 + j, p >> j)    Voss-McCartney: source j is redrawn every 2^j pixels      */
/*   jumps   J(p) = sum_{q<=p} [u(62, q) < rate] sigma_j z(31, q)   the baseline keeps every shift (sequential sum)     */
/* Random numbers are counter based (so that any implementation draws the same ones in any order):                     */
/*   r(stream, idx) = mix(mix(seed + GOLDEN (stream + 1)) + GOLDEN (idx + 1)),  mix = the SplitMix64 finaliser          */
/*   u = ((r >> 11) + 0.5) 2^-53 in (0,1);  z(s, idx) = sqrt(-2 ln u(2s, idx)) cos(2 pi u(2s + 1, idx))  (Box-Muller)   */
/*   sensor a uses the streams 128 a + (...).                                                                          */
/* Gradient (optional): along the fast axis ix, central differences inside a row, one-sided at its two ends, in signal */
/* units per pixel; taken of the noisy signal.                                                                         */
typedef struct {
    int32_t profile;       /* 0 Lorentzian, 1 Gaussian, 2 linear */
    int32_t pink_octaves;  /* K, 0..30 */
    double v0, width, amplitude;
    double white_sigma, pink_sigma, jump_rate, jump_sigma;
    uint64_t seed;
} qo_sensor_params;

#define QO_GOLDEN 0x9E3779B97F4A7C15ull
static uint64_t qo_mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
uint64_t qo_rng_u64(uint64_t seed, uint64_t stream, uint64_t idx)
{
    return qo_mix64(qo_mix64(seed + QO_GOLDEN * (stream + 1)) + QO_GOLDEN * (idx + 1));
}
double qo_rng_uniform(uint64_t seed, uint64_t stream, uint64_t idx)
{
    return ((double)(qo_rng_u64(seed, stream, idx) >> 11) + 0.5) * 0x1.0p-53;
}
double qo_rng_normal(uint64_t seed, uint64_t stream, uint64_t idx)
{
    double u1 = qo_rng_uniform(seed, 2 * stream, idx), u2 = qo_rng_uniform(seed, 2 * stream + 1, idx);
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

double qo_sensor_profile(const qo_sensor_params *q, double vs)
{
    double x = (vs - q->v0) / q->width;
    if (q->profile == 0) return q->amplitude / (1.0 + x * x);
    if (q->profile == 1) return q->amplitude * exp(-0.5 * x * x);
    return q->amplitude * x;
}

int qo_sensor_response(const double *Vs /* [P][ns] */, int64_t P, int ns, int64_t W, const qo_sensor_params *prm /* [ns] */,
                       double *S /* [P][ns] */, double *G /* [P][ns] or NULL */)
{
    if (P < 0 || ns < 1 || W < 1 || (P % W) != 0) return 1;
    for (int a = 0; a < ns; a++) {
        const qo_sensor_params *q = prm + a;
        if (q->profile < 0 || q->profile > 2 || !(q->width > 0.0) || q->pink_octaves < 0 || q->pink_octaves > 30 ||
            q->white_sigma < 0.0 || q->pink_sigma < 0.0 || q->jump_sigma < 0.0 || !(q->jump_rate >= 0.0 && q->jump_rate <= 1.0))
            return 1;
        uint64_t st = 128ull * (uint64_t)a;
        double J = 0.0;
        for (int64_t p = 0; p < P; p++) {
            double s = qo_sensor_profile(q, Vs[p * ns + a]);
            if (q->white_sigma > 0.0) s += q->white_sigma * qo_rng_normal(q->seed, st + 0, (uint64_t)p);
            if (q->pink_sigma > 0.0 && q->pink_octaves > 0) {
                double acc = 0.0;
                for (int j = 0; j < q->pink_octaves; j++) acc += qo_rng_normal(q->seed, st + 1 + (uint64_t)j, (uint64_t)p >> j);
                s += q->pink_sigma / sqrt((double)q->pink_octaves) * acc;
            }
            if (q->jump_rate > 0.0 && q->jump_sigma > 0.0) {
                if (qo_rng_uniform(q->seed, 2 * (st + 62), (uint64_t)p) < q->jump_rate)
                    J += q->jump_sigma * qo_rng_normal(q->seed, st + 31, (uint64_t)p);
                s += J;
            }
            S[p * ns + a] = s;
        }
    }
    if (G) {
        int64_t H = P / W;
        for (int64_t iy = 0; iy < H; iy++)
            for (int64_t ix = 0; ix < W; ix++)
                for (int a = 0; a < ns; a++) {
                    const double *row = S + iy * W * ns + a;
                    double g;
                    if (W == 1) g = 0.0;
                    else if (ix == 0) g = row[ns] - row[0];
                    else if (ix == W - 1) g = row[(W - 1) * ns] - row[(W - 2) * ns];
                    else g = 0.5 * (row[(ix + 1) * ns] - row[(ix - 1) * ns]);
                    G[(iy * W + ix) * ns + a] = g;
                }
    }
    return 0;
}

int qo_sizeof_model(void) { return (int)sizeof(qo_model); }
int qo_has_openmp(void)
{
#ifdef _OPENMP
    return 1;
#else
    return 0;
#endif
}
