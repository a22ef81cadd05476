/*
 * afs_oracle.c -- plain, slow, fp64 CPU oracle for the Walsh-Fourier PGD hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  The product (paper_2606_06656_b200/)
 * shares no code with it and must never route through it.
 *
 * Every function follows PAPER.md (P:Lnn = /root/reference/PAPER.md line nn) step by step, in the
 * paper's notation; where the paper is silent or garbled the reading is the one listed in
 * DESIGN.md ("Readings", G1..G23).  Nothing here is blocked, fused or reordered for speed, with
 * one stated exception: orc_fe_B(mode=2) is a prefix/suffix-table form of the definitional
 * leave-one-out gradient (mode=1); the tests pin mode 2 to mode 1 to 1e-13.
 *
 * Polarity: True -> -1, False -> +1.  A literal is a signed 1-based int32: +(v+1) is x_v,
 * -(v+1) is NOT x_v, relaxed value y = sigma * x_v (G7).  A constraint's expansion is -1 when
 * satisfied, +1 when violated.
 *
 * Parity pins: every function below is pinned by tests/test_oracle_*.py (brute-force Walsh
 * transform, +-1 corner invariant, exact finite differences, multiprecision, metamorphic
 * identities); nothing is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ORC_OR = 0, ORC_XOR = 1, ORC_AMO = 2, ORC_EO = 3, ORC_EK = 4, ORC_NAE = 5, ORC_CARD = 6 };

/* ------------------------------------------------------------------------------------------
 * Constraint semantics (section 2.2; Table 2): is the constraint true when
 * exactly t of its L literals are true?  XOR: k is the required parity (1 = odd; G2).
 * CARD: t >= k, with k = 0 always true and k = L+1 never true (G5).  EK: t == k.
 * ------------------------------------------------------------------------------------------ */
int orc_pred(int type, int L, int k, int t)
{
    switch (type) {
    case ORC_OR:   return t >= 1;
    case ORC_XOR:  return (t & 1) == (k & 1);
    case ORC_AMO:  return t <= 1;
    case ORC_EO:   return t == 1;
    case ORC_EK:   return t == k;
    case ORC_NAE:  return t > 0 && t < L;
    case ORC_CARD: return t >= k;
    default:       return 0;
    }
}

/* sp_t = -1 if f is true when t literals are true and +1 otherwise. sp has L+1 entries. */
int orc_spectrum(int type, int L, int k, int *sp)
{
    if (type < 0 || type > 6 || L < 1) return -1;
    for (int t = 0; t <= L; ++t) sp[t] = orc_pred(type, L, k, t) ? -1 : 1;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O1.  Coefficients, eq. (3), exact integer arithmetic, L <= 62.
 *   a_0 = 2^-L sum_i C(L,i) sp_i
 *   a_s = [rho^(s-1)] g(rho) / ( C(L-1,s-1) 2^(L-1) ),   s >= 1
 *   g(rho) = sum_{i=0}^{L-1} d_i C(L-1,i) (1+rho)^(L-1-i) (1-rho)^i,   d_i = (sp_i - sp_{i+1})/2
 * The integer coefficients of (1+rho)^a (1-rho)^b are built by repeated exact multiplication
 * by (1+rho) and (1-rho) in __int128 (|g_j| < 2^122 for L <= 62); numerator and denominator
 * are converted to long double (64-bit mantissa, relative error 2^-64 each), divided once and
 * rounded to double: the result is within 1 ulp of the exact rational value.
 * ------------------------------------------------------------------------------------------ */
typedef __int128 i128;

static void binom_row(int n, i128 *c) /* c[0..n] = C(n,i) */
{
    c[0] = 1;
    for (int i = 1; i <= n; ++i) c[i] = c[i - 1] * (n - i + 1) / i;
}

int orc_coeffs_eq3(int type, int L, int k, double *a)
{
    if (type < 0 || type > 6 || L < 1 || L > 62) return -1;
    int sp[64];
    orc_spectrum(type, L, k, sp);
    i128 cL[64], cL1[64];
    binom_row(L, cL);
    binom_row(L - 1, cL1);
    /* |S| = 0 */
    i128 s0 = 0;
    for (int i = 0; i <= L; ++i) s0 += cL[i] * sp[i];
    a[0] = (double)((long double)s0 / ldexpl(1.0L, L));
    /* g(rho): degree L-1, integer coefficients */
    i128 g[64];
    for (int j = 0; j < L; ++j) g[j] = 0;
    for (int i = 0; i <= L - 1; ++i) {
        int two_d = sp[i] - sp[i + 1]; /* 2 d_i in {-2,0,2} */
        if (two_d == 0) continue;
        i128 poly[64];
        for (int j = 0; j < L; ++j) poly[j] = 0;
        poly[0] = 1;
        int deg = 0;
        for (int r = 0; r < L - 1 - i; ++r) { /* times (1+rho) */
            for (int j = deg + 1; j >= 1; --j) poly[j] += poly[j - 1];
            ++deg;
        }
        for (int r = 0; r < i; ++r) {         /* times (1-rho) */
            for (int j = deg + 1; j >= 1; --j) poly[j] -= poly[j - 1];
            ++deg;
        }
        for (int j = 0; j < L; ++j) g[j] += (i128)(two_d / 2) * cL1[i] * poly[j];
    }
    for (int s = 1; s <= L; ++s) {
        long double num = (long double)g[s - 1];
        long double den = (long double)cL1[s - 1] * ldexpl(1.0L, L - 1);
        a[s] = (double)(num / den);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O2.  Evaluator A: the literal form.  FE = sum_i a_i e_i(y) (eq. (1),(2); G1), the
 * e_i by the O(L^2) recurrence  e_i <- e_i + y_j e_{i-1}.  Gradient: d e_i / d y_j =
 * e_{i-1}(y without j), so dFE/dy_j = sum_{i>=1} a_i e_{i-1}(y \ j), the ESPs of the other
 * L-1 literals rebuilt from scratch for every j (O(L^3)).
 * Refuses (returns 1) when the conditioning guard  sum_i |a_i e_i| * 1.1e-16 > 1e-9  trips:
 * the literal form loses cond * 2^-53 (the paper's "floating-point ceiling").
 * ------------------------------------------------------------------------------------------ */
static void esp(int L, const double *y, int skip, double *e /* L+1 */)
{
    for (int i = 0; i <= L; ++i) e[i] = 0.0;
    e[0] = 1.0;
    int cnt = 0;
    for (int j = 0; j < L; ++j) {
        if (j == skip) continue;
        ++cnt;
        for (int i = cnt; i >= 1; --i) e[i] += y[j] * e[i - 1];
    }
}

int orc_fe_A(int type, int L, int k, const double *y, double *fe, double *grad)
{
    if (L < 1 || L > 62) return -1;
    double a[64], e[64];
    if (orc_coeffs_eq3(type, L, k, a)) return -1;
    esp(L, y, -1, e);
    double s = 0.0, sabs = 0.0;
    for (int i = 0; i <= L; ++i) { s += a[i] * e[i]; sabs += fabs(a[i] * e[i]); }
    if (sabs * 1.1e-16 > 1e-9) return 1;
    *fe = s;
    if (grad) {
        for (int j = 0; j < L; ++j) {
            esp(L, y, j, e);
            double gj = 0.0, gabs = 0.0;
            for (int i = 1; i <= L; ++i) { gj += a[i] * e[i - 1]; gabs += fabs(a[i] * e[i - 1]); }
            if (gabs * 1.1e-16 > 1e-9) return 1;
            grad[j] = gj;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O2'.  Evaluator B: the count basis (reading G10).  The Fourier expansion is THE multilinear
 * polynomial agreeing with f on {+-1}^L; E[f(Y)] for independent Y_j in {+-1} with
 * mean y_j is multilinear and agrees on the corners, hence FE(y) = sum_t sp_t Pr[T = t],
 * T = number of true literals, Pr[literal j true] = p_j = (1 - y_j)/2.  q = pmf of T by
 *      q_t <- q_t u_j + q_{t-1} p_j,   u_j = (1 + y_j)/2.
 * Gradient: dFE/dy_j = sum_t d_t q_t^{(-j)}, d_t the discrete derivative of the spectrum
 * (P:L52), q^{(-j)} the pmf over the other L-1 literals.
 *   mode 1: q^{(-j)} recomputed from scratch without literal j (definitional, O(L^3)).
 *   mode 2: q_t^{(-j)} = sum_u Pre_j[u] Suf_{j+1}[t-u] from full prefix / suffix pmf tables.
 * ------------------------------------------------------------------------------------------ */
static void pmf_skip(int L, const double *y, int skip, double *q /* L+1 */)
{
    for (int t = 0; t <= L; ++t) q[t] = 0.0;
    q[0] = 1.0;
    int cnt = 0;
    for (int j = 0; j < L; ++j) {
        if (j == skip) continue;
        double p = 0.5 * (1.0 - y[j]), u = 0.5 * (1.0 + y[j]);
        ++cnt;
        for (int t = cnt; t >= 1; --t) q[t] = q[t] * u + q[t - 1] * p;
        q[0] = q[0] * u;
    }
}

int orc_fe_B(int type, int L, int k, const double *y, double *fe, double *grad, int mode)
{
    if (type < 0 || type > 6 || L < 1) return -1;
    int *sp = (int *)malloc((size_t)(L + 1) * sizeof(int));
    double *q = (double *)malloc((size_t)(L + 1) * sizeof(double));
    if (!sp || !q) { free(sp); free(q); return -2; }
    orc_spectrum(type, L, k, sp);
    pmf_skip(L, y, -1, q);
    double s = 0.0;
    for (int t = 0; t <= L; ++t) s += sp[t] * q[t];
    *fe = s;
    int rc = 0;
    if (grad && mode != 2) {
        for (int j = 0; j < L; ++j) {
            pmf_skip(L, y, j, q); /* entries 0..L-1 */
            double gj = 0.0;
            for (int t = 0; t <= L - 1; ++t) gj += 0.5 * (sp[t] - sp[t + 1]) * q[t];
            grad[j] = gj;
        }
    } else if (grad) {
        size_t W = (size_t)L + 1;
        double *pre = (double *)calloc(W * W, sizeof(double)); /* pre[j] = pmf of literals 0..j-1 */
        double *suf = (double *)calloc(W * W, sizeof(double)); /* suf[j] = pmf of literals j..L-1 */
        if (!pre || !suf) { rc = -2; }
        else {
            pre[0] = 1.0;
            for (int j = 0; j < L; ++j) {
                double p = 0.5 * (1.0 - y[j]), u = 0.5 * (1.0 + y[j]);
                const double *a = pre + (size_t)j * W; double *b = pre + (size_t)(j + 1) * W;
                b[0] = a[0] * u;
                for (int t = 1; t <= j + 1; ++t) b[t] = a[t] * u + a[t - 1] * p;
            }
            suf[(size_t)L * W] = 1.0;
            for (int j = L - 1; j >= 0; --j) {
                double p = 0.5 * (1.0 - y[j]), u = 0.5 * (1.0 + y[j]);
                const double *a = suf + (size_t)(j + 1) * W; double *b = suf + (size_t)j * W;
                b[0] = a[0] * u;
                for (int t = 1; t <= L - j; ++t) b[t] = a[t] * u + a[t - 1] * p;
            }
            for (int j = 0; j < L; ++j) {
                const double *a = pre + (size_t)j * W, *b = suf + (size_t)(j + 1) * W;
                double gj = 0.0;
                for (int t = 0; t <= L - 1; ++t) {
                    int two_d = sp[t] - sp[t + 1];
                    if (two_d == 0) continue;
                    /* u literals true among the first j, t-u among the last L-1-j */
                    int ulo = t - (L - 1 - j); if (ulo < 0) ulo = 0;
                    int uhi = t < j ? t : j;
                    double c = 0.0;
                    for (int u = ulo; u <= uhi; ++u) c += a[u] * b[t - u];
                    gj += 0.5 * two_d * c;
                }
                grad[j] = gj;
            }
        }
        free(pre); free(suf);
    }
    free(sp); free(q);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * O3.  F(b) = sum_k FE_{C_k}(X_b) (eq. (5), unit weights G9);
 *      G[b,v] = sum over literals (k,j) of variable v of sigma_j dFE_k/dy_j, in index order
 *      (ascending constraint id, then position).
 * evaluator: 0 = A (literal, L <= 62, may refuse -> returns 1), 1 = B definitional, 2 = B tables.
 * X, G are [B,n] row-major fp64; F is [B].  G or F may be NULL.
 * ------------------------------------------------------------------------------------------ */
static int check_instance(int n, int64_t m, const int64_t *row_ptr, const int32_t *lits,
                          const int32_t *types, const int32_t *k)
{
    if (n < 1 || m < 0) return -1;
    /* G8: the multilinear expansion assumes distinct variables inside a constraint, so the
     * same variable twice is rejected.  seen[v] = 1 + the last constraint that used variable v. */
    int64_t *seen = (int64_t *)calloc((size_t)n, sizeof(int64_t));
    if (!seen) return -1;
    int bad = 0;
    for (int64_t c = 0; c < m && !bad; ++c) {
        int64_t L = row_ptr[c + 1] - row_ptr[c];
        if (L < 1 || types[c] < 0 || types[c] > 6) { bad = 1; break; }
        if (types[c] == ORC_NAE && L < 2) { bad = 1; break; }            /* G6 */
        if ((types[c] == ORC_EK || types[c] == ORC_CARD) && (k[c] < 0 || k[c] > L + 1)) { bad = 1; break; }
        if (types[c] == ORC_XOR && (k[c] < 0 || k[c] > 1)) { bad = 1; break; }
        for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
            int32_t l = lits[e];
            if (l == 0 || l > n || l < -n) { bad = 1; break; }
            int32_t v = (l < 0 ? -l : l) - 1;
            if (seen[v] == c + 1) { bad = 1; break; }                    /* G8 */
            seen[v] = c + 1;
        }
    }
    free(seen);
    return bad ? -1 : 0;
}

static int eval_one(int n, int64_t m, const int64_t *row_ptr, const int32_t *lits,
                    const int32_t *types, const int32_t *k, const double *x,
                    double *F, double *g /* n or NULL */, int evaluator, int Lmax,
                    double *ybuf, double *gbuf)
{
    double f = 0.0;
    if (g) for (int v = 0; v < n; ++v) g[v] = 0.0;
    for (int64_t c = 0; c < m; ++c) {
        int L = (int)(row_ptr[c + 1] - row_ptr[c]);
        const int32_t *lc = lits + row_ptr[c];
        for (int j = 0; j < L; ++j) {
            int v = abs(lc[j]) - 1;
            ybuf[j] = lc[j] > 0 ? x[v] : -x[v];
        }
        double fe;
        int rc = evaluator == 0 ? orc_fe_A(types[c], L, k[c], ybuf, &fe, g ? gbuf : NULL)
                                : orc_fe_B(types[c], L, k[c], ybuf, &fe, g ? gbuf : NULL, evaluator);
        if (rc) return rc;
        f += fe;
        if (g) for (int j = 0; j < L; ++j) {
            int v = abs(lc[j]) - 1;
            g[v] += lc[j] > 0 ? gbuf[j] : -gbuf[j];   /* chain rule through the literal sign */
        }
    }
    (void)Lmax;
    if (F) *F = f;
    return 0;
}

static int max_len(int64_t m, const int64_t *row_ptr)
{
    int64_t L = 1;
    for (int64_t c = 0; c < m; ++c) if (row_ptr[c + 1] - row_ptr[c] > L) L = row_ptr[c + 1] - row_ptr[c];
    return (int)L;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int orc_eval_grad(int n, int64_t m, const int64_t *row_ptr, const int32_t *lits,
                  const int32_t *types, const int32_t *k, const double *X, int B,
                  double *F, double *G, int evaluator, int nthreads)
{
    if (check_instance(n, m, row_ptr, lits, types, k)) return -1;
    int Lmax = max_len(m, row_ptr);
    int err = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    (void)nthreads;
#pragma omp parallel
    {
        double *ybuf = (double *)malloc((size_t)Lmax * sizeof(double));
        double *gbuf = (double *)malloc((size_t)Lmax * sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int b = 0; b < B; ++b) {
            int rc = eval_one(n, m, row_ptr, lits, types, k, X + (size_t)b * n,
                              F ? F + b : NULL, G ? G + (size_t)b * n : NULL, evaluator, Lmax, ybuf, gbuf);
            if (rc) {
#pragma omp critical
                err = rc;
            }
        }
        free(ybuf); free(gbuf);
    }
    return err;
}

/* ------------------------------------------------------------------------------------------
 * O5.  Rounding and satisfaction count (satisfied iff sum_k FE(sign X) = -m).
 * s_v = True iff x_v < 0; x >= 0 (including +-0.0) and NaN round to False (G13).  Integers only:
 * t_k = number of true literals, constraint satisfied iff orc_pred(type, L, k, t_k).
 * assign (may be NULL) receives -1 for True, +1 for False.
 * ------------------------------------------------------------------------------------------ */
static int32_t count_one(int n, int64_t m, const int64_t *row_ptr, const int32_t *lits,
                         const int32_t *types, const int32_t *k, const double *x, int8_t *assign)
{
    (void)n;
    int32_t sat = 0;
    if (assign) for (int v = 0; v < n; ++v) assign[v] = x[v] < 0.0 ? -1 : 1;
    for (int64_t c = 0; c < m; ++c) {
        int L = (int)(row_ptr[c + 1] - row_ptr[c]);
        int t = 0;
        for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
            int v = abs(lits[e]) - 1;
            int var_true = x[v] < 0.0;
            t += lits[e] > 0 ? var_true : !var_true;
        }
        sat += orc_pred(types[c], L, k[c], t);
    }
    return sat;
}

int orc_round_count(int n, int64_t m, const int64_t *row_ptr, const int32_t *lits,
                    const int32_t *types, const int32_t *k, const double *X, int B,
                    int8_t *assign, int32_t *sat)
{
    if (check_instance(n, m, row_ptr, lits, types, k)) return -1;
#pragma omp parallel for schedule(static)
    for (int b = 0; b < B; ++b)
        sat[b] = count_one(n, m, row_ptr, lits, types, k, X + (size_t)b * n,
                           assign ? assign + (size_t)b * n : NULL);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O4 + O6.  Batched projected gradient descent (readings G11, G12, G14, G16):
 *   entry: fixed coordinates (mask[v] != 0) are overwritten with mask[v]
 *   for t = 0 .. steps:  round and count X_t; if sat > best (strictly) keep (sat, sign X_t, t)
 *                        if t < steps:  X_{t+1} = clip(X_t - lr * grad F(X_t), -1, +1) on free
 *                                       coordinates; fixed coordinates keep their value
 * X [B,n] fp64 in/out.  traj (NULL or [(steps+1),B,n]) receives every iterate, sat_hist (NULL or
 * [(steps+1),B]) every count.  Restarts are independent, hence the OpenMP loop.
 * ------------------------------------------------------------------------------------------ */
int orc_pgd_run(int n, int64_t m, const int64_t *row_ptr, const int32_t *lits,
                const int32_t *types, const int32_t *k, double *X, int B, int steps, double lr,
                const int8_t *mask, int8_t *best_assign, int32_t *best_sat, int32_t *best_step,
                double *traj, int32_t *sat_hist, int evaluator, int nthreads)
{
    if (check_instance(n, m, row_ptr, lits, types, k) || steps < 0) return -1;
    int Lmax = max_len(m, row_ptr);
    int err = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    (void)nthreads;
#pragma omp parallel
    {
        double *ybuf = (double *)malloc((size_t)Lmax * sizeof(double));
        double *gbuf = (double *)malloc((size_t)Lmax * sizeof(double));
        double *g = (double *)malloc((size_t)n * sizeof(double));
        int8_t *cur = (int8_t *)malloc((size_t)n);
#pragma omp for schedule(dynamic, 1)
        for (int b = 0; b < B; ++b) {
            double *x = X + (size_t)b * n;
            if (mask) for (int v = 0; v < n; ++v) if (mask[v]) x[v] = (double)mask[v];
            int32_t best = -1;
            for (int t = 0; t <= steps; ++t) {
                int32_t s = count_one(n, m, row_ptr, lits, types, k, x, cur);
                if (sat_hist) sat_hist[(size_t)t * B + b] = s;
                if (traj) memcpy(traj + ((size_t)t * B + b) * n, x, (size_t)n * sizeof(double));
                if (s > best) {
                    best = s;
                    if (best_assign) memcpy(best_assign + (size_t)b * n, cur, (size_t)n);
                    if (best_step) best_step[b] = t;
                }
                if (t == steps) break;
                int rc = eval_one(n, m, row_ptr, lits, types, k, x, NULL, g, evaluator, Lmax, ybuf, gbuf);
                if (rc) {
#pragma omp critical
                    err = rc;
                    break;
                }
                for (int v = 0; v < n; ++v) {
                    if (mask && mask[v]) continue;
                    double xn = x[v] - lr * g[v];
                    if (xn > 1.0) xn = 1.0;
                    if (xn < -1.0) xn = -1.0;
                    x[v] = xn;
                }
            }
            if (best_sat) best_sat[b] = best;
        }
        free(ybuf); free(gbuf); free(g); free(cur);
    }
    return err;
}

/* ------------------------------------------------------------------------------------------
 * PGD with per-restart convergence detection ("the small step size satisfies convergence criteria
 * prematurely"; L152-L164: restarts converge at different times and "all batch elements must iterate together;
 * idling converged elements waste compute"; the criterion itself is not printed: DESIGN.md reading G24).
 *   A restart stops after the first step t -> t+1 with  max_v |X_{t+1}[v] - X_t[v]| < tol  (free coordinates); its
 *   iterate stays X_{t+1} from then on, conv_step[b] = t+1 = the number of steps it took; -1 if it never stops within
 *   max_steps.  Every iterate it reaches is rounded and counted (X_0 .. X_{conv_step}), best as in orc_pgd_run.
 *   tol <= 0 never stops a restart: identical to orc_pgd_run.
 * Outputs for the histograms of Fig. 4-5: final_sat[b] = satisfied constraints of the returned X
 * (#unsatisfied = m - final_sat), final_F[b] = objective of the returned X ("energy"), conv_step[b] ("steps").
 * ------------------------------------------------------------------------------------------ */
int orc_pgd_run_conv(int n, int64_t m, const int64_t *row_ptr, const int32_t *lits,
                     const int32_t *types, const int32_t *k, double *X, int B, int max_steps, double lr,
                     const int8_t *mask, double tol, int8_t *best_assign, int32_t *best_sat, int32_t *best_step,
                     int32_t *conv_step, int32_t *final_sat, double *final_F, int evaluator, int nthreads)
{
    if (check_instance(n, m, row_ptr, lits, types, k) || max_steps < 0) return -1;
    int Lmax = max_len(m, row_ptr);
    int err = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    (void)nthreads;
#pragma omp parallel
    {
        double *ybuf = (double *)malloc((size_t)Lmax * sizeof(double));
        double *gbuf = (double *)malloc((size_t)Lmax * sizeof(double));
        double *g = (double *)malloc((size_t)n * sizeof(double));
        int8_t *cur = (int8_t *)malloc((size_t)n);
#pragma omp for schedule(dynamic, 1)
        for (int b = 0; b < B; ++b) {
            double *x = X + (size_t)b * n;
            if (mask) for (int v = 0; v < n; ++v) if (mask[v]) x[v] = (double)mask[v];
            int32_t best = -1, conv = -1, s = 0;
            for (int t = 0; t <= max_steps; ++t) {
                s = count_one(n, m, row_ptr, lits, types, k, x, cur);
                if (s > best) {
                    best = s;
                    if (best_assign) memcpy(best_assign + (size_t)b * n, cur, (size_t)n);
                    if (best_step) best_step[b] = t;
                }
                if (t == max_steps || conv >= 0) break;
                int rc = eval_one(n, m, row_ptr, lits, types, k, x, NULL, g, evaluator, Lmax, ybuf, gbuf);
                if (rc) {
#pragma omp critical
                    err = rc;
                    break;
                }
                double delta = 0.0;
                for (int v = 0; v < n; ++v) {
                    if (mask && mask[v]) continue;
                    double xn = x[v] - lr * g[v];
                    if (xn > 1.0) xn = 1.0;
                    if (xn < -1.0) xn = -1.0;
                    double d = fabs(xn - x[v]);
                    if (d > delta) delta = d;
                    x[v] = xn;
                }
                if (delta < tol) conv = t + 1;
            }
            if (best_sat) best_sat[b] = best;
            if (conv_step) conv_step[b] = conv;
            if (final_sat) final_sat[b] = s;
            if (final_F) {
                double F = 0.0;
                int rc = eval_one(n, m, row_ptr, lits, types, k, x, &F, NULL, evaluator, Lmax, ybuf, gbuf);
                if (rc) {
#pragma omp critical
                    err = rc;
                }
                final_F[b] = F;
            }
        }
        free(ybuf); free(gbuf); free(g); free(cur);
    }
    return err;
}

/* ------------------------------------------------------------------------------------------
 * Per-constraint weights ("adaptive constraint weighting -- informed by per-constraint gradient
 * magnitudes"; L188 (i); reading G25).  eq. (5) with weights:  F_w(X) = sum_k w_k FE_{C_k}(X), hence
 * dF_w/dx_v = sum_k w_k sigma dFE_k/dy.  New functions; the unweighted ones above are untouched.
 *   gm (NULL or [m]) receives the per-constraint gradient magnitude summed over the batch, UNWEIGHTED:
 *   gm[k] = sum_b sum_j |dFE_k/dy_j (X_b)|  (the l1 norm is this build's reading of "gradient magnitude").
 * ------------------------------------------------------------------------------------------ */
static int eval_one_w(int n, int64_t m, const int64_t *row_ptr, const int32_t *lits,
                      const int32_t *types, const int32_t *k, const double *w, const double *x,
                      double *F, double *g /* n or NULL */, double *gm /* m or NULL */, int evaluator,
                      double *ybuf, double *gbuf)
{
    double f = 0.0;
    if (g) for (int v = 0; v < n; ++v) g[v] = 0.0;
    for (int64_t c = 0; c < m; ++c) {
        int L = (int)(row_ptr[c + 1] - row_ptr[c]);
        const int32_t *lc = lits + row_ptr[c];
        for (int j = 0; j < L; ++j) {
            int v = abs(lc[j]) - 1;
            ybuf[j] = lc[j] > 0 ? x[v] : -x[v];
        }
        double fe;
        int need_g = (g != NULL) || (gm != NULL);
        int rc = evaluator == 0 ? orc_fe_A(types[c], L, k[c], ybuf, &fe, need_g ? gbuf : NULL)
                                : orc_fe_B(types[c], L, k[c], ybuf, &fe, need_g ? gbuf : NULL, evaluator);
        if (rc) return rc;
        const double wc = w ? w[c] : 1.0;
        f += wc * fe;
        if (g) for (int j = 0; j < L; ++j) {
            int v = abs(lc[j]) - 1;
            g[v] += wc * (lc[j] > 0 ? gbuf[j] : -gbuf[j]);
        }
        if (gm) {
            double s = 0.0;
            for (int j = 0; j < L; ++j) s += fabs(gbuf[j]);
            gm[c] = s;
        }
    }
    if (F) *F = f;
    return 0;
}

int orc_eval_grad_w(int n, int64_t m, const int64_t *row_ptr, const int32_t *lits,
                    const int32_t *types, const int32_t *k, const double *w, const double *X, int B,
                    double *F, double *G, double *GM /* m or NULL, summed over the batch */, int evaluator)
{
    if (check_instance(n, m, row_ptr, lits, types, k)) return -1;
    int Lmax = max_len(m, row_ptr);
    double *ybuf = (double *)malloc((size_t)Lmax * sizeof(double));
    double *gbuf = (double *)malloc((size_t)Lmax * sizeof(double));
    double *gm1 = GM ? (double *)malloc((size_t)(m ? m : 1) * sizeof(double)) : NULL;
    if (GM) for (int64_t c = 0; c < m; ++c) GM[c] = 0.0;
    int err = 0;
    for (int b = 0; b < B && !err; ++b) {          /* plain loop: the batch sum of GM is taken in restart order */
        err = eval_one_w(n, m, row_ptr, lits, types, k, w, X + (size_t)b * n, F ? F + b : NULL,
                         G ? G + (size_t)b * n : NULL, gm1, evaluator, ybuf, gbuf);
        if (GM && !err) for (int64_t c = 0; c < m; ++c) GM[c] += gm1[c];
    }
    free(ybuf); free(gbuf); free(gm1);
    return err;
}

int orc_pgd_run_w(int n, int64_t m, const int64_t *row_ptr, const int32_t *lits,
                  const int32_t *types, const int32_t *k, const double *w, double *X, int B, int steps, double lr,
                  const int8_t *mask, int8_t *best_assign, int32_t *best_sat, int32_t *best_step, int evaluator)
{
    if (check_instance(n, m, row_ptr, lits, types, k) || steps < 0) return -1;
    int Lmax = max_len(m, row_ptr);
    int err = 0;
#pragma omp parallel
    {
        double *ybuf = (double *)malloc((size_t)Lmax * sizeof(double));
        double *gbuf = (double *)malloc((size_t)Lmax * sizeof(double));
        double *g = (double *)malloc((size_t)n * sizeof(double));
        int8_t *cur = (int8_t *)malloc((size_t)n);
#pragma omp for schedule(dynamic, 1)
        for (int b = 0; b < B; ++b) {
            double *x = X + (size_t)b * n;
            if (mask) for (int v = 0; v < n; ++v) if (mask[v]) x[v] = (double)mask[v];
            int32_t best = -1;
            for (int t = 0; t <= steps; ++t) {
                int32_t s = count_one(n, m, row_ptr, lits, types, k, x, cur);   /* counts do not see the weights */
                if (s > best) {
                    best = s;
                    if (best_assign) memcpy(best_assign + (size_t)b * n, cur, (size_t)n);
                    if (best_step) best_step[b] = t;
                }
                if (t == steps) break;
                int rc = eval_one_w(n, m, row_ptr, lits, types, k, w, x, NULL, g, NULL, evaluator, ybuf, gbuf);
                if (rc) {
#pragma omp critical
                    err = rc;
                    break;
                }
                for (int v = 0; v < n; ++v) {
                    if (mask && mask[v]) continue;
                    double xn = x[v] - lr * g[v];
                    if (xn > 1.0) xn = 1.0;
                    if (xn < -1.0) xn = -1.0;
                    x[v] = xn;
                }
            }
            if (best_sat) best_sat[b] = best;
        }
        free(ybuf); free(gbuf); free(g); free(cur);
    }
    return err;
}
