/*
 * cs_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded fp64 CPU implementation of Algorithm 1 / Algorithm 2 of
 * "Rapid Convergence of First-Order Numerical Algorithms via Adaptive Conditioning"
 * (arXiv 2103.00736), written from the paper (/root/reference/PAPER.md, cited as P:<line>) in the
 * paper's order and notation.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code, header, table or
 * helper with the CUDA library under paper_2103_00736_b200/csrc/ and neither includes the other.
 *
 * Readings of the paper where it is silent or garbled (SURVEY.md 8(c) a-w):
 *   - A^dagger = A'(AA')^{-1} (n x m), range(A') is a subspace, abs_A(v) = 2 A^dagger A v - v
 *     (pinned by (27d) P:509 and (37b) P:591).
 *   - o is constant over a cone block, O = o^alpha, alpha = min{1, t/(ln max o - ln min o)} with the
 *     natural log and alpha = 1 when the spread is 0.
 *   - numerator and denominator of o are floored at o_floor (paper silent on 0/0).
 *   - O is absolute: A_hat = A*O from the pristine A at every conditioning (P:233-240 use A,b,c).
 *   - x,z of steps 19-20 use p from step 16 and s AFTER step 18.
 *   - no row scaling: D^AC = I.
 *   - size-1 Lorentz cone = one orthant coordinate (P:52-56 with n_i = 1; LPs use R^n_+ P:148).
 *   - how A^dagger is applied is not stated: dense Cholesky of (A_hat A_hat') for small m, otherwise
 *     Jacobi-preconditioned CG from a zero start to a tight tolerance ("exact" solve).
 *   - y = (w_d - w)/mu is a derived dual multiplier (the paper never forms y).
 *   - stop rule (16) needs a competing solver; replaced by the relative KKT residual below.
 *
 * Parity unpinned: none of the functions below; the ill-conditioned map (x,z) -> O after a late
 * conditioning is pinned only through x,z.
 *
 * All sums are sequential left-to-right.  No blocking, fusion or reordering.
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

typedef struct orc_solver {
    /* problem (1): min c'x s.t. Ax=b, x in K   [P:41-56] */
    int64_t m, n, nnz;
    int32_t *row_ptr, *col_idx;
    double *val;      /* pristine A (CSR)            */
    double *val_hat;  /* A_hat = A*O (same pattern)  */
    double *b, *c, *c_hat;
    int64_t n_lin, n_soc;
    int32_t *soc_size;
    /* parameters */
    double mu, t, o_floor;
    int solve_mode;   /* 1 = dense Cholesky, 2 = Jacobi-PCG */
    double pcg_tol;
    int64_t pcg_max;
    /* state of Algorithm 2 */
    int64_t l;        /* iteration counter (step 1,3) */
    double *O;        /* diagonal of O                */
    double *d, *s, *p, *r, *x, *z;
    double *w, *w_d;  /* (A_hat A_hat')^{-1} A_hat p  and the multiplier behind d */
    double *chol;     /* m*m lower Cholesky factor of A_hat A_hat' (solve_mode 1) */
    double *jac;      /* diag(A_hat A_hat') (solve_mode 2) */
    int64_t n_cond, pcg_steps_total, pcg_steps_last;
    double fp_res;    /* ||s_new - s||_2 of the last pass */
    int pcg_fail;
} orc_solver;

/* ------------------------------------------------------------------------------------------ */
/* Definition 1 [P:98-104]: proj_C(v) = argmin_{u in C} ||u - v||_2 ; abs_C(v) = 2 proj_C(v) - v */
/* ------------------------------------------------------------------------------------------ */

/* Projection onto one Lorentz cone K_k = { w : w_1 >= ||w_2..k||_2 } [P:54] (textbook closed form;
 * the paper does not print it).  k = 1 gives max(v,0). */
static void proj_lorentz(const double *v, double *out, int64_t k) {
    double t = v[0], nu = 0.0;
    for (int64_t j = 1; j < k; ++j) nu += v[j] * v[j];
    nu = sqrt(nu);
    if (nu <= t) {                 /* v in K: projection is v */
        for (int64_t j = 0; j < k; ++j) out[j] = v[j];
    } else if (nu <= -t) {         /* -v in K (polar): projection is 0 */
        for (int64_t j = 0; j < k; ++j) out[j] = 0.0;
    } else {                       /* otherwise: ((t+nu)/2) * (1, u/nu) */
        double a = 0.5 * (t + nu);
        out[0] = a;
        for (int64_t j = 1; j < k; ++j) out[j] = a * v[j] / nu;
    }
}

/* proj_K for K = R^{n_lin}_+ x K_{soc_size[0]} x ... [P:52-56] */
void orc_proj_cone(const double *v, double *out, int64_t n_lin, int64_t n_soc, const int32_t *soc_size) {
    for (int64_t j = 0; j < n_lin; ++j) proj_lorentz(v + j, out + j, 1);
    int64_t h = n_lin;
    for (int64_t i = 0; i < n_soc; ++i) {
        proj_lorentz(v + h, out + h, soc_size[i]);
        h += soc_size[i];
    }
}

/* abs_K(v) = 2 proj_K(v) - v  [P:102-104] */
void orc_abs_cone(const double *v, double *out, int64_t n_lin, int64_t n_soc, const int32_t *soc_size) {
    orc_proj_cone(v, out, n_lin, n_soc, soc_size);
    int64_t n = n_lin;
    for (int64_t i = 0; i < n_soc; ++i) n += soc_size[i];
    for (int64_t j = 0; j < n; ++j) out[j] = 2.0 * out[j] - v[j];
}

/* ------------------------------------------------------------------------------------------ */
/* sparse products with A_hat = A*O (CSR)                                                      */
/* ------------------------------------------------------------------------------------------ */

static void mat_vec(const orc_solver *S, const double *val, const double *v, double *out) { /* out = A v */
    for (int64_t i = 0; i < S->m; ++i) {
        double acc = 0.0;
        for (int32_t k = S->row_ptr[i]; k < S->row_ptr[i + 1]; ++k) acc += val[k] * v[S->col_idx[k]];
        out[i] = acc;
    }
}

static void mat_tvec(const orc_solver *S, const double *val, const double *y, double *out) { /* out = A' y */
    for (int64_t j = 0; j < S->n; ++j) out[j] = 0.0;
    for (int64_t i = 0; i < S->m; ++i)
        for (int32_t k = S->row_ptr[i]; k < S->row_ptr[i + 1]; ++k) out[S->col_idx[k]] += val[k] * y[i];
}

/* ------------------------------------------------------------------------------------------ */
/* "solve": w = (A_hat A_hat')^{-1} rhs  -- the linear solve hidden in A^dagger [P:66, P:74]   */
/* ------------------------------------------------------------------------------------------ */

/* dense lower Cholesky of G = A_hat A_hat' (row-major m x m); returns 0 on success */
static int build_cholesky(orc_solver *S) {
    const int64_t m = S->m, n = S->n;
    double *G = S->chol;
    double *dense_row = (double *)calloc((size_t)(n > 0 ? n : 1), sizeof(double));
    if (!dense_row) return 1;
    for (int64_t i = 0; i < m; ++i) {
        for (int32_t k = S->row_ptr[i]; k < S->row_ptr[i + 1]; ++k) dense_row[S->col_idx[k]] = S->val_hat[k];
        for (int64_t q = 0; q <= i; ++q) {                    /* G[i][q] = <row i, row q> */
            double acc = 0.0;
            for (int32_t k = S->row_ptr[q]; k < S->row_ptr[q + 1]; ++k) acc += S->val_hat[k] * dense_row[S->col_idx[k]];
            G[i * m + q] = acc;
        }
        for (int32_t k = S->row_ptr[i]; k < S->row_ptr[i + 1]; ++k) dense_row[S->col_idx[k]] = 0.0;
    }
    free(dense_row);
    /* symmetric diagonal equilibration G <- E G E, E = diag(G)^{-1/2} (kept in S->jac as G_ii): the
     * same solve, w = E (EGE)^{-1} E rhs, but the factorisation error is governed by cond(EGE)
     * instead of cond(G) (van der Sluis); matters for the badly row-scaled config 2. */
    for (int64_t i = 0; i < m; ++i) {
        if (!(G[i * m + i] > 0.0)) return 3;
        S->jac[i] = G[i * m + i];
    }
    for (int64_t i = 0; i < m; ++i)
        for (int64_t q = 0; q <= i; ++q) G[i * m + q] = G[i * m + q] / (sqrt(S->jac[i]) * sqrt(S->jac[q]));
    /* textbook Cholesky-Banachiewicz, in place on the lower triangle */
    for (int64_t i = 0; i < m; ++i) {
        for (int64_t j = 0; j <= i; ++j) {
            double acc = G[i * m + j];
            for (int64_t k = 0; k < j; ++k) acc -= G[i * m + k] * G[j * m + k];
            if (i == j) {
                if (!(acc > 0.0)) return 2;                    /* not positive definite: rank-deficient A */
                G[i * m + i] = sqrt(acc);
            } else {
                G[i * m + j] = acc / G[j * m + j];
            }
        }
    }
    return 0;
}

/* one application of the factor: w = E (L L')^{-1} E rhs */
static void cholesky_apply(const orc_solver *S, const double *rhs, double *w) {
    const int64_t m = S->m;
    const double *Lc = S->chol;
    for (int64_t i = 0; i < m; ++i) {                          /* L t = E rhs */
        double acc = rhs[i] / sqrt(S->jac[i]);
        for (int64_t k = 0; k < i; ++k) acc -= Lc[i * m + k] * w[k];
        w[i] = acc / Lc[i * m + i];
    }
    for (int64_t i = m - 1; i >= 0; --i) {                     /* L' w = t */
        double acc = w[i];
        for (int64_t k = i + 1; k < m; ++k) acc -= Lc[k * m + i] * w[k];
        w[i] = acc / Lc[i * m + i];
    }
    for (int64_t i = 0; i < m; ++i) w[i] = w[i] / sqrt(S->jac[i]);   /* w = E (.) */
}

/* "Exact" solve (reading (s): the paper hides a solve inside A^dagger and treats it as exact): the
 * factor is applied, then ORC_REFINE steps of textbook iterative refinement against the operator
 * itself, res = rhs - A_hat (A_hat' w) evaluated with the sparse products (not with the rounded,
 * formed G), w += (L L')^{-1} res.  Each step contracts the error by ~ eps * cond(EGE), so two steps
 * leave the solve at the rounding level of the residual evaluation even for the cond ~ 1e13 systems
 * of config 2. */
#define ORC_REFINE 2
static void cholesky_solve(const orc_solver *S, const double *rhs, double *w) {
    const int64_t m = S->m, n = S->n;
    cholesky_apply(S, rhs, w);
    double *u = (double *)malloc(sizeof(double) * (size_t)n), *res = (double *)malloc(sizeof(double) * (size_t)m);
    double *dw = (double *)malloc(sizeof(double) * (size_t)m);
    for (int step = 0; step < ORC_REFINE; ++step) {
        mat_tvec(S, S->val_hat, w, u);                         /* u = A_hat' w           */
        mat_vec(S, S->val_hat, u, res);                        /* res = A_hat A_hat' w   */
        for (int64_t i = 0; i < m; ++i) res[i] = rhs[i] - res[i];
        cholesky_apply(S, res, dw);
        for (int64_t i = 0; i < m; ++i) w[i] += dw[i];
    }
    free(u); free(res); free(dw);
}

/* Jacobi-preconditioned CG on (A_hat A_hat') w = rhs from w = 0 (textbook PCG).  Stops when
 * sqrt(r'M^{-1}r) <= pcg_tol * sqrt(rhs'M^{-1}rhs) or at pcg_max (flagged in pcg_fail).  Returns the
 * number of steps. */
static int64_t pcg_solve(orc_solver *S, const double *rhs, double *w) {
    const int64_t m = S->m, n = S->n;
    double *r = (double *)malloc(sizeof(double) * (size_t)m), *zv = (double *)malloc(sizeof(double) * (size_t)m);
    double *pv = (double *)malloc(sizeof(double) * (size_t)m), *q = (double *)malloc(sizeof(double) * (size_t)m);
    double *u = (double *)malloc(sizeof(double) * (size_t)n);
    double rz = 0.0, ref = 0.0;
    for (int64_t i = 0; i < m; ++i) { w[i] = 0.0; r[i] = rhs[i]; zv[i] = r[i] / S->jac[i]; pv[i] = zv[i]; }
    for (int64_t i = 0; i < m; ++i) rz += r[i] * zv[i];
    ref = rz;
    int64_t it = 0;
    const double thresh = S->pcg_tol * S->pcg_tol * ref;
    while (rz > thresh && it < S->pcg_max) {
        mat_tvec(S, S->val_hat, pv, u);                        /* u = A_hat' p          */
        mat_vec(S, S->val_hat, u, q);                          /* q = A_hat A_hat' p    */
        double pq = 0.0;
        for (int64_t i = 0; i < m; ++i) pq += pv[i] * q[i];
        if (!(pq > 0.0)) break;
        double alpha = rz / pq;
        for (int64_t i = 0; i < m; ++i) { w[i] += alpha * pv[i]; r[i] -= alpha * q[i]; }
        double rz_new = 0.0;
        for (int64_t i = 0; i < m; ++i) { zv[i] = r[i] / S->jac[i]; rz_new += r[i] * zv[i]; }
        double beta = rz_new / rz;
        for (int64_t i = 0; i < m; ++i) pv[i] = zv[i] + beta * pv[i];
        rz = rz_new;
        ++it;
    }
    if (it >= S->pcg_max && rz > thresh) S->pcg_fail |= 2;
    free(r); free(zv); free(pv); free(q); free(u);
    S->pcg_steps_last = it;
    S->pcg_steps_total += it;
    return it;
}

static void solve_normal(orc_solver *S, const double *rhs, double *w) {
    if (S->solve_mode == 1) { cholesky_solve(S, rhs, w); S->pcg_steps_last = 0; }
    else pcg_solve(S, rhs, w);
}

/* out = A_hat^dagger rhs = A_hat' (A_hat A_hat')^{-1} rhs ; keeps the multiplier in w_out  [P:37, P:66] */
static void apply_pinv(orc_solver *S, const double *rhs, double *w_out, double *out) {
    solve_normal(S, rhs, w_out);
    mat_tvec(S, S->val_hat, w_out, out);
}

/* abs over the subspace range{A_hat'}: out = 2 A_hat^dagger A_hat v - v  [P:63, (37b) P:591] */
static void abs_range(orc_solver *S, const double *v, double *w_out, double *out) {
    double *Av = (double *)malloc(sizeof(double) * (size_t)S->m);
    mat_vec(S, S->val_hat, v, Av);
    apply_pinv(S, Av, w_out, out);
    for (int64_t j = 0; j < S->n; ++j) out[j] = 2.0 * out[j] - v[j];
    free(Av);
}

/* ------------------------------------------------------------------------------------------ */
/* Algorithm 2, steps 11-14 for a GIVEN positive diagonal O  [P:233-240]                        */
/* ------------------------------------------------------------------------------------------ */
static int apply_scaling(orc_solver *S) {
    const int64_t m = S->m, n = S->n;
    /* A_hat = A O (from the pristine A), c_hat = O'c   [P:235-238, (13) P:258-266] */
    for (int64_t i = 0; i < m; ++i)
        for (int32_t k = S->row_ptr[i]; k < S->row_ptr[i + 1]; ++k) S->val_hat[k] = S->val[k] * S->O[S->col_idx[k]];
    for (int64_t j = 0; j < n; ++j) S->c_hat[j] = S->O[j] * S->c[j];
    if (S->solve_mode == 1) {
        int rc = build_cholesky(S);
        if (rc) return rc;
    } else {
        for (int64_t i = 0; i < m; ++i) {
            double acc = 0.0;
            for (int32_t k = S->row_ptr[i]; k < S->row_ptr[i + 1]; ++k) acc += S->val_hat[k] * S->val_hat[k];
            if (!(acc > 0.0)) return 3;                        /* empty row */
            S->jac[i] = acc;
        }
    }
    /* step 13: d = (AO)^dagger b + (mu/2)(abs_{A_hat}(O'c) - O'c)   [P:237-238, Alg.1 step 2 P:66] */
    double *t1 = (double *)malloc(sizeof(double) * (size_t)n), *t2 = (double *)malloc(sizeof(double) * (size_t)n);
    double *w1 = (double *)malloc(sizeof(double) * (size_t)m), *w2 = (double *)malloc(sizeof(double) * (size_t)m);
    apply_pinv(S, S->b, w1, t1);                               /* (AO)^dagger b, multiplier w1       */
    abs_range(S, S->c_hat, w2, t2);                            /* abs(c_hat),    multiplier w2       */
    for (int64_t j = 0; j < n; ++j) S->d[j] = t1[j] + 0.5 * S->mu * (t2[j] - S->c_hat[j]);
    /* d = A_hat'(w1 + mu w2) - mu c_hat  => multiplier behind d (used only for the derived y) */
    for (int64_t i = 0; i < m; ++i) S->w_d[i] = w1[i] + S->mu * w2[i];
    free(t1); free(t2); free(w1); free(w2);
    /* step 14: s = O^{-1} x - mu O z   [P:239-240] */
    for (int64_t j = 0; j < n; ++j) S->s[j] = S->x[j] / S->O[j] - S->mu * S->O[j] * S->z[j];
    S->n_cond += 1;
    return 0;
}

/* Algorithm 2, steps 5-11: o per cone from the current (x,z), then O = o^alpha   [P:222-234] */
static void conditioning_rule(orc_solver *S) {
    double *o = S->O;                                          /* filled with o first, then O */
    double omax = 0.0, omin = 0.0;
    int first = 1;
    int64_t h = 0;
    const int64_t n_cones = S->n_lin + S->n_soc;
    for (int64_t i = 0; i < n_cones; ++i) {
        int64_t ni = (i < S->n_lin) ? 1 : S->soc_size[i - S->n_lin];
        double tail = 0.0;
        for (int64_t j = h + 1; j < h + ni; ++j) tail += S->x[j] * S->x[j];
        double num = fabs(S->x[h] - sqrt(tail));               /* |x_{h+1} - ||x_{h+2..h+n_i}||_2|  [P:228] */
        double den = fabs(S->z[h]);                            /* |z_{h+1}|                          */
        if (num < S->o_floor) num = S->o_floor;                /* reading (g): floor both            */
        if (den < S->o_floor) den = S->o_floor;
        double oi = num / den;
        for (int64_t j = h; j < h + ni; ++j) o[j] = oi;        /* steps 6-8: same value over the block */
        if (first || oi > omax) omax = oi;
        if (first || oi < omin) omin = oi;
        first = 0;
        h += ni;
    }
    /* step 11: O = diag{|o|}^min{1, t/(log max o - log min o)}   [P:234] */
    double spread = log(omax) - log(omin);
    double alpha = (spread <= S->t) ? 1.0 : S->t / spread;
    for (int64_t j = 0; j < S->n; ++j) S->O[j] = exp(alpha * log(o[j]));
}

/* Algorithm 2, steps 16-20: one pass   [P:243-249] */
static void one_pass(orc_solver *S) {
    const int64_t n = S->n;
    /* 16: p = abs_{O^{-1}K}(s) = abs_K(s)  (O is a positive multiple of I on each block) */
    orc_abs_cone(S->s, S->p, S->n_lin, S->n_soc, S->soc_size);
    /* 17: r = abs_{A_hat}(p) */
    abs_range(S, S->p, S->w, S->r);
    /* 18: s = s/2 - r/2 + d */
    double dd = 0.0;
    for (int64_t j = 0; j < n; ++j) {
        double s_new = S->s[j] / 2.0 - S->r[j] / 2.0 + S->d[j];
        dd += (s_new - S->s[j]) * (s_new - S->s[j]);
        S->s[j] = s_new;
    }
    S->fp_res = sqrt(dd);
    /* 19: x = O(p+s)/2 ; 20: z = O^{-1}(p-s)/(2 mu) */
    for (int64_t j = 0; j < n; ++j) {
        S->x[j] = S->O[j] * (S->p[j] + S->s[j]) / 2.0;
        S->z[j] = (S->p[j] - S->s[j]) / (2.0 * S->mu) / S->O[j];
    }
}

/* Algorithm 2 main loop, k_iter more passes; L = sorted list of conditioning iterations.
 * Step 4: condition when l in L u {1}   [P:216-254].  Returns 0, or a non-zero solve error. */
int orc_run(orc_solver *S, int64_t k_iter, const int64_t *L, int64_t nL) {
    for (int64_t it = 0; it < k_iter; ++it) {
        S->l += 1;                                             /* step 3 */
        int in_L = (S->l == 1);
        for (int64_t q = 0; q < nL; ++q) if (L[q] == S->l) in_L = 1;
        if (in_L) {                                            /* step 4 */
            conditioning_rule(S);                              /* steps 5-11 */
            int rc = apply_scaling(S);                         /* steps 12-14 */
            if (rc) return rc;
        }
        one_pass(S);                                           /* steps 16-20 */
    }
    return 0;
}

/* Step 4 with a "user-defined criteria" instead of a set L [P:295]: the paper leaves the criterion
 * open; the reading taken here (reading (y)) is a stall test on the fixed-point residual
 * f_l = ||s_l - s_{l-1}||_2 of pass l:
 *     condition at the start of iteration l > 1  iff  (l-1) is a multiple of `window`
 *                                               and  f_{l-1} > ratio * f_{l-1-lag}
 *                                               and  f_{l-1} > f_floor
 * with 1 <= lag < window, so that both residuals were measured after the previous conditioning (which
 * can only have happened at the start of iteration l-window or earlier) and therefore in the same
 * scaled space; f_floor keeps a run that has converged to rounding noise from conditioning on noise.
 * Iteration 1 always conditions (L u {1}).  f_hist[l] must hold max(l)+1 doubles
 * (f_hist[0] unused); cond_iters receives the iterations that conditioned (at most cap of them).
 * Returns the number of conditionings of this call, or -1 on a solve error. */
int64_t orc_run_stall(orc_solver *S, int64_t k_iter, int64_t window, int64_t lag, double ratio, double f_floor,
                      double *f_hist, int64_t *cond_iters, int64_t cap) {
    int64_t n_c = 0;
    if (window < 2 || lag < 1 || lag >= window) return -1;
    for (int64_t it = 0; it < k_iter; ++it) {
        S->l += 1;                                             /* step 3 */
        const int64_t l = S->l;
        int cond = (l == 1);
        if (l > 1 && (l - 1) % window == 0 && f_hist[l - 1] > ratio * f_hist[l - 1 - lag] &&
            f_hist[l - 1] > f_floor) cond = 1;
        if (cond) {                                            /* step 4 */
            conditioning_rule(S);                              /* steps 5-11 */
            if (apply_scaling(S)) return -1;                   /* steps 12-14 */
            if (n_c < cap) cond_iters[n_c] = l;
            n_c += 1;
        }
        one_pass(S);                                           /* steps 16-20 */
        f_hist[l] = S->fp_res;
    }
    return n_c;
}

/* Fixed equilibration, the practice the paper argues against [P:130-132: "matrix equilibration
 * heuristics such as Sinkhorn-Knopp and Ruiz methods ... equalizing l_p norm for each row through
 * diagonal choices of D and E"; P:148-152 uses the l_2 norms].  The paper gives no listing; this is
 * Ruiz's simultaneous square-root iteration in the l_2 norm (reading (z)):
 *     B = D A E ;  r_i = ||row_i(B)||_2 ;  c_j = ||col_j(B)||_2
 *     D_i <- D_i / sqrt(r_i) ;  E_j <- E_j / sqrt(c_j / tau) ,  tau = sqrt(m/n)
 * (rows are driven to norm 1 and columns to norm tau: sum r_i^2 = sum c_j^2 forces m = n tau^2).
 * E has to commute with the cone [P:122-126 E^{-1}K = K], i.e. be constant on a Lorentz block: c_j^2
 * is replaced by its mean over the block.  Empty rows / columns keep their factor.  D is returned
 * for the pins only: abs_{A_hat} does not depend on a row scaling (D^AC = I). */
void orc_ruiz(const orc_solver *S, int64_t n_iter, double *D, double *E) {
    const int64_t m = S->m, n = S->n;
    const double tau = sqrt((double)m / (double)n);
    double *r2 = (double *)malloc(sizeof(double) * (size_t)(m > 0 ? m : 1));
    double *c2 = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    for (int64_t i = 0; i < m; ++i) D[i] = 1.0;
    for (int64_t j = 0; j < n; ++j) E[j] = 1.0;
    for (int64_t it = 0; it < n_iter; ++it) {
        for (int64_t j = 0; j < n; ++j) c2[j] = 0.0;
        for (int64_t i = 0; i < m; ++i) {
            double acc = 0.0;
            for (int64_t q = S->row_ptr[i]; q < S->row_ptr[i + 1]; ++q) {
                const int64_t j = S->col_idx[q];
                const double bij = D[i] * S->val[q] * E[j];
                acc += bij * bij;
                c2[j] += bij * bij;
            }
            r2[i] = acc;
        }
        int64_t a = S->n_lin;                                  /* block means over the Lorentz cones */
        for (int64_t k = 0; k < S->n_soc; ++k) {
            const int64_t sz = S->soc_size[k];
            double mean = 0.0;
            for (int64_t j = a; j < a + sz; ++j) mean += c2[j];
            mean /= (double)sz;
            for (int64_t j = a; j < a + sz; ++j) c2[j] = mean;
            a += sz;
        }
        for (int64_t i = 0; i < m; ++i) if (r2[i] > 0.0) D[i] /= sqrt(sqrt(r2[i]));
        for (int64_t j = 0; j < n; ++j) if (c2[j] > 0.0) E[j] /= sqrt(sqrt(c2[j]) / tau);
    }
    free(r2); free(c2);
}

/* ------------------------------------------------------------------------------------------ */
/* handle management and accessors (plumbing)                                                  */
/* ------------------------------------------------------------------------------------------ */
static double *dalloc(int64_t k) { return (double *)calloc((size_t)(k > 0 ? k : 1), sizeof(double)); }

void orc_destroy(orc_solver *S) {
    if (!S) return;
    free(S->row_ptr); free(S->col_idx); free(S->val); free(S->val_hat); free(S->b); free(S->c); free(S->c_hat);
    free(S->soc_size); free(S->O); free(S->d); free(S->s); free(S->p); free(S->r); free(S->x); free(S->z);
    free(S->w); free(S->w_d); free(S->chol); free(S->jac);
    free(S);
}

/* solve_mode: 0 = auto (Cholesky when m <= 2000), 1 = Cholesky, 2 = Jacobi-PCG.
 * Initial point: x = z = e_K (1 on every cone's first coordinate, 0 elsewhere) => o = 1, O = I, s = 0
 * (reading (j); the paper only says "initial points x, z" P:214-215). */
orc_solver *orc_create(int64_t m, int64_t n, const int32_t *row_ptr, const int32_t *col_idx, const double *val,
                       const double *b, const double *c, int64_t n_lin, int64_t n_soc, const int32_t *soc_size,
                       double mu, double t, double o_floor, int solve_mode, double pcg_tol, int64_t pcg_max) {
    orc_solver *S = (orc_solver *)calloc(1, sizeof(orc_solver));
    if (!S) return NULL;
    int64_t nnz = row_ptr[m], tot = n_lin;
    for (int64_t i = 0; i < n_soc; ++i) tot += soc_size[i];
    if (tot != n || mu <= 0.0 || t <= 0.0) { free(S); return NULL; }
    S->m = m; S->n = n; S->nnz = nnz; S->n_lin = n_lin; S->n_soc = n_soc;
    S->mu = mu; S->t = t; S->o_floor = o_floor; S->pcg_tol = pcg_tol; S->pcg_max = pcg_max;
    S->solve_mode = solve_mode ? solve_mode : (m <= 2000 ? 1 : 2);
    S->row_ptr = (int32_t *)malloc(sizeof(int32_t) * (size_t)(m + 1));
    S->col_idx = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nnz > 0 ? nnz : 1));
    S->soc_size = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_soc > 0 ? n_soc : 1));
    S->val = dalloc(nnz); S->val_hat = dalloc(nnz); S->b = dalloc(m); S->c = dalloc(n); S->c_hat = dalloc(n);
    S->O = dalloc(n); S->d = dalloc(n); S->s = dalloc(n); S->p = dalloc(n); S->r = dalloc(n);
    S->x = dalloc(n); S->z = dalloc(n); S->w = dalloc(m); S->w_d = dalloc(m);
    S->chol = (S->solve_mode == 1) ? dalloc(m * m) : NULL;
    S->jac = dalloc(m);
    memcpy(S->row_ptr, row_ptr, sizeof(int32_t) * (size_t)(m + 1));
    memcpy(S->col_idx, col_idx, sizeof(int32_t) * (size_t)nnz);
    memcpy(S->val, val, sizeof(double) * (size_t)nnz);
    memcpy(S->b, b, sizeof(double) * (size_t)m);
    memcpy(S->c, c, sizeof(double) * (size_t)n);
    if (n_soc) memcpy(S->soc_size, soc_size, sizeof(int32_t) * (size_t)n_soc);
    for (int64_t j = 0; j < n; ++j) S->O[j] = 1.0;
    int64_t h = n_lin;
    for (int64_t j = 0; j < n_lin; ++j) { S->x[j] = 1.0; S->z[j] = 1.0; }
    for (int64_t i = 0; i < n_soc; ++i) { S->x[h] = 1.0; S->z[h] = 1.0; h += soc_size[i]; }
    return S;
}

/* starting point of Algorithm 2 (input line); only meaningful before the first pass */
void orc_set_point(orc_solver *S, const double *x, const double *z) {
    memcpy(S->x, x, sizeof(double) * (size_t)S->n);
    memcpy(S->z, z, sizeof(double) * (size_t)S->n);
}

/* Fix the diagonal O by hand (a FIXED preconditioner E of eq.(4)-(5)) and run steps 12-14
 * from the current (x,z).  Marks iteration 1's mandatory conditioning as done when l == 0 by
 * advancing nothing: the caller then uses orc_run_fixed. */
int orc_set_scaling(orc_solver *S, const double *O) {
    memcpy(S->O, O, sizeof(double) * (size_t)S->n);
    return apply_scaling(S);
}

/* k_iter passes of steps 16-20 with O left as it is (Algorithm 1 on the scaled data) */
void orc_run_fixed(orc_solver *S, int64_t k_iter) {
    for (int64_t it = 0; it < k_iter; ++it) { S->l += 1; one_pass(S); }
}

/* any pointer may be NULL */
void orc_get(const orc_solver *S, double *x, double *z, double *y, double *s, double *O, double *p, double *d) {
    size_t nb = sizeof(double) * (size_t)S->n;
    if (x) memcpy(x, S->x, nb);
    if (z) memcpy(z, S->z, nb);
    if (s) memcpy(s, S->s, nb);
    if (O) memcpy(O, S->O, nb);
    if (p) memcpy(p, S->p, nb);
    if (d) memcpy(d, S->d, nb);
    if (y) for (int64_t i = 0; i < S->m; ++i) y[i] = (S->w_d[i] - S->w[i]) / S->mu;   /* derived, see header */
}

void orc_counters(const orc_solver *S, int64_t out[6]) {
    out[0] = S->l; out[1] = S->n_cond; out[2] = S->pcg_steps_total; out[3] = S->pcg_steps_last;
    out[4] = S->solve_mode; out[5] = S->pcg_fail;
}

/* building blocks exposed so that the tests can pin them one by one */
void orc_pinv_apply(orc_solver *S, const double *rhs_m, double *out_n) {       /* A_hat^dagger rhs */
    double *w = dalloc(S->m);
    apply_pinv(S, rhs_m, w, out_n);
    free(w);
}
void orc_abs_range(orc_solver *S, const double *v_n, double *out_n) {          /* abs_{A_hat}(v)  */
    double *w = dalloc(S->m);
    abs_range(S, v_n, w, out_n);
    free(w);
}
void orc_mat_vec(const orc_solver *S, const double *v_n, double *out_m) { mat_vec(S, S->val_hat, v_n, out_m); }
void orc_mat_tvec(const orc_solver *S, const double *y_m, double *out_n) { mat_tvec(S, S->val_hat, y_m, out_n); }

/* ------------------------------------------------------------------------------------------ */
/* KKT residuals in the ORIGINAL coordinates (the conditions (24),(34) P:480-487).  */
/* The paper's own stop rule (16) P:330-338 is relative to a competing solver; this relative    */
/* form is the build's definition:                                                  */
/*   out[0] pres_abs = ||Ax-b||_2            out[1] pres_rel = pres_abs/(1+||b||_2)             */
/*   out[2] dres_abs = ||c-z-A'y||_2         out[3] dres_rel = dres_abs/(1+||c||_2)             */
/*   out[4] gap_abs  = |c'x-b'y|             out[5] gap_rel  = gap_abs/(1+|c'x|+|b'y|)          */
/*   out[6] cone_viol_rel = (||x-proj_K x||+||z-proj_K z||)/(1+||x||+||z||)                     */
/*   out[7] kkt_rel = max(out[1],out[3],out[5],out[6])   out[8] c'x   out[9] b'y   out[10] fp_res */
/* ------------------------------------------------------------------------------------------ */
static double norm2(const double *v, int64_t k) {
    double acc = 0.0;
    for (int64_t j = 0; j < k; ++j) acc += v[j] * v[j];
    return sqrt(acc);
}

void orc_residuals(const orc_solver *S, double out[11]) {
    const int64_t m = S->m, n = S->n;
    double *y = dalloc(m), *Ax = dalloc(m), *Aty = dalloc(n), *t = dalloc(n);
    for (int64_t i = 0; i < m; ++i) y[i] = (S->w_d[i] - S->w[i]) / S->mu;
    mat_vec(S, S->val, S->x, Ax);
    mat_tvec(S, S->val, y, Aty);
    double pres = 0.0, dres = 0.0, cx = 0.0, by = 0.0;
    for (int64_t i = 0; i < m; ++i) { pres += (Ax[i] - S->b[i]) * (Ax[i] - S->b[i]); by += S->b[i] * y[i]; }
    for (int64_t j = 0; j < n; ++j) {
        double e = S->c[j] - S->z[j] - Aty[j];
        dres += e * e;
        cx += S->c[j] * S->x[j];
    }
    pres = sqrt(pres); dres = sqrt(dres);
    double vx = 0.0, vz = 0.0;
    orc_proj_cone(S->x, t, S->n_lin, S->n_soc, S->soc_size);
    for (int64_t j = 0; j < n; ++j) vx += (S->x[j] - t[j]) * (S->x[j] - t[j]);
    orc_proj_cone(S->z, t, S->n_lin, S->n_soc, S->soc_size);
    for (int64_t j = 0; j < n; ++j) vz += (S->z[j] - t[j]) * (S->z[j] - t[j]);
    out[0] = pres; out[1] = pres / (1.0 + norm2(S->b, m));
    out[2] = dres; out[3] = dres / (1.0 + norm2(S->c, n));
    out[4] = fabs(cx - by); out[5] = out[4] / (1.0 + fabs(cx) + fabs(by));
    out[6] = (sqrt(vx) + sqrt(vz)) / (1.0 + norm2(S->x, n) + norm2(S->z, n));
    double k = out[1];
    if (out[3] > k) k = out[3];
    if (out[5] > k) k = out[5];
    if (out[6] > k) k = out[6];
    out[7] = k; out[8] = cx; out[9] = by; out[10] = S->fp_res;
    free(y); free(Ax); free(Aty); free(t);
}
