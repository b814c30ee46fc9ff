/*
 * cs.h -- C ABI of libcs.so: the B200 (sm_100a) hot path of arXiv 2103.00736, Algorithm 2
 * (operator-splitting conic solver with adaptive conditioning).
 *
 *      minimise c'x  s.t.  Ax = b,  x in K = R^{n_lin}_+ x K_{q_1} x ... x K_{q_k}      (1) PAPER.md:41-56
 *
 * Citations "P:<line>" refer to /root/reference/PAPER.md.  Every step of the path (sparse products,
 * cone reflections, the normal-equation solve hidden in A^dagger, the averaged update, residual norms,
 * the conditioning rescale) runs in CUDA kernels on ONE device; there is no CPU fallback.
 *
 * Conventions
 *   - All floating point is IEEE fp64.  Indices are int32, sizes int64.
 *   - Every array argument is a plain pointer; where an argument can be host or device memory the
 *     call takes a cs_mem tag saying which.  Host arrays may be pageable or pinned.
 *   - Ownership: the library copies what it needs during the call and never keeps a caller pointer.
 *     Outputs are written into caller-owned buffers.  The handle owns all its device memory.
 *   - A handle is bound to the device that is current at cs_create and to the CUDA stream passed
 *     there (NULL = legacy default stream).  It is not thread-safe.
 *   - Errors: every call returns a cs_status; nothing throws or aborts across the ABI.  The text of
 *     the last error of a handle is available from cs_last_error.
 *   - Calls are asynchronous on the handle's stream unless stated otherwise.
 */
#ifndef CS_H_
#define CS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cs_solver cs_solver; /* opaque */

typedef enum {
    CS_OK = 0,
    CS_EINVAL = 1, /* NULL / shape / unsorted or duplicate CSR indices / cone sizes do not sum to n / empty row */
    CS_ENOMEM = 2, /* host or device allocation failed                                                           */
    CS_ECUDA = 3,  /* a CUDA runtime call failed; text in cs_last_error                                          */
    CS_ESTATE = 4, /* call not valid in the current state                                                        */
    CS_ECGMAX = 5  /* an inner CG solve hit cg_max_iter since the last cs_residuals (not fatal)                  */
} cs_status;

typedef enum { CS_HOST = 0, CS_DEVICE = 1 } cs_mem;

/* A in CSR.  row_ptr[0] = 0, non-decreasing, row_ptr[m] = nnz; col_idx sorted and unique within a row;
 * every row must hold at least one entry (A is assumed to have full row rank: the proofs use
 * A A^dagger = I).  All three arrays live in the memory space named by `where`. */
typedef struct {
    int64_t m, n, nnz;
    const int32_t *row_ptr; /* [m+1] */
    const int32_t *col_idx; /* [nnz] */
    const double *val;      /* [nnz] */
    cs_mem where;
} cs_csr;

/* K: n_lin leading orthant coordinates (Lorentz cones of size 1) followed by n_soc Lorentz
 * cones of sizes soc_size[i] >= 1; n_lin + sum soc_size == n.  soc_size is a HOST array (may be NULL
 * when n_soc == 0). */
typedef struct {
    int64_t n_lin;
    int64_t n_soc;
    const int32_t *soc_size;
} cs_cones;

/* Parameters of Algorithm 2 (input line P:214-215) and of the inner solve.
 *   mu       fixed mu > 0; the experiments use 1
 *   t        cap on ln(max O / min O) in step 11; 9.2 for LP, 1.7 for SOCP
 *   o_floor  absolute floor of numerator and denominator of o_i in step 7 (paper silent on 0/0)
 *   cg_tol   inner solve stops when ||residual||_2 <= cg_tol * ||rhs||_2, both measured on the
 *            row-equilibrated system (D A_hat)(D A_hat)' with D = diag(1/||row_i(A_hat)||_2).  The residual is
 *            the recurrence residual of CG, which keeps shrinking below the rounding level of the true one; the
 *            default DBL_EPSILON = 2.22e-16 (the recurrence residual below one ulp of the right-hand side) takes the
 *            solve to that floor ("exact" projections, the parity setting: an in-run conditioning amplifies what is
 *            left of the solve error by 1e3-1e4)
 *   cg_reduce    inexact projections (0 = off, the default): the solve of a pass also stops once the residual of
 *            the WARM START has been reduced by this factor, ||residual||_2 <= max(cg_tol ||rhs||_2,
 *            cg_reduce ||residual at the warm start||_2).  The warm-start residual shrinks as the outer iteration
 *            converges (w converges to mu D^{-1} y), so the projection error shrinks with it -- an adaptive
 *            tolerance with the fixed point unchanged; 0 < cg_reduce < 1.
 *   cg_max_iter  cap on CG steps per solve
 *   precond  preconditioner of the inner CG beyond the Jacobi row equilibration: 0 = automatic (when t >= 4, i.e. when a
 *            conditioning may spread O^2 over many decades: FSAI(5) if the two matrix copies take 16-100 MB, else FSAI(1)),
 *            1 = none, 2 = FSAI(1): a sparse
 *            approximate inverse factor with one off-diagonal entry per row, 3 = FSAI(5): up to five per row
 *            (csrc/cs_fsaip.cuh; 35-55 % fewer CG steps than FSAI(1) on configs 1, 2 and on replicas of config 4, at
 *            3-4x the cost of its application: it pays on configs 1 and 2, not on the full-size config 4).
 *            Both are rebuilt on the device at every conditioning and change the number of CG steps, not
 *            the solution of the solve.
 *   dense_m_threshold  dense factor-apply instead of CG where A is small enough that the solve truly is a dense
 *            contraction (B north_star; S 8(a) a3, S 8(f).3), for m <= dense_m_threshold (<= 24576; 0 = never):
 *            - problems that run on one CTA (nnz <= 8192) with m <= 256: every conditioning forms A~A~' (m x m, fp64) and
 *              factors it by Cholesky in that CTA; every pass applies the factor (two triangular solves + one step of
 *              iterative refinement);
 *            - dense-STORED inputs (nnz >= m n / 2: the paper's own workloads, section V-A, V-D P:366-371) on
 *              many CTAs: every conditioning forms M = A~A~', its blocked Cholesky factor and the explicit inverse
 *              M^-1 = L^-T L^-1 (hand-written fp64 kernels, csrc/cs_dense.cuh); every pass is w += M^-1 r followed by one
 *              or two steps of iterative refinement against M (the second only when the first one's residual is not yet a
 *              hundred times below cg_tol, squared) -- dense matrix-vector products only.
 *              The limit 24576 covers the paper's largest dense LP (n = 30000, m = 24000); the path's buffers
 *              (A~ as [m][n] and four m x m matrices: 24 GB there) are allocated at the first conditioning that uses it,
 *              and if the device cannot hold them the solve stays with CG (not an error).
 *            No CG steps are counted.  Default: 128, or 24576 for a dense-stored input.  A Cholesky pivot below 1e-12
 *            (the diagonal of A~A~' is 1: numerically rank-deficient A) falls back to CG for that scaling.
 * cs_set_params may be called at any time; mu, t, o_floor, precond, dense_m_threshold take effect at the next
 * cs_condition (or at the implicit first conditioning), cg_* at the next solve. */
typedef struct {
    double mu, t, o_floor, cg_tol, cg_reduce;
    int32_t cg_max_iter;
    int32_t precond;
    int32_t dense_m_threshold;
    int32_t reserved;
} cs_params;

/* Residuals of the KKT conditions (24) P:480-487 in ORIGINAL coordinates, for the current iterate
 * x = O(p+s)/2, z = O^{-1}(p-s)/(2mu) (steps 19-20) and the derived multiplier y = D w/mu, where
 * w is the solution of the pass's single solve (A~A~') w = b~ - A~(p - mu c^):
 *   pres_abs = ||Ax-b||_2 (16a)      pres_rel = pres_abs/(1+||b||_2)
 *   dres_abs = ||c-z-A'y||_2                dres_rel = dres_abs/(1+||c||_2)
 *   gap_abs  = |c'x-b'y|  (cf. 16b)  gap_rel  = gap_abs/(1+|c'x|+|b'y|)
 *   cone_viol_rel = (||x-proj_K x||_2+||z-proj_K z||_2)/(1+||x||_2+||z||_2)
 *   kkt_rel  = max(pres_rel, dres_rel, gap_rel, cone_viol_rel)
 *   pobj = c'x, dobj = b'y, fp_res = ||s_new - s||_2 of the last pass (Lemma 3b). */
typedef struct {
    int64_t iter;           /* passes of steps 16-18 done so far (l of Algorithm 2) */
    int64_t cg_steps_total; /* CG steps over all solves so far                       */
    int64_t cg_steps_cond;  /* ... of which inside cs_condition (0: d is folded into the pass) */
    int32_t cg_steps_last;  /* CG steps of the most recent solve                     */
    int32_t n_conditionings;
    int32_t cg_hit_max;     /* 1 if some solve hit cg_max_iter since the last cs_residuals */
    int32_t dense_refine2;  /* passes so far whose dense factor-apply took its second refinement step (dense_m_threshold) */
    double pres_abs, pres_rel, dres_abs, dres_rel, gap_abs, gap_rel, cone_viol_rel, kkt_rel, pobj, dobj, fp_res;
} cs_resid;

/* Build a solver for (A,b,c,K): validates the input, copies it to the device, builds the CSC copy of A
 * and the work partitions.  b[m], c[n] live in `vec_where`.  Parameters start at mu=1, t=9.2 (n_soc=0)
 * or 1.7 (n_soc>0), o_floor=1e-16, cg_tol=2.22e-16 (DBL_EPSILON), cg_reduce=0, cg_max_iter=20000, precond=0,
 * dense_m_threshold=128 (24576 for a dense-stored A); the starting point is x=z=e_K (1 on each cone's first coordinate), which makes the
 * mandatory first conditioning (l=1) the identity and s=0.  Synchronous.  On failure *out is NULL. */
cs_status cs_create(cs_solver **out, const cs_csr *A, const double *b, const double *c, cs_mem vec_where,
                    const cs_cones *K, void *cuda_stream);

cs_status cs_set_params(cs_solver *S, const cs_params *p);
cs_status cs_get_params(const cs_solver *S, cs_params *p);

/* Starting point (x,z) of Algorithm 2, each [n] in `where`.  Only before the first
 * cs_iterate / cs_condition (else CS_ESTATE). */
cs_status cs_set_point(cs_solver *S, const double *x, const double *z, cs_mem where);

/* Optional warm start of the inner solve from a dual vector y[m] in `where` -- cs_solution's y of an earlier run (the
 * multiplier of Ax = b, y = (w_d - w)/mu; derived, S 8(c) reading (o)): the solve's unknown is w = mu D^-1 y in
 * the row scaling D of the moment, so a run resumed from (x, z, O) of a checkpoint (cs_set_point, cs_set_scaling) starts its
 * first solve where the checkpointed run's last one ended instead of at w = 0.  It changes the number of CG steps of the first
 * passes, not the iterates (the solve is exact, reading (s)); without it the start is w = 0.  Only before the first
 * cs_iterate / cs_condition / cs_set_scaling (else CS_ESTATE); uses the value of mu in force at the call. */
cs_status cs_set_dual(cs_solver *S, const double *y, cs_mem where);

/* k passes of steps 16-18: p = abs_K(s); r = abs_{A_hat}(p); s = s/2 - r/2 + d.
 * x,z of steps 19-20 are formed lazily by cs_condition / cs_residuals / cs_solution.  If no
 * conditioning has happened yet, the l=1 conditioning of step 4 runs first.  One kernel launch for
 * all k passes; no host synchronisation. */
cs_status cs_iterate(cs_solver *S, int64_t k);

/* Steps 5-14 from the current (x,z): o per cone, O = o^alpha, A_hat = D A O (D = row
 * equilibration, mathematically inert), c_hat = O c, and the recast s = O^{-1}x - mu O z.  Step 13's vector d
 * is folded into the pass (s+ = (s+p)/2 - mu c^ + A~'w), so a conditioning needs no linear solve.
 * The schedule L is the caller's: L = {300,400,...} is cs_iterate(299); cs_condition(); cs_iterate(100); ... */
cs_status cs_condition(cs_solver *S);

/* Replace step 5-11's rule by a caller-given positive diagonal O[n] (a FIXED preconditioner E of
 * eq.(4)-(5)), then steps 12-14.  Block-constant O is the caller's responsibility. */
cs_status cs_set_scaling(cs_solver *S, const double *O, cs_mem where);

/* Fixed equilibration: n_sweeps of Ruiz's simultaneous square-root iteration in the l2 norm on the pristine A
 * (the practice of P:130-132, "equalizing l_p norm for each row through diagonal choices of D and E"; l2 as
 * in P:148-152), entirely on the device:  B = D A E;  D_i <- D_i / sqrt(||row_i(B)||_2);
 * E_j <- E_j / sqrt(||col_j(B)||_2 / sqrt(m/n)), the squared column norms averaged over a Lorentz block so
 * that E commutes with K.  Then O := E is installed exactly as cs_set_scaling does (steps
 * 12-14).  This is the "fixed-scaling run" comparator of Algorithm 2; D is inert for the method.
 * n_sweeps >= 0 (0 installs O = I).  One kernel launch + the conditioning launch, no host synchronisation. */
cs_status cs_equilibrate(cs_solver *S, int32_t n_sweeps);

/* Step 4 of Algorithm 2 as a whole-run driver ("Adaptive conditioning can be done based
 * on a user-defined criteria or in the simplest case, at a set of user-defined iterations L").
 *   rule CS_RULE_SET   : L = {first, first+every, first+2*every, ...}  (eq.(17): 300,100; eq.(18): 200,100;
 *                        first <= 0: L empty; every <= 0: L = {first}).
 *   rule CS_RULE_STALL : with f_l = ||s_l - s_{l-1}||_2 the fixed-point residual of pass l, condition at the
 *                        start of iteration l > 1 iff (l-1) is a multiple of `window` and
 *                        f_{l-1} > ratio * f_{l-1-lag}  and  f_{l-1} > f_floor   (1 <= lag < window; both
 *                        residuals belong to the current scaling; f_floor keeps a converged run from
 *                        conditioning on rounding noise).  Costs two 8-byte read-backs per window.
 * Iteration 1 always conditions (L u {1}).  l is the handle's pass counter (cs_resid.iter), so calls
 * can be chained; the stall rule's lagged residual does not carry over from one call to the next (the first
 * window of a call that starts off a window boundary takes no decision).
 * Stops after max_iter passes, or earlier at the first multiple of check_every (> 0) where kkt_rel <= tol
 * (tol <= 0: never).  *out gets the residuals of the final iterate.  cond_iters (may be NULL) receives the
 * iterations that conditioned, at most cond_cap of them; *n_cond (may be NULL) their number.
 * Synchronous.  Returns CS_ECGMAX like cs_residuals. */
enum { CS_RULE_SET = 0, CS_RULE_STALL = 1 };
typedef struct {
    int64_t max_iter, check_every;
    double tol;
    int32_t rule, reserved;
    int64_t first, every;      /* CS_RULE_SET   */
    int64_t window, lag;       /* CS_RULE_STALL */
    double ratio, f_floor;
} cs_schedule;
cs_status cs_solve(cs_solver *S, const cs_schedule *sch, cs_resid *out, int64_t *cond_iters, int64_t cond_cap,
                   int64_t *n_cond);

/* Residual norms of the current iterate; ONE device->host copy and a stream synchronisation.
 * Returns CS_ECGMAX (with *out filled) if a solve hit cg_max_iter since the previous call. */
cs_status cs_residuals(cs_solver *S, cs_resid *out);

/* Copy out the current x[n], z[n], y[m], s[n], O[n] (original coordinates for x,z,y; scaled for s).
 * Any pointer may be NULL.  Synchronous when where == CS_HOST. */
cs_status cs_solution(cs_solver *S, double *x, double *z, double *y, double *s, double *O, cs_mem where);

/* The ONE entry point that allocates nothing -- no handle, no cudaMalloc/cudaFree, no allocating library routine --
 * for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid it): the cone
 * part of the residual norms (a6; P:566-572 x in K, z in K) of a caller-held iterate,
 *     out[0] = ||x - proj_K x||_2   out[1] = ||z - proj_K z||_2   out[2] = ||x||_2   out[3] = ||z||_2
 *     out[4] = cone_viol_rel = (out[0] + out[1]) / (1 + out[2] + out[3])          (cs_resid.cone_viol_rel)
 * x_dev, z_dev: DEVICE arrays [n] in the caller's order (orthant coordinates first, then the Lorentz blocks of K);
 * out: 5 doubles in `out_where` (CS_HOST: synchronous; CS_DEVICE: asynchronous on `cuda_stream`).
 * Its scratch (cone offsets, per-CTA partial sums) is a file-scope device array of 145 KB that every GPU loading the
 * library holds until exit; hence the LIMIT K->n_soc <= 32768 Lorentz cones (any n_lin, n < 2^31), beyond which the
 * call returns CS_EINVAL with the limit in cs_last_error(NULL).  All calls share that array: calls that overlap on
 * the GPU (other streams, other host threads) race -- serialise them.  Runs on the current device. */
cs_status cs_cone_violation_static(const double *x_dev, const double *z_dev, int64_t n, const cs_cones *K, double *out,
                                   cs_mem out_where, void *cuda_stream);

/* Number of kernels the library has launched on this handle so far (for bench accounting). */
int64_t cs_kernel_launches(const cs_solver *S);

const char *cs_last_error(const cs_solver *S);
void cs_destroy(cs_solver *S);

#ifdef __cplusplus
}
#endif
#endif /* CS_H_ */
