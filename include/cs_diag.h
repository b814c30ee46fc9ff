/*
 * cs_diag.h -- DIAGNOSTICS of libcs.so, not part of the product ABI of cs.h: instrumentation that
 * bench.py and profiles/ use to explain the numbers (per-phase device time of k_iterate, the gather ceiling of the
 * SM's load path, the latency of the grid barrier).  Nothing on the hot path depends on these calls.
 */
#ifndef CS_DIAG_H_
#define CS_DIAG_H_

#include "cs.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Device time per phase of k_iterate so far, in ns, measured on the device between grid barriers:
 * out[0] cone reflect, [1] rhs pass, [2] CG pass K1 (A~'r, columns), [3] CG pass K2 (A~u, rows),
 * [4] A~'w + s-update pass, [5] grid reductions/barriers, [6] preconditioner application z = G'G r, [7] reserved.  One D2H copy + sync. */
cs_status cs_diag_phase_times(cs_solver *S, double out[8]);

/* Diagnostic (no handle, current device, default stream, synchronous): time n_idx uniformly random 8-byte
 * gathers from an n_vec-element vector with the launch shape of the solver's sparse passes (indices
 * streamed, 8 gathers in flight per thread), and the same loop without the gathers.  The difference is the
 * LSU/L1TEX gather ceiling that bounds the sparse passes on irregular matrices. */
cs_status cs_diag_gather_probe(int64_t n_vec, int64_t n_idx, double *us_gather, double *us_stream_only);

/* cs_create with the layout build chosen by hand: build_mode 0 = as cs_create (on the device from 100,000 non-zeros on), 1 = on
 * the host, 2 = on the device (csrc/cs_build.cuh).  The two builds produce identical layouts; the GPU test compares them with */
cs_status cs_diag_create(cs_solver **out, const cs_csr *A, const double *b, const double *c, cs_mem vec_where, const cs_cones *K,
                         void *cuda_stream, int32_t build_mode);
/* ... FNV-1a digests of the handle's layout arrays (slices, indices, pristine values, chunk tables, compressed views, fusion
 * marks, permutations, b, c) and its counters, 32 words.  Synchronous, copies the arrays to the host: small problems only. */
cs_status cs_diag_layout_digest(cs_solver *S, uint64_t out[32]);

/* Diagnostic (no handle, current device, default stream, synchronous): L2 -> SM read bandwidth in GB/s -- `reps` passes
 * of 16-byte loads over a `bytes`-sized buffer that stays in L2 (choose bytes well below the 126 MB of L2), best of 4. */
cs_status cs_diag_l2_probe(int64_t bytes, int32_t reps, double *gbs);

/* Diagnostic: run n empty grid barriers (each a 1-value all-reduce over all CTAs, result checked) in one
 * launch and report the mean latency in microseconds.  Synchronous. */
cs_status cs_diag_barrier_probe(cs_solver *S, int32_t n, double *us_per_barrier);

#ifdef __cplusplus
}
#endif
#endif /* CS_DIAG_H_ */
