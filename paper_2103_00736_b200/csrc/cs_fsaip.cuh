// cs_fsaip.cuh -- FSAI(P): factorised sparse approximate inverse of M = A~A~' (unit diagonal) with up to kFsP off-diagonal
// entries per row (cs_params.precond = 3; S 8(f).1 "better inner preconditioner").  G is lower triangular in the internal
// row order; row i's pattern S_i = {partners} + {i}, the partners being the kFsP rows k < i with the largest |M_ik| among
// the kFsTop strongest short rows of row i's kFsC strongest columns; g_i = M[S_i,S_i]^-1 e_i / sqrt((M[S_i,S_i]^-1)_ii), so
// that G M G' has unit diagonal and CG runs with z = G'(G r).  Like FSAI(1) the pattern depends on the scaled values, so it
// is rebuilt ON THE DEVICE inside k_condition.  Measured on CPU replicas of config 4 after continuous conditioning:
// Jacobi 3906 PCG steps, FSAI(1) 1309, FSAI(3) 975, FSAI(5) 707.  It changes the number of CG steps, not the solution.
//
// Storage (struct-of-arrays, coalesced over rows): fp_idx[p][m] partner (or -1), fp_val[p][m] its coefficient, fp_val[kFsP][m]
// the diagonal; transposed lists for the G' pass: fp_tptr[m+1], fp_tcnt[m] (kept entries), fp_trow / fp_tval.
// Bounds on one thread's serial work: rows longer than kShortMax and columns longer than kFsaiColMax take no part, and a
// row keeps at most kFsaiListMax of the rows that chose it (the smallest indices; the others drop that partner).
#pragma once
#include "cs_kernels.cuh"

namespace csd {

constexpr int kFsP = 5, kFsC = 3, kFsTop = 6;
constexpr int kFsColMax = 64, kFsListMax = 32;

// <row i, row k> over the row-major compressed view (entries of a short row are in no particular order)
__device__ __forceinline__ double fsp_row_dot(const Ctx &c, int i, int k) {
    const int a0 = c.Rc.ptr[i], a1 = c.Rc.ptr[i + 1], b0 = c.Rc.ptr[k], b1 = c.Rc.ptr[k + 1];
    double s = 0.0;
    for (int e = a0; e < a1; ++e) {
        const int jj = c.Rc.idx[e];
        for (int f = b0; f < b1; ++f)
            if (c.Rc.idx[f] == jj) { s += c.R.val[c.Rc.pos[e]] * c.R.val[c.Rc.pos[f]]; break; }
    }
    return s;
}

// pattern and coefficients of row i (a short row); returns the number of partners, sel[] ascending, g[0..np) theirs, g[np] diagonal
__device__ __forceinline__ int fsp_row(const Ctx &c, int i, int (&sel)[kFsP], double (&g)[kFsP + 1]) {
    const int a0 = c.Rc.ptr[i], a1 = c.Rc.ptr[i + 1];
    int jc[kFsC];
    double jv[kFsC];
#pragma unroll
    for (int q = 0; q < kFsC; ++q) { jc[q] = -1; jv[q] = -1.0; }
    for (int e = a0; e < a1; ++e) {                              // the kFsC strongest columns of the row
        double a = fabs(c.R.val[c.Rc.pos[e]]);
        int j = c.Rc.idx[e];
#pragma unroll
        for (int q = 0; q < kFsC; ++q)
            if (a > jv[q]) { const double ta = jv[q]; const int tj = jc[q]; jv[q] = a; jc[q] = j; a = ta; j = tj; }
    }
    int cand[kFsC * kFsTop], nc = 0;
    for (int q = 0; q < kFsC; ++q) {
        if (jc[q] < 0) continue;
        for (int t = 0; t < kFsTop; ++t) {
            const int k = c.fp_ctop[kFsTop * jc[q] + t];
            if (k < 0 || k >= i) continue;
            bool dup = false;
            for (int u = 0; u < nc; ++u) dup |= cand[u] == k;
            if (!dup) cand[nc++] = k;
        }
    }
    // the kFsP candidates with the largest |mu| (ties: the smaller row index, so that the choice is deterministic)
    double mu[kFsP];
    int np = 0;
    for (int u = 0; u < nc; ++u) {
        double v = fsp_row_dot(c, i, cand[u]);
        int k = cand[u];
        if (!(fabs(v) > 1e-12)) continue;
        for (int q = 0; q < np; ++q)
            if (fabs(v) > fabs(mu[q]) || (fabs(v) == fabs(mu[q]) && k < sel[q])) {
                const double tv = mu[q]; const int tk = sel[q]; mu[q] = v; sel[q] = k; v = tv; k = tk;
            }
        if (np < kFsP) { mu[np] = v; sel[np] = k; ++np; }
    }
    for (int a = 1; a < np; ++a) {                               // ascending row index
        const int k = sel[a]; const double v = mu[a];
        int b = a - 1;
        while (b >= 0 && sel[b] > k) { sel[b + 1] = sel[b]; mu[b + 1] = mu[b]; --b; }
        sel[b + 1] = k; mu[b + 1] = v;
    }
    // Gram matrix of S_i (lower triangle), Cholesky, g = L^-T e_last * L_last,last
    double L[(kFsP + 1) * (kFsP + 1)];
    const int ns = np + 1;
    for (int a = 0; a < np; ++a) {
        for (int b = 0; b < a; ++b) L[a * ns + b] = fsp_row_dot(c, sel[a], sel[b]);
        L[a * ns + a] = fsp_row_dot(c, sel[a], sel[a]);
        L[np * ns + a] = mu[a];
    }
    L[np * ns + np] = fsp_row_dot(c, i, i);
    bool ok = true;
    for (int a = 0; a < ns && ok; ++a) {
        for (int b = 0; b <= a; ++b) {
            double s = L[a * ns + b];
            for (int q = 0; q < b; ++q) s -= L[a * ns + q] * L[b * ns + q];
            if (a == b) { if (!(s > 1e-10)) { ok = false; break; } L[a * ns + a] = sqrt(s); }
            else L[a * ns + b] = s / L[b * ns + b];
        }
    }
    if (!ok) { g[0] = 1.0; return 0; }                           // numerically dependent rows: no partners for this row
    // y = L^-T u with u = e_last / L_nn; g = y * L_nn  =>  g_last = 1 / L_nn, g_a = -(sum_{b>a} L[b][a] g_b) / L[a][a]
    g[np] = 1.0 / L[np * ns + np];
    for (int a = np - 1; a >= 0; --a) {
        double s = 0.0;
        for (int b = a + 1; b < ns; ++b) s += L[b * ns + a] * g[b];
        g[a] = -s / L[a * ns + a];
    }
    return np;
}

__device__ __forceinline__ void fsaip_build(const Ctx &c, GridCtl &gc) {
    const int tid = blockIdx.x * kBlock + threadIdx.x, nth = gridDim.x * kBlock, m = c.m;
    // P1: the kFsTop strongest short rows of every column (columns longer than kFsColMax propose nothing)
    for (int j = tid; j < c.n; j += nth) {
        int bi[kFsTop];
        double bv[kFsTop];
#pragma unroll
        for (int q = 0; q < kFsTop; ++q) { bi[q] = -1; bv[q] = -1.0; }
        const int ce = c.Cc.ptr[j + 1] - c.Cc.ptr[j] <= kFsColMax ? c.Cc.ptr[j + 1] : c.Cc.ptr[j];
        for (int e = c.Cc.ptr[j]; e < ce; ++e) {
            int i = c.Cc.idx[e];
            if (i < c.n_long) continue;
            double a = fabs(c.C.val[c.Cc.pos[e]]);
#pragma unroll
            for (int q = 0; q < kFsTop; ++q)
                if (a > bv[q]) { const double ta = bv[q]; const int ti = bi[q]; bv[q] = a; bi[q] = i; a = ta; i = ti; }
        }
#pragma unroll
        for (int q = 0; q < kFsTop; ++q) c.fp_ctop[kFsTop * j + q] = bi[q];
    }
    for (int i = tid; i < m; i += nth) c.fp_tcnt[i] = 0;
    gc.sync();
    // P2: pattern and coefficients per row; count the transposed lists
    for (int i = tid; i < m; i += nth) {
        int sel[kFsP];
        double g[kFsP + 1];
        int np = 0;
        g[0] = 1.0;
        if (i >= c.n_long) np = fsp_row(c, i, sel, g);
#pragma unroll
        for (int q = 0; q < kFsP; ++q) {
            c.fp_idx[(size_t)q * m + i] = q < np ? sel[q] : -1;
            c.fp_val[(size_t)q * m + i] = q < np ? g[q] : 0.0;
        }
        c.fp_val[(size_t)kFsP * m + i] = g[np];
        for (int q = 0; q < np; ++q) atomicAdd(c.fp_tcnt + sel[q], 1);
    }
    gc.sync();
    // P3: exclusive scan of the counts -> fp_tptr (every CTA scans its own contiguous range; f_blk holds the CTA totals)
    const int per = (m + gridDim.x - 1) / gridDim.x, lo = min(m, (int)blockIdx.x * per), hi = min(m, lo + per);
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        int sum = 0;
        for (int i = lo + lane; i < hi; i += 32) sum += c.fp_tcnt[i];
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
        if (lane == 0) c.f_blk[blockIdx.x] = sum;
    }
    gc.sync();
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        int base = 0;
        for (int b = lane; b < (int)blockIdx.x; b += 32) base += c.f_blk[b];
        for (int o = 16; o > 0; o >>= 1) base += __shfl_xor_sync(0xffffffffu, base, o);
        for (int i0 = lo; i0 < hi; i0 += 32) {
            const int i = i0 + lane;
            const int cnt = i < hi ? c.fp_tcnt[i] : 0;
            int inc = cnt;
            for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
            if (i < hi) { c.fp_tptr[i] = base + inc - cnt; c.fp_tcnt[i] = 0; }
            base += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (lane == 0 && hi == m && lo < hi) c.fp_tptr[m] = base;
    }
    gc.sync();
    // P4: fill the lists (arrival order), then P5: order them by row and cap them
    for (int i = tid; i < m; i += nth)
        for (int q = 0; q < kFsP; ++q) {
            const int k = c.fp_idx[(size_t)q * m + i];
            if (k < 0) break;
            const int pos = c.fp_tptr[k] + atomicAdd(c.fp_tcnt + k, 1);
            c.fp_trow[pos] = i;
            c.fp_tval[pos] = c.fp_val[(size_t)q * m + i];
        }
    gc.sync();
    for (int k = tid; k < m; k += nth) {
        const int a = c.fp_tptr[k], b = c.fp_tptr[k + 1], keep = min(b - a, kFsListMax);
        for (int e = a; e < a + keep; ++e) {                     // selection sort of the `keep` smallest row indices
            int best = e, x = c.fp_trow[e];
            for (int f = e + 1; f < b; ++f) { const int y = c.fp_trow[f]; if (y < x) { x = y; best = f; } }
            const int tr = c.fp_trow[e]; const double tv = c.fp_tval[e];
            c.fp_trow[e] = c.fp_trow[best]; c.fp_tval[e] = c.fp_tval[best];
            c.fp_trow[best] = tr; c.fp_tval[best] = tv;
        }
        for (int e = a + keep; e < b; ++e) {                     // dropped: row i forgets partner k (G stays lower triangular, G'G SPD)
            const int i = c.fp_trow[e];
            for (int q = 0; q < kFsP; ++q)
                if (c.fp_idx[(size_t)q * m + i] == k) c.fp_val[(size_t)q * m + i] = 0.0;
        }
        c.fp_tcnt[k] = keep;
    }
}

// t = G r over rows [k_begin, m)
__device__ __forceinline__ void fsaip_pass_a(const Ctx &c, int k_begin) {
    const int tid = blockIdx.x * kBlock + threadIdx.x, nth = gridDim.x * kBlock, m = c.m;
    for (int k = k_begin + tid; k < m; k += nth) {
        int idx[kFsP];
        double val[kFsP], rv[kFsP];
#pragma unroll
        for (int q = 0; q < kFsP; ++q) { idx[q] = c.fp_idx[(size_t)q * m + k]; val[q] = c.fp_val[(size_t)q * m + k]; }
#pragma unroll
        for (int q = 0; q < kFsP; ++q) rv[q] = idx[q] >= 0 ? c.r[idx[q]] : 0.0;
        double acc = c.fp_val[(size_t)kFsP * m + k] * c.r[k];
#pragma unroll
        for (int q = 0; q < kFsP; ++q) acc += val[q] * rv[q];
        c.t1[k] = acc;
    }
}
// z = G' t over rows [k_begin, m); returns this thread's share of r'z
__device__ __forceinline__ double fsaip_pass_b(const Ctx &c, int k_begin) {
    const int tid = blockIdx.x * kBlock + threadIdx.x, nth = gridDim.x * kBlock, m = c.m;
    double rz = 0.0;
    for (int k = k_begin + tid; k < m; k += nth) {
        const int e0 = c.fp_tptr[k], e1 = e0 + c.fp_tcnt[k];
        double acc = c.fp_val[(size_t)kFsP * m + k] * c.t1[k];
        for (int e = e0; e < e1; ++e) acc += c.fp_tval[e] * c.t1[c.fp_trow[e]];
        c.z[k] = acc;
        rz += c.r[k] * acc;
    }
    return rz;
}

}  // namespace csd
