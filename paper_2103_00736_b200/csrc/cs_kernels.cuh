// cs_kernels.cuh -- the persistent cooperative kernels of libcs.so.
//
//   k_iterate   : k passes of Algorithm 2 steps 16-18 incl. the inner CG on (A~ A~')
//   k_condition : Algorithm 2 steps 5-14; step 13's d is folded into the pass, so no solve here
//   k_residuals : KKT residual norms of the current iterate
//
// A~ = D A O is the row-equilibrated, column-conditioned matrix; D = diag(1/||row_i(A O)||_2) is
// mathematically inert for the iterates ((DA)^dagger(DA) = A^dagger A) and makes diag(A~A~') = I,
// i.e. it IS the Jacobi preconditioner in split form.
#pragma once
#include "cs_device.cuh"
#include "cs_dense.cuh"

namespace csd {

// ---------------------------------------------------------------------------------------------
// Lorentz blocks by size class (B north_star: "one warp or CTA per cone chosen by block size"; S 8(a) a1):
//   small  (<= kConeSmall entries)  : kConeLanes = 8 lanes per block, 4 blocks per warp
//   medium (<= kConeMedium entries) : one warp per block
//   large                           : one CTA per block (block-wide sum through shared memory)
// c.cone_cls lists the cone ids class by class (cs_create).  `sum(j, is_head, t)` adds coordinate j's contribution to
// the double2 t; `apply(a, b, t, l, W)` is then called by all W lanes/threads of the group (l = 0..W-1) with the
// complete sums of block [a, b).  All sums have a fixed order.  Every thread of the grid must call this together.
// ---------------------------------------------------------------------------------------------
template <class Sum, class Apply>
__device__ __forceinline__ void cone_sweep(const Ctx &c, Sum sum, Apply apply) {
    const int tid = blockIdx.x * kBlock + threadIdx.x, nth = gridDim.x * kBlock, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gwarp = tid >> 5, nwarps = nth >> 5;
    {   // small
        const int sub = lane / kConeLanes, sl = lane % kConeLanes;
        constexpr int CPW = 32 / kConeLanes;
        for (int base = gwarp * CPW; base < c.n_cone_small; base += nwarps * CPW) {
            const int q = base + sub;
            const bool act = q < c.n_cone_small;
            const int ci = act ? __ldg(c.cone_cls + q) : 0;
            const int a = act ? __ldg(c.cone_off + ci) : 0, b = act ? __ldg(c.cone_off + ci + 1) : 0;
            double2 t = make_double2(0.0, 0.0);
            for (int j = a + sl; j < b; j += kConeLanes) sum(j, j == a, t);
            t.x = group_reduce<kConeLanes>(t.x);
            t.y = group_reduce<kConeLanes>(t.y);
            if (act) apply(a, b, t, sl, kConeLanes);
        }
    }
    for (int q = gwarp; q < c.n_cone_medium; q += nwarps) {   // medium: one warp per block
        const int ci = __ldg(c.cone_cls + c.n_cone_small + q);
        const int a = __ldg(c.cone_off + ci), b = __ldg(c.cone_off + ci + 1);
        double2 t = make_double2(0.0, 0.0);
        for (int j = a + lane; j < b; j += 32) sum(j, j == a, t);
        t.x = group_reduce<32>(t.x);
        t.y = group_reduce<32>(t.y);
        apply(a, b, t, lane, 32);
    }
    if (c.n_cone_large) {                                     // large: one CTA per block
        __shared__ double red[2][kWarps];
        for (int q = blockIdx.x; q < c.n_cone_large; q += gridDim.x) {
            const int ci = __ldg(c.cone_cls + c.n_cone_small + c.n_cone_medium + q);
            const int a = __ldg(c.cone_off + ci), b = __ldg(c.cone_off + ci + 1);
            double2 t = make_double2(0.0, 0.0);
            for (int j = a + (int)threadIdx.x; j < b; j += kBlock) sum(j, j == a, t);
            t.x = group_reduce<32>(t.x);
            t.y = group_reduce<32>(t.y);
            __syncthreads();                                  // the previous block's sums have been read
            if (lane == 0) { red[0][warp] = t.x; red[1][warp] = t.y; }
            __syncthreads();
            t = make_double2(0.0, 0.0);
            for (int w = 0; w < kWarps; ++w) { t.x += red[0][w]; t.y += red[1][w]; }
            apply(a, b, t, (int)threadIdx.x, kBlock);
        }
    }
}

// abs_K on one Lorentz block (Def.1; closed form of the projection onto {t >= ||u||}):
//   ||u|| <= t : v ;  ||u|| <= -t : -v ;  else (||u||, (t/||u||) u).   nu2 = ||u||^2; `f(j, p_j)` receives every coordinate.
template <class F>
__device__ __forceinline__ void soc_abs_apply(const double *s, int a, int b, double nu2, int l, int W, F &f) {
    const double t = s[a], nu = sqrt(nu2);
    if (nu <= t) {
        for (int j = a + l; j < b; j += W) f(j, s[j]);
    } else if (nu <= -t) {
        for (int j = a + l; j < b; j += W) f(j, -s[j]);
    } else {
        const double sc = t / nu;
        for (int j = a + l; j < b; j += W) f(j, j == a ? nu : sc * s[j]);
    }
}

// step 16: p = abs_K(s) ; also the two vectors the rhs pass gathers:
//   u := p - mu c^            (q = b~ - A~ u is the right-hand side of this pass's solve)
//   e := p - mu c^ + g        (r0 = b~ - A~ e is its residual at the warm start w, g = A~'w kept from before)
__device__ __forceinline__ void phase_cone_reflect(const Ctx &c) {
    const int tid = blockIdx.x * kBlock + threadIdx.x, nth = gridDim.x * kBlock;
    auto put = [&](int j, double pj) {
        const double uj = pj - c.mu * c.chat[j];
        c.p[j] = pj;
        c.u[j] = uj;
        c.e[j] = uj + c.g[j];
    };
    for (int j = tid; j < c.n_lin; j += nth) put(j, fabs(c.s[j]));
    if (c.n_soc)
        cone_sweep(c, [&](int j, bool head, double2 &t) { if (!head) { const double x = c.s[j]; t.x += x * x; } },
                   [&](int a, int b, double2 t, int l, int W) { soc_abs_apply(c.s, a, b, t.x, l, W, put); });
}

// ---------------------------------------------------------------------------------------------
// The ONE solve of a pass: with w_p = (A~A~')^{-1} A~ p and w_d = (A~A~')^{-1}(b~ + mu A~ c^),
// s+ = (s+p)/2 - A~'w_p + d and d = A~'w_d - mu c^ give s+ = (s+p)/2 - mu c^ + A~'w with
// (A~A~') w = b~ - A~(p - mu c^): neither d nor a solve at conditioning time is needed, and w = mu D^{-1} y
// converges to the (scaling-independent) dual solution, which makes the warm start effective.
// Inner solve: CG on (A~ A~') w = q, started from the current w with residual r already in c.r and
// rho = ||r||^2, qq = ||q||^2 known.  Two sparse passes and two grid reductions per step:
//   K1 (columns):  u = A~' z + beta u          sigma = ||u||^2       (u == A~' v by induction)
//   K2 (rows):     v = z + beta v ; w += alpha v ; r -= alpha (A~ u) ; ||r||^2
// with alpha = r'z/sigma (v'A~A~'v = ||A~'v||^2), beta = r'z_new / r'z, and z = r (Jacobi-equilibrated CG) or
// z = G'G r (FSAI(1), one more light pass and one more barrier per step).  Returns the steps done.
// ---------------------------------------------------------------------------------------------
struct TermDot {    // sum_k a_k x[j_k]  (A~' r, A~ u, A~' w, A~ c^ ...)
    const double *x;
    typedef double G;
    __device__ __forceinline__ G fetch(int j) const { return x[j]; }
    __device__ __forceinline__ void fma(double a, G g, double (&acc)[1]) const { acc[0] += a * g; }
};
struct NoPre {};
struct EpiK1 {
    double *u; double beta; double sigma;
    struct Pre { double u; };
    __device__ __forceinline__ Pre pre(int j) const { return Pre{u[j]}; }
    __device__ __forceinline__ double operator()(int j, const double (&a)[1], const Pre &q) {
        const double uj = a[0] + beta * q.u;
        u[j] = uj;
        sigma += uj * uj;
        return uj;           // the fused column pass multiplies the column's heavy-row entries with it
    }
};
struct EpiK2 {       // z = preconditioned residual (== r when the FSAI preconditioner is off)
    double *v, *w, *r; const double *z; double alpha, beta; double rho;
    double *z_long; int n_long;      // FSAI on: rows [0, n_long) (longer than kShortMax) have G = I, so z = r is written here
    double rz_long;                  // ... and their share of r'z = ||r||^2 over them
    struct Pre { double r, z, v, w; };
    __device__ __forceinline__ Pre pre(int i) const { return Pre{r[i], z[i], v[i], w[i]}; }
    __device__ __forceinline__ void operator()(int i, const double (&a)[1], const Pre &q) {
        const double vi = q.z + beta * q.v;
        v[i] = vi;
        w[i] = q.w + alpha * vi;
        const double rn = q.r - alpha * a[0];
        r[i] = rn;
        if (i < n_long) { z_long[i] = rn; rz_long += rn * rn; }
        rho += rn * rn;
    }
};

// z = G'G r for the FSAI(1) factor G (one off-diagonal entry per row, cs_kernels_cond.cuh builds it); returns
// r'z.  G'G is applied as ONE sparse symmetric operator assembled at build time:
//   z_k = dd_k r_k + ee_k r_{partner(k)} + sum_{e in list(k)} cc_e r_{tidx[e]}
// with dd_k = gd_k^2 + sum_{i in list(k)} gm_i^2, ee_k = gd_k gm_k, cc_e = gd_i gm_i (i = tidx[e]); list(k) = the
// rows whose partner is k, sorted, so the sum has a fixed order.  One light m-vector pass and one barrier.
#ifndef CS_FSAI_NB
#define CS_FSAI_NB 2
#endif
// CS_FSAI_NB rows per thread at a time: the loads of a row form a dependent chain (partner / list bounds -> list
// entry -> r), so the rows of a batch are interleaved by hand to keep several chains in flight (latency-bound).
// fsai_pass(c, k_begin): rows [k_begin, m), returns this thread's share of r'z (no grid reduction).
__device__ __forceinline__ double fsai_pass(const Ctx &c, int k_begin) {
    const int tid = blockIdx.x * kBlock + threadIdx.x, nth = gridDim.x * kBlock;
    constexpr int NB = CS_FSAI_NB;
    double rz = 0.0;
    for (int k0 = k_begin + tid; k0 < c.m; k0 += NB * nth) {
        int pk[NB], e0[NB], e1[NB];
        double rk[NB], acc[NB], rp[NB], ee[NB];
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            const int k = k0 + q * nth;
            const bool ok = k < c.m;
            pk[q] = ok ? c.f_partner[k] : -1;
            e0[q] = ok ? c.f_tptr[k] : 0;
            e1[q] = ok ? e0[q] + c.f_tcur[k] : 0;          // f_tcur: list length after the build (capped, cs_kernels_cond.cuh)
            rk[q] = ok ? c.r[k] : 0.0;
            acc[q] = ok ? c.f_gd[k] : 0.0;                 // f_gd holds dd after the build
            ee[q] = ok ? c.f_gm[k] : 0.0;                  // f_gm holds ee
        }
#pragma unroll
        for (int q = 0; q < NB; ++q) rp[q] = pk[q] >= 0 ? c.r[pk[q]] : 0.0;
        int i0[NB];
        double c0[NB];
#pragma unroll
        for (int q = 0; q < NB; ++q) {                     // first list entry of each row (most lists hold 0-2 rows)
            const bool has = e0[q] < e1[q];
            i0[q] = has ? c.f_tidx[e0[q]] : -1;
            c0[q] = has ? c.f_tc[e0[q]] : 0.0;
        }
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            acc[q] = acc[q] * rk[q] + ee[q] * rp[q];
            if (i0[q] >= 0) acc[q] += c0[q] * c.r[i0[q]];
        }
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            for (int e = e0[q] + 1; e < e1[q]; ++e) acc[q] += c.f_tc[e] * c.r[c.f_tidx[e]];
            const int k = k0 + q * nth;
            if (k < c.m) { c.z[k] = acc[q]; rz += rk[q] * acc[q]; }
        }
    }
    return rz;
}
__device__ __forceinline__ double apply_fsai(const Ctx &c, GridCtl &gc) {
    double red[1] = {fsai_pass(c, 0)};
    grid_reduce<1>(red, gc);
    return red[0];
}

// ---------------------------------------------------------------------------------------------
// Dense factor-apply path (cs_params.dense_m_threshold): one CTA, M = A~A~' in c.dM.
// dense_factor: M from the two compressed views (thread i owns row i: fixed summation order), then an in-place
// right-looking Cholesky on the lower triangle; the strict upper triangle and c.dMd keep M for the refinement.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void dense_factor(const Ctx &c) {
    const int m = c.m;
    double *M = c.dM;
    for (int i = threadIdx.x; i < m; i += kBlock) {
        double *row = M + (size_t)i * m;
        for (int j = 0; j < m; ++j) row[j] = 0.0;
        for (int e = c.Rc.ptr[i]; e < c.Rc.ptr[i + 1]; ++e) {
            const int k = c.Rc.idx[e];
            const double a = c.R.val[c.Rc.pos[e]];
            for (int f = c.Cc.ptr[k]; f < c.Cc.ptr[k + 1]; ++f) row[c.Cc.idx[f]] += a * c.C.val[c.Cc.pos[f]];
        }
        c.dMd[i] = row[i];
    }
    bool ok = true;
    for (int k = 0; k < m; ++k) {
        __syncthreads();
        const double piv = M[(size_t)k * m + k];
        if (!(piv > 1e-12)) { ok = false; break; }            // diag(A~A~') = 1: a relative test; uniform over the CTA (same pivot)
        const double d = sqrt(piv);
        __syncthreads();
        if (threadIdx.x == 0) M[(size_t)k * m + k] = d;
        for (int i = k + 1 + threadIdx.x; i < m; i += kBlock) M[(size_t)i * m + k] /= d;
        __syncthreads();
        const int t = m - k - 1;                              // trailing (i, j), k < j <= i < m
        for (int q = threadIdx.x; q < t * t; q += kBlock) {
            const int i = k + 1 + q / t, j = k + 1 + q % t;
            if (j <= i) M[(size_t)i * m + j] -= M[(size_t)i * m + k] * M[(size_t)j * m + k];
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) c.sc->dense_ok = ok ? 1 : 0;
}

// x <- L^-T L^-1 x on one warp (x in global scratch, m <= 256; every lane computes the same pivots)
__device__ __forceinline__ void dense_llt_solve(const double *M, int m, double *x, int lane) {
    for (int k = 0; k < m; ++k) {                             // forward: L y = x
        __syncwarp();
        const double yk = x[k] / M[(size_t)k * m + k];
        __syncwarp();
        if (lane == 0) x[k] = yk;
        for (int i = k + 1 + lane; i < m; i += 32) x[i] -= M[(size_t)i * m + k] * yk;
    }
    for (int k = m - 1; k >= 0; --k) {                        // backward: L' w = y (row k of L = column k of L')
        __syncwarp();
        const double wk = x[k] / M[(size_t)k * m + k];
        __syncwarp();
        if (lane == 0) x[k] = wk;
        for (int i = lane; i < k; i += 32) x[i] -= M[(size_t)k * m + i] * wk;
    }
    __syncwarp();
}

// w += M^-1 r with one step of iterative refinement against the stored M (r = residual of the warm start w)
__device__ __forceinline__ void dense_solve(const Ctx &c) {
    const int m = c.m, lane = threadIdx.x & 31;
    double *d1 = c.dv, *d2 = c.dv + m;
    if (threadIdx.x < 32) {
        for (int i = lane; i < m; i += 32) d1[i] = c.r[i];
        dense_llt_solve(c.dM, m, d1, lane);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < m; i += kBlock) {           // r2 = r - M d1
        double a = c.dMd[i] * d1[i];
        for (int j = 0; j < i; ++j) a += c.dM[(size_t)j * m + i] * d1[j];
        for (int j = i + 1; j < m; ++j) a += c.dM[(size_t)i * m + j] * d1[j];
        d2[i] = c.r[i] - a;
    }
    __syncthreads();
    if (threadIdx.x < 32) dense_llt_solve(c.dM, m, d2, lane);
    __syncthreads();
    for (int i = threadIdx.x; i < m; i += kBlock) c.w[i] += d1[i] + d2[i];
    __syncthreads();
}

// Heavy-row fusion (cs_device.cuh): shared-memory accumulators of the column pass.  fuse_zero before the pass;
// fuse_flush after it: the CTA's sums per fused row in a fixed order (class A: lanes by butterfly, then warps in
// order; class B: warps in order) -> c.fpart[row][CTA], which K2's finishing step adds up in CTA order.
__device__ __forceinline__ void fuse_zero(const Ctx &c) {
    double *A = FuseAcc::smem(), *B = A + kFuseOffB;
    for (int i = threadIdx.x; i < c.n_fa * kBlock; i += kBlock) A[i] = 0.0;
    for (int i = threadIdx.x; i < kWarps * kFuseB; i += kBlock) B[i] = 0.0;
    __syncthreads();
}
__device__ __forceinline__ void fuse_flush(const Ctx &c, double *scratch /* [kFuseA * kWarps] */) {
    const double *A = FuseAcc::smem(), *B = A + kFuseOffB;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    for (int i = 0; i < c.n_fa; ++i) {
        const double v = group_reduce<32>(A[i * kBlock + threadIdx.x]);
        if (lane == 0) scratch[i * kWarps + warp] = v;
    }
    __syncthreads();
    if (threadIdx.x < c.n_fa) {
        double acc = scratch[threadIdx.x * kWarps];
        for (int w = 1; w < kWarps; ++w) acc += scratch[threadIdx.x * kWarps + w];
        __stcg(c.fpart + (size_t)threadIdx.x * gridDim.x + blockIdx.x, acc);
    }
    for (int i = threadIdx.x; i < c.n_fb; i += kBlock) {
        double acc = B[i];
        for (int w = 1; w < kWarps; ++w) acc += B[w * kFuseB + i];
        __stcg(c.fpart + (size_t)(c.n_fa + i) * gridDim.x + blockIdx.x, acc);
    }
    __syncthreads();
}

// Grid dense path (cs_dense.cuh): w += M^-1 r with the explicit inverse and up to kDenseRefine steps of iterative refinement
// against the stored M = A~A~'.  Dense GEMVs: one warp per row, lanes along the row (coalesced), butterfly reduction.
//   x = Minv r ;  repeat: t = r - M x ; x += Minv t        (x in dv[0..m), t in dv[m..2m))
// The first refinement step always runs.  Its residual t measures what the explicit inverse leaves, eps0 = ||t|| / ||r||, and
// a step shrinks the residual by about that factor again; the second step runs unless eps0^2 is already a hundred times below
// cg_tol -- the criterion the CG path stops on (cs.h), with a margin for eps0 underestimating ||I - M Minv||.
// dense_gemv_rows returns this thread's share of sum_i out_i^2.
__device__ __forceinline__ double dense_gemv_rows(const double *A, const double *v, int m, int gwarp, int nwarps, int lane,
                                                  double *out, const double *base, double sign, const double *add) {
    double ss = 0.0;
    for (int i = gwarp; i < m; i += nwarps) {                 // out_i = (base ? base_i : 0) + sign * <A_i, v> + (add ? add_i : 0)
        const double *Ai = A + (size_t)i * m;
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
        int k = lane;
        for (; k + 96 < m; k += 128) {
            s0 += Ai[k] * v[k]; s1 += Ai[k + 32] * v[k + 32]; s2 += Ai[k + 64] * v[k + 64]; s3 += Ai[k + 96] * v[k + 96];
        }
        for (; k < m; k += 32) s0 += Ai[k] * v[k];
        const double s = group_reduce<32>((s0 + s1) + (s2 + s3));
        if (lane == 0) {
            const double o = (base ? base[i] : 0.0) + sign * s + (add ? add[i] : 0.0);
            out[i] = o;
            ss += o * o;
        }
    }
    return ss;
}
__device__ __forceinline__ void dense_apply_grid(const Ctx &c, GridCtl &gc, double rr /* ||r||^2 */) {
    const int lane = threadIdx.x & 31, gwarp = blockIdx.x + gridDim.x * (threadIdx.x >> 5), nwarps = (gridDim.x * kBlock) >> 5;
    double *x = c.dv, *t = c.dv + c.m;
    dense_gemv_rows(c.gMinv, c.r, c.m, gwarp, nwarps, lane, x, nullptr, 1.0, nullptr);          // x = Minv r
    gc.sync();
    for (int it = 0; it < kDenseRefine; ++it) {
        double tt[1] = {dense_gemv_rows(c.gM, x, c.m, gwarp, nwarps, lane, t, c.r, -1.0, nullptr)};   // t = r - M x
        grid_reduce<1>(tt, gc);                                                                  // ||t||^2, and the barrier
        double *xn = c.dv + 2 * c.m + (it & 1) * c.m;                                           // ping-pong: x is read by every warp
        dense_gemv_rows(c.gMinv, t, c.m, gwarp, nwarps, lane, xn, x, 1.0, nullptr);             // x' = x + Minv t
        gc.sync();
        x = xn;
        if (!(tt[0] > 0.01 * c.cg_tol * rr)) break;            // uniform over the grid (grid_reduce returns the same bits everywhere)
        if (it == 0 && blockIdx.x == 0 && threadIdx.x == 0) c.sc->dense_refine2 += 1;
    }
    for (int i = blockIdx.x * kBlock + threadIdx.x; i < c.m; i += gridDim.x * kBlock) c.w[i] += x[i];
    gc.sync();
}

// The two passes over A~ of a dense-path iteration (the right-hand side and steps 17-18) read the row-major dense copy
// Ad [m][n] that the conditioning has scattered (cs_dense.cuh) instead of the sliced sparse copies: 8 bytes per entry instead
// of 12, contiguous vector reads instead of gathers.  Fixed summation orders.
//   dense_rows_pair: (sum_j Ad[i][j] x[j], sum_j Ad[i][j] y[j]) per row i -> epi(i, .): one warp per row, lanes along the row
template <class Epi>
__device__ __forceinline__ void dense_rows_pair(const Ctx &c, const double *x, const double *y, Epi &epi) {
    const int lane = threadIdx.x & 31, gwarp = blockIdx.x + gridDim.x * (threadIdx.x >> 5), nwarps = (gridDim.x * kBlock) >> 5;
    const int n = c.n;
    for (int i = gwarp; i < c.m; i += nwarps) {
        const double *row = c.gAd + (size_t)i * n;
        double a0 = 0.0, a1 = 0.0;
        int j = lane;
        for (; j + 224 < n; j += 256) {                          // 8 independent row loads in flight
            double v[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) v[q] = __ldcs(row + j + 32 * q);
#pragma unroll
            for (int q = 0; q < 8; ++q) { a0 += v[q] * x[j + 32 * q]; a1 += v[q] * y[j + 32 * q]; }
        }
        for (; j < n; j += 32) { const double v = __ldcs(row + j); a0 += v * x[j]; a1 += v * y[j]; }
        a0 = group_reduce<32>(a0);
        a1 = group_reduce<32>(a1);
        if (lane == 0) { const double acc[2] = {a0, a1}; epi(i, acc, epi.pre(i)); }
    }
}
//   dense_cols: sum_i Ad[i][j] w[i] per column j -> epi(j, .).  Work items (64 columns, a range of rows), one warp each, two
//   columns per lane; the items' partial sums go through c.gpart [row range][n] and are added in range order after a barrier.
template <class Epi>
__device__ __forceinline__ void dense_cols(const Ctx &c, const double *w, Epi &epi, GridCtl &gc) {
    const int lane = threadIdx.x & 31, gwarp = blockIdx.x + gridDim.x * (threadIdx.x >> 5), nwarps = (gridDim.x * kBlock) >> 5;
    const int n = c.n, m = c.m, G = (n + 63) / 64;
    const int nsplit = max(1, min(nwarps / G, m));               // row ranges: as many as fill the machine
    const int per = (m + nsplit - 1) / nsplit;
    for (int t = gwarp; t < G * nsplit; t += nwarps) {
        const int g = t % G, rs = t / G, r0 = rs * per, r1 = min(m, r0 + per);
        const int j0 = g * 64 + lane, j1 = j0 + 32;              // this lane's two columns
        double a0 = 0.0, a1 = 0.0;
        const double *col = c.gAd + (size_t)r0 * n;
        int i = r0;
        for (; i + 3 < r1; i += 4) {                             // 8 independent loads in flight
            double v0[4], v1[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                v0[q] = j0 < n ? __ldcs(col + (size_t)q * n + j0) : 0.0;
                v1[q] = j1 < n ? __ldcs(col + (size_t)q * n + j1) : 0.0;
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) { const double wi = w[i + q]; a0 += v0[q] * wi; a1 += v1[q] * wi; }
            col += (size_t)4 * n;
        }
        for (; i < r1; ++i, col += n) {
            const double wi = w[i];
            if (j0 < n) a0 += __ldcs(col + j0) * wi;
            if (j1 < n) a1 += __ldcs(col + j1) * wi;
        }
        if (j0 < n) __stcg(c.gpart + (size_t)rs * n + j0, a0);
        if (j1 < n) __stcg(c.gpart + (size_t)rs * n + j1, a1);
    }
    gc.sync();
    for (int j = blockIdx.x * kBlock + threadIdx.x; j < n; j += gridDim.x * kBlock) {
        typename Epi::Pre pre = epi.pre(j);
        double a = 0.0;
        for (int rs = 0; rs < nsplit; ++rs) a += __ldcg(c.gpart + (size_t)rs * n + j);
        const double acc[1] = {a};
        epi(j, acc, pre);
    }
}

__device__ __forceinline__ void fsaip_pass_a(const Ctx &c, int k_begin);      // cs_fsaip.cuh
__device__ __forceinline__ double fsaip_pass_b(const Ctx &c, int k_begin);
// r'z with z = (preconditioner) r over ALL rows, one grid reduction (start of a solve)
__device__ __forceinline__ double apply_precond(const Ctx &c, GridCtl &gc) {
    if (c.fsai == 2) {
        fsaip_pass_a(c, 0);
        gc.sync();
        double red[1] = {fsaip_pass_b(c, 0)};
        grid_reduce<1>(red, gc);
        return red[0];
    }
    return apply_fsai(c, gc);
}

__device__ __forceinline__ int cg_solve(const Ctx &c, GridCtl &gc, double rr, double qq, bool &hit_max) {
    // stop on ||r|| <= max(cg_tol ||q||, cg_reduce ||r at the warm start||) (equilibrated system; cs.h)
    const double thresh = fmax(c.cg_tol * c.cg_tol * qq, c.cg_reduce * c.cg_reduce * rr);
    const double *zsrc = c.fsai ? c.z : c.r;
    const bool fused = c.n_fa + c.n_fb > 0;                  // uniform over the grid
    double beta = 0.0;
    int steps = 0;
    hit_max = false;
    if (!(rr > thresh)) return 0;
    double rz = c.fsai ? apply_precond(c, gc) : rr;        // r'z, z = G'G r
    while (rr > thresh) {
        if (steps >= c.cg_max_iter) { hit_max = true; break; }
        TermDot t1{zsrc};
        EpiK1 e1{c.u, beta, 0.0};
        if (fused) {                                       // u = A~'z + beta u = A~'v, and the heavy rows' share of A~u
            fuse_zero(c);
            seg_reduce<1, false, 0, TermDot, EpiK1, FuseAcc>(c.C, t1, e1, gc, FuseAcc{c.n_fa});
            fuse_flush(c, gc.smem);
        } else {
            seg_reduce<1, false>(c.C, t1, e1, gc);
        }
        gc.lap(kPhK1);
        double red[1] = {e1.sigma};
        grid_reduce<1>(red, gc);
        gc.lap(kPhReduce);
        const double sigma = red[0];
        if (!(sigma > 0.0)) break;
        const double alpha = rz / sigma;
        TermDot t2{c.u};
        EpiK2 e2{c.v, c.w, c.r, zsrc, alpha, beta, 0.0, c.z, c.fsai ? c.n_long : 0, 0.0};
        seg_reduce<1, false, 1>(c.R, t2, e2, gc);          // K2 view: without the entries the column pass has done
        gc.lap(kPhK2);
        double rz_new;
        if (c.fsai) {
            // z = G'G r for the short rows in the same phase as K2's finishing step (the long rows, whose sums that step
            // completes, have G = I and got z = r from the epilogue; no short row's z reads a long row's r): one barrier
            // and one reduction for both ||r||^2 and r'z
            if (!c.R.n_multi_k2) gc.sync();                // otherwise seg_reduce's own barrier has made r complete
            double red2[2] = {e2.rho, 0.0};
            if (c.fsai == 2) { fsaip_pass_a(c, c.n_long); gc.sync(); red2[1] = fsaip_pass_b(c, c.n_long); }   // FSAI(P): t = G r, z = G't
            else red2[1] = fsai_pass(c, c.n_long);
            gc.lap(kPhPrecond);
            red2[1] += e2.rz_long;                         // the long rows' share, from K2's epilogue
            grid_reduce<2>(red2, gc);
            gc.lap(kPhReduce);
            rr = red2[0];
            rz_new = red2[1];
        } else {
            red[0] = e2.rho;
            grid_reduce<1>(red, gc);
            gc.lap(kPhReduce);
            rr = red[0];
            rz_new = rr;
        }
        beta = rz_new / rz;
        rz = rz_new;
        ++steps;
    }
    return steps;
}

// ---------------------------------------------------------------------------------------------
// k_iterate
// ---------------------------------------------------------------------------------------------
struct TermPair {   // (sum a x[j], sum a y[j]): both gathers of the rhs pass
    const double *p, *e;
    typedef double2 G;
    __device__ __forceinline__ G fetch(int j) const { return make_double2(p[j], e[j]); }
    __device__ __forceinline__ void fma(double a, G g, double (&acc)[2]) const {
        acc[0] += a * g.x;
        acc[1] += a * g.y;
    }
};
struct EpiRhs {     // q = b~ - A~(p - mu c^) ; r = q - A~A~'w = b~ - A~ e ; qq = ||q||^2 ; rho = ||r||^2
    double *r; const double *btil; double qq, rho;
    typedef NoPre Pre;
    __device__ __forceinline__ Pre pre(int) const { return Pre{}; }
    __device__ __forceinline__ void operator()(int i, const double (&a)[2], const Pre &) {
        const double q = btil[i] - a[0], ri = btil[i] - a[1];
        r[i] = ri;
        qq += q * q;
        rho += ri * ri;
    }
};
struct EpiUpdate {  // steps 17-18 with d folded in: s <- (s+p)/2 - mu c^ + A~'w
    double *s, *g; const double *p, *chat; double mu; double fp2;
    struct Pre { double s, p, c; };
    __device__ __forceinline__ Pre pre(int j) const { return Pre{s[j], p[j], chat[j]}; }
    __device__ __forceinline__ void operator()(int j, const double (&a)[1], const Pre &q) {
        const double sj = q.s;
        const double sn = 0.5 * (sj + q.p) - mu * q.c + a[0];
        g[j] = a[0];
        s[j] = sn;
        fp2 += (sn - sj) * (sn - sj);
    }
};

// DENSE = true is the one-CTA build whose solve is the dense factor-apply; it is a separate instantiation so that
// the sparse kernel's code (register allocation, schedule) is exactly what the profiles measured.
template <bool DENSE>
__device__ __forceinline__ void iterate_body(const Ctx &c, long long k_iter) {
    __shared__ double smem[kMaxRed * kWarps];
    GridCtl gc(c.partials, smem, c.bar);
    long long cg_total = 0;
    int cg_last = 0;
    bool any_max = false;
    double fp2 = 0.0;
    for (long long it = 0; it < k_iter; ++it) {
        gc.lap(kPhReduce);
        phase_cone_reflect(c);                                   // step 16
        gc.sync();
        gc.lap(kPhCone);
        TermPair tq{c.u, c.e};
        EpiRhs eq{c.r, c.btil, 0.0, 0.0};
        if (DENSE && c.dense == 2) dense_rows_pair(c, c.u, c.e, eq);   // the dense copy of A~ (grid dense path)
        else seg_reduce<2, false>(c.R, tq, eq, gc);
        gc.lap(kPhRhs);
        double red[2] = {eq.qq, eq.rho};
        grid_reduce<2>(red, gc);
        gc.lap(kPhReduce);
        bool hm;
        if (DENSE && c.dense == 2 && *c.g_ok) { dense_apply_grid(c, gc, red[1]); cg_last = 0; hm = false; }   // dense factor-apply (grid)
        else if (DENSE && c.dense == 1 && c.sc->dense_ok) { dense_solve(c); cg_last = 0; hm = false; }   // dense factor-apply (one CTA)
        else cg_last = cg_solve(c, gc, red[1], red[0], hm);      // w = (A~A~')^{-1} (b~ - A~(p - mu c^)) = w_d - w_p
        any_max |= hm;
        cg_total += cg_last;
        TermDot tw{c.w};
        EpiUpdate eu{c.s, c.g, c.p, c.chat, c.mu, 0.0};
        if (DENSE && c.dense == 2) dense_cols(c, c.w, eu, gc);   // steps 17-18 over the dense copy
        else seg_reduce<1, false>(c.C, tw, eu, gc);              // steps 17-18
        gc.lap(kPhUpdate);
        double rf[1] = {eu.fp2};
        grid_reduce<1>(rf, gc);
        gc.lap(kPhReduce);
        fp2 = rf[0];
    }
    gc.flush(c.sc);
    if (blockIdx.x == 0 && threadIdx.x == 0 && k_iter > 0) {
        c.sc->iter += k_iter;
        c.sc->cg_steps_total += cg_total;
        c.sc->cg_steps_last = cg_last;
        c.sc->fp_res2 = fp2;
        if (any_max) c.sc->cg_hit_max = 1;
    }
}

__global__ void __launch_bounds__(kBlock, CS_MINB) k_iterate(Ctx c, long long k_iter) { iterate_body<false>(c, k_iter); }
__global__ void __launch_bounds__(kBlock, CS_MINB) k_iterate_dense(Ctx c, long long k_iter) { iterate_body<true>(c, k_iter); }

}  // namespace csd
