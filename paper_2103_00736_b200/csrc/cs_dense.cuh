// cs_dense.cuh -- dense factor-apply path for problems on many CTAs (B north_star: "a dense factor-apply kernel only
// where A is small enough that it is truly a dense contraction"; S 8(f).3: the paper's own dense shapes, section V-A
// P:342-346 and V-D P:366-371).  For a dense-stored A with m <= kDenseGridMax:
//   at every conditioning   Ad = A~ (m x n, row-major)          k_dense_scatter
//                           M  = Ad Ad'                          k_dense_aat        (unit diagonal: A~ is row-equilibrated)
//                           M  = L L'   (blocked, right-looking) k_chol_diag / k_chol_panel / k_chol_update / k_chol_update_panel
//                           Z  = L^-T   (row j = column j of L^-1)  k_dense_diag_inv, k_dense_trinv_blk
//                           Minv = Z Z' = M^-1                   k_dense_aat
//   at every pass           w += M^-1 r by dense_apply_grid (cs_kernels.cuh): x = Minv r, then up to kDenseRefine steps of
//                           iterative refinement x += Minv (r - M x) against the stored M -- dense GEMVs only.
// All sums have a fixed order (no atomics).  fp64 throughout; plain DFMA (no tensor cores: B200's fp64 tensor rate equals
// its vector rate).  Measured from m = 2320 to m = 24000 (the paper's largest LP): DESIGN.md 10.
#pragma once
#include "cs_device.cuh"

namespace csd {

constexpr int kDenseGridMax = 24576; // largest m of the grid dense path: covers the paper's largest dense LP, n = 30000, m = 24000;
                                     // four m x m fp64 matrices + A~ [m][n] = 24 GB there, allocated on first use (cs_api.cu)
constexpr int kDenseRefine = 2;      // most refinement steps of the per-pass apply (the second runs only when needed)
constexpr int kCholNB = 32;          // panel width of the blocked Cholesky

// Ad[i][j] = A~_ij from the row-major slice copy (Ad zeroed by the caller)
__global__ void k_dense_scatter(Ctx c, double *Ad) {
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    for (int i = gwarp; i < c.m; i += nwarps)
        for (int e = c.Rc.ptr[i] + lane; e < c.Rc.ptr[i + 1]; e += 32) Ad[(size_t)i * c.n + c.Rc.idx[e]] = c.R.val[c.Rc.pos[e]];
}

// ---- the dense contraction core: a 128 x 128 tile of sum_k A[a0+i][k] B[b0+j][k] ("NT": both operands row-major along k) --
// 256 threads, 8 x 8 outputs per thread in registers (rows ty*4+{0..3} and 64+ty*4+{0..3}, columns likewise with tx: the
// shared-memory reads are 16-byte loads without bank conflicts), operands staged k-major 16 columns at a time, the next
// stage fetched into registers while the current one is consumed.  Plain DFMA: per k a thread does 64 multiply-adds on 8
// 16-byte shared loads, so the FP64 pipe is the bound (B200's fp64 tensor rate equals its vector rate).  Fixed summation order.
constexpr int kGemmT = 128, kGemmK = 16;
struct GemmSmem { double a[kGemmK][kGemmT + 2], b[kGemmK][kGemmT + 2]; };

__device__ __forceinline__ void gemm_nt_tile(const double *A, size_t lda, int ra, int a0, const double *B, size_t ldb, int rb, int b0,
                                             int k0, int k1, GemmSmem &sm, double (&acc)[8][8]) {
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const int lr = tid >> 3, lc = (tid & 7) * 2;                 // loader: rows lr + 32 i, columns lc, lc + 1 of the stage
    double pa[4][2], pb[4][2];
    auto fetch = [&](int kk) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int r = a0 + lr + 32 * i, q = b0 + lr + 32 * i, k = kk + lc;
            pa[i][0] = (r < ra && k < k1) ? A[(size_t)r * lda + k] : 0.0;
            pa[i][1] = (r < ra && k + 1 < k1) ? A[(size_t)r * lda + k + 1] : 0.0;
            pb[i][0] = (q < rb && k < k1) ? B[(size_t)q * ldb + k] : 0.0;
            pb[i][1] = (q < rb && k + 1 < k1) ? B[(size_t)q * ldb + k + 1] : 0.0;
        }
    };
    fetch(k0);
    for (int kk0 = k0; kk0 < k1; kk0 += kGemmK) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            sm.a[lc][lr + 32 * i] = pa[i][0]; sm.a[lc + 1][lr + 32 * i] = pa[i][1];
            sm.b[lc][lr + 32 * i] = pb[i][0]; sm.b[lc + 1][lr + 32 * i] = pb[i][1];
        }
        __syncthreads();
        if (kk0 + kGemmK < k1) fetch(kk0 + kGemmK);
#pragma unroll
        for (int kk = 0; kk < kGemmK; ++kk) {
            double va[8], vb[8];
            *reinterpret_cast<double2 *>(va + 0) = *reinterpret_cast<const double2 *>(&sm.a[kk][ty * 4]);
            *reinterpret_cast<double2 *>(va + 2) = *reinterpret_cast<const double2 *>(&sm.a[kk][ty * 4 + 2]);
            *reinterpret_cast<double2 *>(va + 4) = *reinterpret_cast<const double2 *>(&sm.a[kk][64 + ty * 4]);
            *reinterpret_cast<double2 *>(va + 6) = *reinterpret_cast<const double2 *>(&sm.a[kk][64 + ty * 4 + 2]);
            *reinterpret_cast<double2 *>(vb + 0) = *reinterpret_cast<const double2 *>(&sm.b[kk][tx * 4]);
            *reinterpret_cast<double2 *>(vb + 2) = *reinterpret_cast<const double2 *>(&sm.b[kk][tx * 4 + 2]);
            *reinterpret_cast<double2 *>(vb + 4) = *reinterpret_cast<const double2 *>(&sm.b[kk][64 + tx * 4]);
            *reinterpret_cast<double2 *>(vb + 6) = *reinterpret_cast<const double2 *>(&sm.b[kk][64 + tx * 4 + 2]);
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 8; ++j) acc[i][j] += va[i] * vb[j];
        }
        __syncthreads();
    }
}
// tile (ti, tj), tj <= ti, of the lower triangle from the linear block index
__device__ __forceinline__ void tri_tile(int b, int &ti, int &tj) {
    ti = (int)((sqrt(8.0 * b + 1.0) - 1.0) * 0.5);
    while ((ti + 1) * (ti + 2) / 2 <= b) ++ti;
    while (ti * (ti + 1) / 2 > b) --ti;
    tj = b - ti * (ti + 1) / 2;
}
__device__ __forceinline__ int gemm_row(int t, int i) { return (i < 4 ? 0 : 60) + t * 4 + i; }   // output i of thread coordinate t

// C = A A' for a row-major A [r][k]; C [r][r] full (both triangles written).  One CTA per 128 x 128 tile of the lower triangle.
// tri != 0: A is upper triangular (A[a][i] = 0 for i < a, k = r), so the sum starts at the tile's first row (Minv = Z Z').
__global__ void __launch_bounds__(256) k_dense_aat(const double *A, int r, int k, double *C, int tri) {
    __shared__ __align__(16) GemmSmem sm;
    int ti, tj;
    tri_tile(blockIdx.x, ti, tj);
    const int a0 = ti * kGemmT, b0 = tj * kGemmT, tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    double acc[8][8] = {};
    gemm_nt_tile(A, (size_t)k, r, a0, A, (size_t)k, r, b0, tri ? a0 : 0, k, sm, acc);   // a0 >= b0: both operands are zero before column a0
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int a = a0 + gemm_row(ty, i), b = b0 + gemm_row(tx, j);
            if (a < r && b < r) {
                C[(size_t)a * r + b] = acc[i][j];
                if (ti != tj) C[(size_t)b * r + a] = acc[i][j];
            }
        }
}

// ---- blocked right-looking Cholesky of L (m x m row-major, lower triangle used; starts as a copy of M) -------------
// Two levels: panels of kCholPanel = 128 columns, factored in steps of nb = 32 columns,
// step kb: (1) k_chol_diag factors the nb x nb diagonal block in shared memory (one CTA); a pivot <= 1e-12 (diag(M) = 1:
//              a relative test) clears *ok and is replaced by 1 so that the run stays finite (the caller falls back to CG)
//          (2) k_chol_panel: rows below the block, X D' = L[i][kb:kb+nb] -- one warp per row, lane c owns column c
//          (3) k_chol_update: the rank-32 update of the panel's remaining columns only (64 x 64 tiles, 4 x 4 per thread)
// and after the panel's last step ONE rank-128 update of everything behind it, k_chol_update_panel, through the 128 x 128
// contraction core: a rank-32 update of the whole trailing matrix is bound by reading and writing L (6.5 TFLOP/s at
// m = 8000), the rank-128 one by the FP64 pipe.
constexpr int kCholPanel = 128;
__global__ void __launch_bounds__(kCholNB * kCholNB) k_chol_diag(double *L, int m, int kb, int *ok) {
    __shared__ double d[kCholNB][kCholNB + 1];
    const int nb = min(kCholNB, m - kb), r = threadIdx.x / kCholNB, cc = threadIdx.x % kCholNB;
    if (r < nb && cc < nb) d[r][cc] = L[(size_t)(kb + r) * m + kb + cc];
    __syncthreads();
    for (int k = 0; k < nb; ++k) {
        double piv = d[k][k];
        __syncthreads();
        if (!(piv > 1e-12)) { if (threadIdx.x == 0) *ok = 0; piv = 1.0; }
        const double dk = sqrt(piv);
        if (r == k && cc == k) d[k][k] = dk;
        if (cc == k && r > k && r < nb) d[r][k] /= dk;
        __syncthreads();
        if (r > k && cc > k && cc <= r && r < nb) d[r][cc] -= d[r][k] * d[cc][k];
        __syncthreads();
    }
    if (r < nb && cc <= r) L[(size_t)(kb + r) * m + kb + cc] = d[r][cc];
}

__global__ void __launch_bounds__(256) k_chol_panel(double *L, int m, int kb) {
    __shared__ double d[kCholNB][kCholNB + 1];
    const int nb = min(kCholNB, m - kb), lane = threadIdx.x & 31;
    for (int q = threadIdx.x; q < kCholNB * kCholNB; q += 256) {
        const int r = q / kCholNB, cc = q % kCholNB;
        d[r][cc] = (r < nb && cc <= r) ? L[(size_t)(kb + r) * m + kb + cc] : (r == cc ? 1.0 : 0.0);
    }
    __syncthreads();
    const int gwarp = (blockIdx.x * 256 + threadIdx.x) >> 5, nwarps = (gridDim.x * 256) >> 5;
    for (int i = kb + nb + gwarp; i < m; i += nwarps) {
        double a = lane < nb ? L[(size_t)i * m + kb + lane] : 0.0;
        for (int cidx = 0; cidx < nb; ++cidx) {                    // x_c = a_c / D_cc ; a_q -= x_c D_qc for q > c
            const double xc = __shfl_sync(0xffffffffu, a, cidx) / d[cidx][cidx];
            if (lane == cidx) a = xc;
            else if (lane > cidx) a -= xc * d[lane][cidx];
        }
        if (lane < nb) L[(size_t)i * m + kb + lane] = a;
    }
}

// rank-32 update inside the current 128-wide panel: columns [kb + nb, cend) of the rows below the block
__global__ void __launch_bounds__(256) k_chol_update(double *L, int m, int kb, int cend) {
    __shared__ double pi[kCholNB][65], pj[kCholNB][65];
    const int nb = min(kCholNB, m - kb), base = kb + nb;
    const int ti = blockIdx.x, tj = blockIdx.y;
    if (tj > ti) return;                                         // tile above the diagonal
    const int i0 = base + ti * 64, j0 = base + tj * 64, tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    for (int q = threadIdx.x; q < 64 * kCholNB; q += 256) {
        const int row = q / kCholNB, cc = q % kCholNB;
        pi[cc][row] = (cc < nb && i0 + row < m) ? L[(size_t)(i0 + row) * m + kb + cc] : 0.0;
        pj[cc][row] = (cc < nb && j0 + row < m) ? L[(size_t)(j0 + row) * m + kb + cc] : 0.0;
    }
    __syncthreads();
    double acc[4][4] = {};
#pragma unroll 8
    for (int cc = 0; cc < kCholNB; ++cc) {
        double va[4], vb[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) { va[i] = pi[cc][ty * 4 + i]; vb[i] = pj[cc][tx * 4 + i]; }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j] += va[i] * vb[j];
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int a = i0 + ty * 4 + i, b = j0 + tx * 4 + j;
            if (a < m && b <= a && b < cend) L[(size_t)a * m + b] -= acc[i][j];
        }
}

// rank-(pend - pb) update of everything behind a finished panel: L[a][b] -= sum_{c in [pb, pend)} L[a][c] L[b][c], a >= b >= pend,
// through the 128 x 128 contraction core (one CTA per tile of the lower triangle)
__global__ void __launch_bounds__(256) k_chol_update_panel(double *L, int m, int pb, int pend) {
    __shared__ __align__(16) GemmSmem sm;
    int ti, tj;
    tri_tile(blockIdx.x, ti, tj);
    const int a0 = ti * kGemmT, b0 = tj * kGemmT, tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    const double *P = L + (size_t)pend * m + pb;                 // row i of P = row pend + i of L, columns pb .. pend
    double acc[8][8] = {};
    gemm_nt_tile(P, (size_t)m, m - pend, a0, P, (size_t)m, m - pend, b0, 0, pend - pb, sm, acc);
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int a = pend + a0 + gemm_row(ty, i), b = pend + b0 + gemm_row(tx, j);
            if (a < m && b <= a) L[(size_t)a * m + b] -= acc[i][j];
        }
}

// ---- Z = L^-T (row j of Z = column j of L^-1), blocked ---------------------------------------------------------------
// Column j of X = L^-1 depends on L only, so column groups are independent; inside a group the block rows follow one
// another:  X_JJ = (L_JJ)^-1,   X_IJ = -(L_II)^-1 sum_{K=J}^{I-1} L_IK X_KJ   (64 x 64 blocks of L).
// k_dense_diag_inv inverts every diagonal block once; k_dense_trinv_blk gives one CTA a group of CW columns and walks
// the block rows with 64 x 64 tiles of L in shared memory (each tile serves 64 x CW x 64 multiply-adds, so L is read
// m / (3 CW) times from L2 instead of m / 3 times: 6.9 -> 1.7 ms at m = 2320 with CW = 8).  Heaviest groups (J = 0) have the
// lowest block indices and start first.  Fixed summation order; Z zeroed by the caller (x_i = 0 for i < j's block).
constexpr int kTriNB = 64;

__global__ void __launch_bounds__(kTriNB) k_dense_diag_inv(const double *L, int m, double *Dinv) {
    constexpr int kTri = kTriNB * (kTriNB + 1) / 2;              // packed lower triangles: (i, k) at i (i + 1) / 2 + k
    __shared__ double sl[kTri], sx[kTri];
    const int I = blockIdx.x, b0 = I * kTriNB, j = threadIdx.x;
    for (int r = j; r < kTriNB; ++r) {                           // thread j loads column j; identity-padded past m
        const int gi = b0 + r, gj = b0 + j;
        sl[r * (r + 1) / 2 + j] = (gi < m && gj < m) ? L[(size_t)gi * m + gj] : (r == j ? 1.0 : 0.0);
    }
    __syncthreads();
    for (int i = j; i < kTriNB; ++i) {                           // thread j: column j of the inverse, forward substitution
        double s = i == j ? 1.0 : 0.0;
        for (int k = j; k < i; ++k) s -= sl[i * (i + 1) / 2 + k] * sx[k * (k + 1) / 2 + j];
        sx[i * (i + 1) / 2 + j] = s / sl[i * (i + 1) / 2 + i];
    }
    for (int r = 0; r < kTriNB; ++r) Dinv[((size_t)I * kTriNB + r) * kTriNB + j] = j <= r ? sx[r * (r + 1) / 2 + j] : 0.0;
}

// shared memory of k_dense_trinv_blk (dynamic; 148-186 KB: one CTA per SM): a ring of kTriStages tiles of L (or (L_II)^-1)
// filled by cp.async kTriStages - 1 steps ahead, two stages of the matching rows of X, and the block row of X computed last
// (the next block row's first-hand operand)
constexpr int kTriStages = 4;
template <int CW>
struct TrinvSmem {
    double l[kTriStages][kTriNB][kTriNB + 2];
    double x[2][CW][kTriNB + 2];         // [column of the group][k]
    double fresh[CW][kTriNB + 2];
};
__device__ __forceinline__ void cp_async8(void *dst, const void *src, bool ok) {   // 8 bytes global -> shared, zero-filled if !ok
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    const int n = ok ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" :: "r"(d), "l"(src), "r"(n) : "memory");
}

__device__ __forceinline__ void cp_async16(void *dst, const void *src, bool ok) {  // 16 bytes, both sides 16-byte aligned
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    const int n = ok ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(d), "l"(src), "r"(n) : "memory");
}

// CW columns of L^-1 per CTA (8, 16 or 32: the host picks the widest that still leaves two groups per SM -- a wider group
// reads L fewer times, m / (3 CW) in all, but there are fewer groups and each one's chain of block rows is serial).
// 256 threads (two warps per scheduler: the steps are short and latency-bound); thread (cc = lane % CW, rh = lane / CW) of
// warp w owns rows 8 w + rh + (32 / CW) q, q < CW / 4, of a block row.
// Step (I, K): K < I multiplies the tile L_IK with X_K; K == I multiplies (L_II)^-1 with the finished sum.  The steps of a
// group form one serial chain (the first group's is (m / 64)^2 / 2 steps long), so what matters is the time per step:
// the tiles of L come from HBM and are requested kTriStages - 1 steps ahead; the rows of X (L2, written by this CTA at
// least one block row earlier) are loaded into registers one step ahead; X_{I-1} is still in shared memory (sm.fresh).
constexpr int kTriThreads = 256;
template <int CW>
__global__ void __launch_bounds__(kTriThreads) k_dense_trinv_blk(const double *L, const double *Dinv, int m, double *Z) {
    constexpr int NQ = CW / 4, RS = 32 / CW, ST = kTriStages, NT = kTriThreads, NX = kTriNB * CW / NT;
    extern __shared__ __align__(16) unsigned char trinv_raw[];
    TrinvSmem<CW> &sm = *reinterpret_cast<TrinvSmem<CW> *>(trinv_raw);
    const int c0 = blockIdx.x * CW, J = c0 / kTriNB, nblk = (m + kTriNB - 1) / kTriNB;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, cc = lane & (CW - 1), rh = lane / CW;
    const int gc = c0 + cc;                                      // this thread's column of L^-1 = row of Z
    const int row0 = 8 * w + rh;                                 // its rows of the block row: row0 + RS q
    const bool even = (m & 1) == 0;                              // rows of L start 16-byte aligned: 16-byte cp.async
    auto issue_l = [&](int I, int K, int stage) {                // one group per step, empty past the end of the chain
        if (I < nblk) {
            const double *base = K == I ? Dinv + (size_t)I * kTriNB * kTriNB : L + (size_t)I * kTriNB * m + K * kTriNB;
            const size_t ld = K == I ? (size_t)kTriNB : (size_t)m;
            const int rows = K == I ? kTriNB : min(kTriNB, m - I * kTriNB);   // rows past m are zero-filled
            if (even) {
                for (int t = threadIdx.x; t < kTriNB * kTriNB / 2; t += NT) {
                    const int r = t >> 5, k = (t & 31) * 2;
                    cp_async16(&sm.l[stage][r][k], base + (r < rows ? (size_t)r * ld + k : 0), r < rows);
                }
            } else {
                for (int t = threadIdx.x; t < kTriNB * kTriNB; t += NT) {
                    const int r = t >> 6, k = t & 63;
                    cp_async8(&sm.l[stage][r][k], base + (r < rows ? (size_t)r * ld + k : 0), r < rows);
                }
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    auto advance = [&](int &I, int &K) { if (K < I) ++K; else { ++I; K = J; } };
    int pI = J, pK = J;                                          // the step whose tile of L is requested next
    for (int q = 0; q < ST - 1; ++q) { issue_l(pI, pK, q); advance(pI, pK); }
    int step = 0;
    for (int I = J; I < nblk; ++I) {
        double acc[NQ], xo[NQ];
#pragma unroll
        for (int q = 0; q < NQ; ++q) { acc[q] = 0.0; xo[q] = 0.0; }
        for (int K = J; K <= I; ++K, ++step) {
            const int stage = step % ST;
            issue_l(pI, pK, (step + ST - 1) % ST);
            advance(pI, pK);
            // rows of X for the next step into registers (it needs them from Z only if its K' < I' - 1)
            int nI = I, nK = K;
            advance(nI, nK);
            const bool next_x = nI < nblk && nK < nI - 1;
            double xr[NX];                                       // 64 CW doubles over the CTA's threads
            if (next_x) {
#pragma unroll
                for (int q = 0; q < NX; ++q) {
                    const int t = threadIdx.x + NT * q, c = t >> 6, k = t & 63;
                    xr[q] = c0 + c < m ? __ldcg(Z + (size_t)(c0 + c) * m + nK * kTriNB + k) : 0.0;
                }
            }
            asm volatile("cp.async.wait_group %0;" :: "n"(ST - 1) : "memory");   // this step's tile of L has landed
            if (K == I && I > J) {                               // the finished sum T becomes the operand of (L_II)^-1
#pragma unroll
                for (int q = 0; q < NQ; ++q) sm.x[step & 1][cc][row0 + RS * q] = acc[q];
            }
            __syncthreads();
            if (K == I && I == J) {                              // X_JJ: the group's columns of (L_JJ)^-1
#pragma unroll
                for (int q = 0; q < NQ; ++q) xo[q] = sm.l[stage][row0 + RS * q][gc - J * kTriNB];
            } else {
                const double *xs = K == I - 1 ? sm.fresh[cc] : sm.x[step & 1][cc];
                if (K < I) {
#pragma unroll 4
                    for (int k = 0; k < kTriNB; ++k) {
                        const double x = xs[k];
#pragma unroll
                        for (int q = 0; q < NQ; ++q) acc[q] += sm.l[stage][row0 + RS * q][k] * x;
                    }
                } else {                                         // X_IJ = -(L_II)^-1 T
#pragma unroll 4
                    for (int k = 0; k < kTriNB; ++k) {
                        const double x = xs[k];
#pragma unroll
                        for (int q = 0; q < NQ; ++q) xo[q] -= sm.l[stage][row0 + RS * q][k] * x;
                    }
                }
            }
            __syncthreads();                                     // the stage and sm.x[step & 1] are free again
            if (next_x) {
#pragma unroll
                for (int q = 0; q < NX; ++q) {
                    const int t = threadIdx.x + NT * q;
                    sm.x[(step + 1) & 1][t >> 6][t & 63] = xr[q];
                }
            }
        }
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            const int gi = I * kTriNB + row0 + RS * q;
            sm.fresh[cc][row0 + RS * q] = xo[q];                 // read next as X_I (no reader is left from the previous block row)
            if (gi < m && gc < m) __stcg(Z + (size_t)gc * m + gi, xo[q]);
        }
        __syncthreads();                                         // the group's later block rows read Z (through L2) and sm.fresh
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
}

}  // namespace csd
