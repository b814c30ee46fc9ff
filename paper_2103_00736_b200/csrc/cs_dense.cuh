// cs_dense.cuh -- dense factor-apply path for problems on many CTAs (B north_star: "a dense factor-apply kernel only
// where A is small enough that it is truly a dense contraction"; S 8(f).3: the paper's own dense shapes, section V-A
// P:342-346 and V-D P:366-371).  For a dense-stored A with m <= kDenseGridMax:
//   at every conditioning   Ad = A~ (m x n, row-major)          k_dense_scatter
//                           M  = Ad Ad'                          k_dense_aat        (unit diagonal: A~ is row-equilibrated)
//                           M  = L L'   (blocked, right-looking) k_chol_diag / k_chol_panel / k_chol_update
//                           Z  = L^-T   (row j = column j of L^-1)  k_dense_diag_inv, k_dense_trinv_blk
//                           Minv = Z Z' = M^-1                   k_dense_aat
//   at every pass           w += M^-1 r by dense_apply_grid (cs_kernels.cuh): x = Minv r, then kDenseRefine steps of
//                           iterative refinement x += Minv (r - M x) against the stored M -- dense GEMVs only.
// All sums have a fixed order (no atomics).  fp64 throughout; plain DFMA (no tensor cores: B200's fp64 tensor rate equals
// its vector rate and the matrices are a few thousand wide).
#pragma once
#include "cs_device.cuh"

namespace csd {

constexpr int kDenseGridMax = 4096;  // largest m of the grid dense path (4 m x m fp64 matrices = 537 MB at the limit)
constexpr int kDenseRefine = 2;      // refinement steps of the per-pass apply
constexpr int kCholNB = 32;          // panel width of the blocked Cholesky

// Ad[i][j] = A~_ij from the row-major slice copy (Ad zeroed by the caller)
__global__ void k_dense_scatter(Ctx c, double *Ad) {
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    for (int i = gwarp; i < c.m; i += nwarps)
        for (int e = c.Rc.ptr[i] + lane; e < c.Rc.ptr[i + 1]; e += 32) Ad[(size_t)i * c.n + c.Rc.idx[e]] = c.R.val[c.Rc.pos[e]];
}

// C = A A' for a row-major A [r][k]; C [r][r] full (both triangles written).  One CTA of 256 threads per 64 x 64 tile
// of the lower triangle, 4 x 4 outputs per thread, the k range consumed 16 at a time through shared memory.
// tri != 0: A is upper triangular (A[a][i] = 0 for i < a, k = r), so the sum starts at the tile's first row (Minv = Z Z').
__global__ void __launch_bounds__(256) k_dense_aat(const double *A, int r, int k, double *C, int tri) {
    __shared__ double sa[16][65], sb[16][65];
    // tile (ti, tj) with tj <= ti from the linear block index
    int ti = (int)((sqrt(8.0 * blockIdx.x + 1.0) - 1.0) * 0.5);
    while ((ti + 1) * (ti + 2) / 2 <= (int)blockIdx.x) ++ti;
    while (ti * (ti + 1) / 2 > (int)blockIdx.x) --ti;
    const int tj = blockIdx.x - ti * (ti + 1) / 2;
    const int a0 = ti * 64, b0 = tj * 64, tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    double acc[4][4] = {};
    for (int k0 = tri ? a0 : 0; k0 < k; k0 += 16) {              // a0 >= b0: both operands are zero before column a0
        for (int q = threadIdx.x; q < 64 * 16; q += 256) {       // rows of the tile x 16 columns: 128-byte row pieces
            const int row = q >> 4, col = q & 15;
            const bool okc = k0 + col < k;
            sa[col][row] = (okc && a0 + row < r) ? A[(size_t)(a0 + row) * k + k0 + col] : 0.0;
            sb[col][row] = (okc && b0 + row < r) ? A[(size_t)(b0 + row) * k + k0 + col] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < 16; ++kk) {
            double va[4], vb[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) { va[i] = sa[kk][ty * 4 + i]; vb[i] = sb[kk][tx * 4 + i]; }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] += va[i] * vb[j];
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int a = a0 + ty * 4 + i, b = b0 + tx * 4 + j;
            if (a < r && b < r) {
                C[(size_t)a * r + b] = acc[i][j];
                if (ti != tj) C[(size_t)b * r + a] = acc[i][j];
            }
        }
}

// ---- blocked right-looking Cholesky of L (m x m row-major, lower triangle used; starts as a copy of M) -------------
// step kb: (1) k_chol_diag factors the nb x nb diagonal block in shared memory (one CTA); a pivot <= 1e-12 (diag(M) = 1:
//              a relative test) clears *ok and is replaced by 1 so that the run stays finite (the caller falls back to CG)
//          (2) k_chol_panel: rows below the block, X D' = L[i][kb:kb+nb] -- one warp per row, lane c owns column c
//          (3) k_chol_update: trailing L[i][j] -= sum_c P[i][c] P[j][c] (j <= i), 64 x 64 tiles, 4 x 4 per thread
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

__global__ void __launch_bounds__(256) k_chol_update(double *L, int m, int kb) {
    __shared__ double pi[kCholNB][65], pj[kCholNB][65];
    const int nb = min(kCholNB, m - kb), base = kb + nb;
    int ti = (int)((sqrt(8.0 * blockIdx.x + 1.0) - 1.0) * 0.5);
    while ((ti + 1) * (ti + 2) / 2 <= (int)blockIdx.x) ++ti;
    while (ti * (ti + 1) / 2 > (int)blockIdx.x) --ti;
    const int tj = blockIdx.x - ti * (ti + 1) / 2;
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
            if (a < m && b <= a) L[(size_t)a * m + b] -= acc[i][j];
        }
}

// ---- Z = L^-T (row j of Z = column j of L^-1), blocked ---------------------------------------------------------------
// Column j of X = L^-1 depends on L only, so column groups are independent; inside a group the block rows follow one
// another:  X_JJ = (L_JJ)^-1,   X_IJ = -(L_II)^-1 sum_{K=J}^{I-1} L_IK X_KJ   (64 x 64 blocks of L).
// k_dense_diag_inv inverts every diagonal block once; k_dense_trinv_blk gives one CTA a group of kTriCW columns and walks
// the block rows with 64 x 64 tiles of L in shared memory (each tile serves 64 x kTriCW x 64 multiply-adds, so L is read
// m / (3 kTriCW) times from L2 instead of m / 3 times: 6.9 -> ~1 ms at m = 2320).  Heaviest groups (J = 0) have the
// lowest block indices and start first.  Fixed summation order; Z zeroed by the caller (x_i = 0 for i < j's block).
constexpr int kTriNB = 64, kTriCW = 8;

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

__global__ void __launch_bounds__(128) k_dense_trinv_blk(const double *L, const double *Dinv, int m, double *Z) {
    __shared__ __align__(16) double sl[kTriNB][kTriNB + 2];      // a tile of L, or (L_II)^-1
    __shared__ double sx[kTriNB][kTriCW + 1];                    // the matching rows of X for this group's columns, or T
    const int c0 = blockIdx.x * kTriCW, J = c0 / kTriNB, nblk = (m + kTriNB - 1) / kTriNB;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, cc = lane & (kTriCW - 1), rh = lane / kTriCW;
    const int gc = c0 + cc;                                      // this thread's column of L^-1 = row of Z
    int row[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) row[q] = 16 * w + rh + 4 * q;    // its four rows of the block row
    for (int I = J; I < nblk; ++I) {
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        for (int K = J; K < I; ++K) {                            // T = sum_K L_IK X_KJ
            for (int t = threadIdx.x; t < kTriNB * kTriNB; t += 128) {
                const int r = t >> 6, k = t & 63, gi = I * kTriNB + r;
                sl[r][k] = gi < m ? L[(size_t)gi * m + K * kTriNB + k] : 0.0;
            }
            for (int t = threadIdx.x; t < kTriNB * kTriCW; t += 128) {
                const int c = t >> 6, k = t & 63;
                sx[k][c] = c0 + c < m ? __ldcg(Z + (size_t)(c0 + c) * m + K * kTriNB + k) : 0.0;
            }
            __syncthreads();
#pragma unroll 8
            for (int k = 0; k < kTriNB; ++k) {
                const double x = sx[k][cc];
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[q] += sl[row[q]][k] * x;
            }
            __syncthreads();
        }
        for (int t = threadIdx.x; t < kTriNB * kTriNB; t += 128)
            sl[t >> 6][t & 63] = Dinv[(size_t)I * kTriNB * kTriNB + t];
        double xo[4] = {0.0, 0.0, 0.0, 0.0};
        if (I == J) {                                            // X_JJ: the group's columns of (L_JJ)^-1
            __syncthreads();
#pragma unroll
            for (int q = 0; q < 4; ++q) xo[q] = sl[row[q]][gc - J * kTriNB];
        } else {                                                 // X_IJ = -(L_II)^-1 T
#pragma unroll
            for (int q = 0; q < 4; ++q) sx[row[q]][cc] = acc[q];
            __syncthreads();
#pragma unroll 8
            for (int k = 0; k < kTriNB; ++k) {
                const double x = sx[k][cc];
#pragma unroll
                for (int q = 0; q < 4; ++q) xo[q] -= sl[row[q]][k] * x;
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int gi = I * kTriNB + row[q];
            if (gi < m && gc < m) __stcg(Z + (size_t)gc * m + gi, xo[q]);
        }
        __syncthreads();                                         // the group's later block rows read these (through L2)
    }
}

}  // namespace csd
