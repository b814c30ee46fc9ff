// cs_dense.cuh -- dense factor-apply path for problems on many CTAs (B north_star: "a dense factor-apply kernel only
// where A is small enough that it is truly a dense contraction"; S 8(f).3: the paper's own dense shapes, section V-A
// P:342-346 and V-D P:366-371).  For a dense-stored A with m <= kDenseGridMax:
//   at every conditioning   Ad = A~ (m x n, row-major)          k_dense_scatter
//                           M  = Ad Ad'                          k_dense_aat        (unit diagonal: A~ is row-equilibrated)
//                           M  = L L'   (blocked, right-looking) k_chol_diag / k_chol_panel / k_chol_update
//                           Z  = L^-T   (row j = column j of L^-1)  k_dense_transpose_lower, k_dense_trinv
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
__global__ void __launch_bounds__(256) k_dense_aat(const double *A, int r, int k, double *C) {
    __shared__ double sa[16][65], sb[16][65];
    // tile (ti, tj) with tj <= ti from the linear block index
    int ti = (int)((sqrt(8.0 * blockIdx.x + 1.0) - 1.0) * 0.5);
    while ((ti + 1) * (ti + 2) / 2 <= (int)blockIdx.x) ++ti;
    while (ti * (ti + 1) / 2 > (int)blockIdx.x) --ti;
    const int tj = blockIdx.x - ti * (ti + 1) / 2;
    const int a0 = ti * 64, b0 = tj * 64, tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    double acc[4][4] = {};
    for (int k0 = 0; k0 < k; k0 += 16) {
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

// Lt = L' (upper triangle, row-major): the triangular inverse below reads L by columns
__global__ void __launch_bounds__(256) k_dense_transpose_lower(const double *L, int m, double *Lt) {
    __shared__ double tile[32][33];
    const int bx = blockIdx.x * 32, by = blockIdx.y * 32, tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    if (bx > by + 31) return;                                    // tile entirely above the diagonal of L: nothing stored there
    for (int r = ty; r < 32; r += 8) {
        const int i = by + r, k = bx + tx;
        tile[r][tx] = (i < m && k < m && k <= i) ? L[(size_t)i * m + k] : 0.0;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int k = bx + r, i = by + tx;
        if (k < m && i < m) Lt[(size_t)k * m + i] = tile[tx][r];
    }
}

// Z = L^-T, row j = column j of L^-1: one warp per column j solves L x = e_j forwards, 32 rows at a time.  Lane r owns
// row i = i0 + r of the block: first s_r = sum_{k < i0} L[i][k] x[k] -- a loop over k with no dependence between its
// iterations (Lt[k][i0 + lane] is one coalesced load, x[k] a broadcast) -- then the 32 x 32 diagonal block is solved inside
// the warp with shuffles.  The dependent chain through memory is m/32 steps long instead of m (14.7 -> 6.9 ms at m = 2320;
// what is left is L2 traffic: every column streams the part of L' below it, 4 m^3 / 3 bytes in all -- a tile-sharing blocked
// inverse is the next step).  Z zeroed by the caller (x_k = 0 for k < j).  Fixed summation order.
__global__ void __launch_bounds__(256) k_dense_trinv(const double *Lt, int m, double *Z) {
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * 256 + threadIdx.x) >> 5, nwarps = (gridDim.x * 256) >> 5;
    for (int j = gwarp; j < m; j += nwarps) {
        double *x = Z + (size_t)j * m;
        for (int i0 = j & ~31; i0 < m; i0 += 32) {
            const int i = i0 + lane;
            double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
            int k = j;
            if (i < m) {
                for (; k + 3 < i0; k += 4) {
                    s0 += Lt[(size_t)k * m + i] * __ldcg(x + k);
                    s1 += Lt[(size_t)(k + 1) * m + i] * __ldcg(x + k + 1);
                    s2 += Lt[(size_t)(k + 2) * m + i] * __ldcg(x + k + 2);
                    s3 += Lt[(size_t)(k + 3) * m + i] * __ldcg(x + k + 3);
                }
                for (; k < i0; ++k) s0 += Lt[(size_t)k * m + i] * __ldcg(x + k);
            }
            double rhs = (i == j ? 1.0 : 0.0) - ((s0 + s1) + (s2 + s3));
            const double dg = i < m ? Lt[(size_t)i * m + i] : 1.0;
            for (int cidx = 0; cidx < 32 && i0 + cidx < m; ++cidx) {     // x_c = rhs_c / L_cc ; rhs_r -= L[r][c] x_c for r > c
                const double xc = __shfl_sync(0xffffffffu, rhs, cidx) / __shfl_sync(0xffffffffu, dg, cidx);
                if (lane == cidx) rhs = xc;
                else if (lane > cidx && i < m) rhs -= Lt[(size_t)(i0 + cidx) * m + i] * xc;
            }
            if (i < m && i >= j) __stcg(x + i, rhs);
            __syncwarp();                                        // the next block reads x[i0 .. i0+32) (through L2: __stcg / __ldcg)
        }
    }
}

}  // namespace csd
