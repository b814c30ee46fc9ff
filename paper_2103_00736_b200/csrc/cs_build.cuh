// cs_build.cuh -- cs_create on the device (S 8(f) / VERDICT r1 item 7): validation, the two internally ordered
// compressed copies of A (one radix sort each), the slice fill, the heavy-row fusion marks and the fused rows' partition
// run as kernels on the uploaded CSR.  The host keeps what is O(m + n): the length ordering (counting sort), the prefix
// sums and the slice PLAN (make_sparse, cs_api.cu).  The layouts are bit-identical to the host build's (GPU test).
// The sort is CUB's DeviceRadixSort (a library primitive at set-up time, not on the hot path); everything else is
// hand-written.
#pragma once
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>

#include "cs_device.cuh"

namespace csb {

using csd::kChunk;
using csd::kFuseB;
using csd::kFuseK;
using csd::kShortMax;

// status bits of the validation
enum { kBadIndex = 1, kBadValue = 2, kZeroRow = 4, kEmptyRow = 8 };

// One warp per row of the caller's CSR (one CTA per row for the rows of the list `long_rows`, which the warp kernel skips):
// indices in range, strictly ascending, values finite, row norm > 0; column counts.
constexpr int kValidateLong = 8192;
__device__ __forceinline__ void validate_entries(const int *cidx, const double *val, int a, int b, int first, int stride, int n, int *clen,
                                                 int &bad, double &ss) {
    for (int e = a + first; e < b; e += stride) {
        const int j = cidx[e];
        const double v = val[e];
        if (j < 0 || j >= n || (e > a && j <= cidx[e - 1])) bad |= kBadIndex;
        else atomicAdd(clen + j, 1);
        if (!isfinite(v)) bad |= kBadValue;
        ss += v * v;
    }
}
__global__ void __launch_bounds__(256) k_validate(const int *rptr, const int *cidx, const double *val, int m, int n, int *clen, int *status) {
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * 256 + threadIdx.x) >> 5, nwarps = (gridDim.x * 256) >> 5;
    int bad = 0;
    for (int i = gwarp; i < m; i += nwarps) {
        const int a = rptr[i], b = rptr[i + 1];
        if (b <= a) { bad |= kEmptyRow; continue; }
        if (b - a > kValidateLong) continue;                         // k_validate_long
        double ss = 0.0;
        validate_entries(cidx, val, a, b, lane, 32, n, clen, bad, ss);
        ss = csd::group_reduce<32>(ss);
        if (!(ss > 0.0)) bad |= kZeroRow;
    }
    if (bad) atomicOr(status, bad);
}
__global__ void __launch_bounds__(256) k_validate_long(const int *rptr, const int *cidx, const double *val, const int *long_rows, int n_long,
                                                       int n, int *clen, int *status) {
    __shared__ double red[8];
    for (int q = blockIdx.x; q < n_long; q += gridDim.x) {
        const int i = long_rows[q], a = rptr[i], b = rptr[i + 1];
        int bad = 0;
        double ss = 0.0;
        validate_entries(cidx, val, a, b, (int)threadIdx.x, 256, n, clen, bad, ss);
        ss = csd::group_reduce<32>(ss);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int w = 0; w < 8; ++w) t += red[w];
            if (!(t > 0.0)) bad |= kZeroRow;
        }
        if (bad) atomicOr(status, bad);
    }
}

// length ordering: segments sorted by DECREASING length, stable (ties keep their index order) = an ascending stable radix sort of
// ~length; then the inverse permutation and the lengths in the new order (their exclusive scan is the new pointer array)
__global__ void k_len_keys(const int *ptr_or_len, int is_ptr, int n, unsigned *key, unsigned *iota) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int len = is_ptr ? ptr_or_len[i + 1] - ptr_or_len[i] : ptr_or_len[i];
        key[i] = 0xffffffffu - (unsigned)len;
        iota[i] = (unsigned)i;
    }
}
__global__ void k_iota_tail(int *perm, int from, int n) {
    for (int i = from + blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) perm[i] = i;
}
__global__ void k_invert_and_len(const int *perm, const int *ptr_or_len, int is_ptr, int n, int *inv, int *len_out) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= n; i += gridDim.x * blockDim.x) {
        if (i == n) { len_out[n] = 0; continue; }
        const int src = perm[i];
        inv[src] = i;
        len_out[i] = is_ptr ? ptr_or_len[src + 1] - ptr_or_len[src] : ptr_or_len[src];
    }
}

// sort keys of the two copies, one per stored entry e of row i (warp per row):
//   column-major: (internal column << 32) | internal row
//   row-major   : (internal row << 32) | (long row ? internal column : position in the row)   [short rows keep their order]
__global__ void __launch_bounds__(256) k_keys(const int *rptr, const int *cidx, int m, const int *inv_r, const int *inv_c,
                                              unsigned long long *key_c, unsigned long long *key_r, unsigned int *payload) {
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * 256 + threadIdx.x) >> 5, nwarps = (gridDim.x * 256) >> 5;
    for (int i = gwarp; i < m; i += nwarps) {
        const int a = rptr[i], b = rptr[i + 1];
        const unsigned long long ir = (unsigned long long)(unsigned)inv_r[i];
        const bool is_long = b - a > kShortMax;
        for (int e = a + lane; e < b; e += 32) {
            const unsigned jc = (unsigned)inv_c[cidx[e]];
            key_c[e] = ((unsigned long long)jc << 32) | ir;
            key_r[e] = (ir << 32) | (is_long ? jc : (unsigned)(e - a));
            payload[e] = (unsigned)e;
        }
    }
}

// compressed copies from the sorted keys: minor index = low word of the key (column-major) / internal column of the source
// entry (row-major), value = the source entry's
__global__ void k_gather_c(const unsigned long long *key_sorted, const unsigned int *src, const double *val, int nnz, int *ri2, double *cv2) {
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < nnz; q += gridDim.x * blockDim.x) {
        ri2[q] = (int)(unsigned)(key_sorted[q] & 0xffffffffull);
        cv2[q] = val[src[q]];
    }
}
__global__ void k_gather_r(const unsigned int *src, const int *cidx, const double *val, const int *inv_c, int nnz, int *ci2, double *va2) {
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < nnz; q += gridDim.x * blockDim.x) {
        const unsigned e = src[q];
        ci2[q] = inv_c[cidx[e]];
        va2[q] = val[e];
    }
}

// ---- slice fill: the device twin of make_sparse's fill (cs_api.cu); one warp per slice ----------------------------------
// chunk slices: entry e of the chunk at slot off + e (lane e % 32, row e / 32); short slices: lane -> segment s0 + lane / T,
// its entry k T + lane % T in slice row k.  Padding: value 0, a valid index replicated.  pos[compressed entry] = slot.
// With n_fuse > 0 (column-major copy): fused marks as in make_sparse -- class A always, class B only in the lowest lane of
// the slice that holds the row; fmask byte per lane, bit 16 of the slice descriptor, fused[compressed entry] = 1.
__global__ void __launch_bounds__(256) k_fill_slices(int4 *slices, int n_slice, int n_chunk, const int *chunk_src, const int *chunk_len,
                                                     const int *ptr, const int *cidx, const double *cval, int *idx, double *val0, int *pos,
                                                     int n_fuse, int n_fa, unsigned char *fmask, unsigned char *fused) {
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * 256 + threadIdx.x) >> 5, nwarps = (gridDim.x * 256) >> 5;
    for (int si = gwarp; si < n_slice; si += nwarps) {
        const int4 sl = slices[si];
        const size_t off = (size_t)sl.x;
        const int width = sl.w;
        if (si < n_chunk) {
            const int a = chunk_src[si], clen = chunk_len[si];
            for (int e = lane; e < 32 * width; e += 32) {
                idx[off + e] = cidx[a + min(e, clen - 1)];
                val0[off + e] = e < clen ? cval[a + e] : 0.0;
                if (e < clen) pos[a + e] = (int)(off + e);
            }
            continue;
        }
        const int cnt = sl.z & 255, lgT = (sl.z >> 8) & 7, T = 1 << lgT, s0 = sl.y;
        const int seg = s0 + min(lane >> lgT, cnt - 1), t = lane & (T - 1);
        const int p0 = ptr[seg], len = ptr[seg + 1] - p0;
        for (int k = 0; k < width; ++k) {
            const int e = k * T + t;
            const bool valid = (lane >> lgT) < cnt && e < len;
            idx[off + 32u * k + lane] = len > 0 ? cidx[p0 + min(e, len - 1)] : 0;
            val0[off + 32u * k + lane] = valid ? cval[p0 + e] : 0.0;
            if (valid) pos[p0 + e] = (int)(off + 32u * k + lane);
        }
        if (n_fuse && lgT == 0) {
            // rows of this lane's column among its first kFuseK entries that are fused rows (rows ascend within a column)
            int mine[kFuseK];
#pragma unroll
            for (int k = 0; k < kFuseK; ++k) {
                const int i = (lane < cnt && k < len) ? cidx[p0 + k] : 0x7fffffff;
                mine[k] = i < n_fuse ? i : -1;
            }
#pragma unroll
            for (int k = 1; k < kFuseK; ++k) if (mine[k - 1] < 0) mine[k] = -1;     // stop at the first row >= n_fuse
            unsigned char fb = 0;
#pragma unroll
            for (int k = 0; k < kFuseK; ++k) {
                bool take = mine[k] >= 0;
                // class B: not if a LOWER lane holds this row in any of its positions (every lane takes part in the shuffles)
                for (int src = 0; src < 31; ++src) {
#pragma unroll
                    for (int k2 = 0; k2 < kFuseK; ++k2) {
                        const int other = __shfl_sync(0xffffffffu, mine[k2], src);
                        if (take && mine[k] >= n_fa && src < lane && other == mine[k]) take = false;
                    }
                }
                if (take) { fb |= (unsigned char)(1u << k); fused[p0 + k] = 1; }
            }
            fmask[(size_t)(si - n_chunk) * 32 + lane] = fb;
            if (__any_sync(0xffffffffu, fb != 0) && lane == 0) slices[si].z = sl.z | (1 << 16);
        }
    }
}

// ---- fused rows of the row-major copy: unfused entries first, fused ones behind them (each part keeps its order) ---------
// flag[e] = 1 if entry e of fused row r (e < rp2[n_fuse]) was marked in the column-major copy (rows ascend within a column,
// so row r sits among the first entries of its column); flag[rp2[n_fuse]] = 0 closes the scan.
__global__ void k_fused_flags(const int *rp2, const int *ci2, const int *cp2, const int *ri2, const unsigned char *fused_c, int n_fuse, int *flag) {
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    for (int r = 0; r < n_fuse; ++r)
        for (int e = rp2[r] + gwarp * 32 + lane; e < rp2[r + 1]; e += nwarps * 32) {
            const int j = ci2[e];
            int f = 0;
            for (int q = cp2[j]; q < cp2[j + 1]; ++q) {
                const int i = ri2[q];
                if (i == r) { f = fused_c[q]; break; }
                if (i > r) break;
            }
            flag[e] = f;
        }
    if (blockIdx.x == 0 && threadIdx.x == 0) flag[rp2[n_fuse]] = 0;
}
// sc = exclusive scan of flag over [0, rp2[n_fuse]]; split[r] = unfused entries of row r
__global__ void k_fused_partition(const int *rp2, const int *flag, const int *sc, int n_fuse, const int *ci2, const double *va2,
                                  int *ci2_out, double *va2_out, int *split) {
    const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    for (int r = 0; r < n_fuse; ++r) {
        const int base = rp2[r], end = rp2[r + 1], nf = sc[end] - sc[base], sp = (end - base) - nf;
        if (tid == 0) split[r] = sp;
        for (int e = base + tid; e < end; e += nth) {
            const int fb = sc[e] - sc[base];
            const int dst = flag[e] ? base + sp + fb : base + (e - base - fb);
            ci2_out[dst] = ci2[e];
            va2_out[dst] = va2[e];
        }
    }
}

// initial vectors: v = value; e_K = 1 on the orthant coordinates and on every Lorentz block's first coordinate
__global__ void k_fill(double *v, int n, double value) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) v[i] = value;
}
__global__ void k_unit_cone_point(double *x, double *z, int n, int n_lin, const int *cone_off, int n_soc) {
    const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    for (int j = tid; j < n; j += nth) { const double v = j < n_lin ? 1.0 : 0.0; x[j] = v; z[j] = v; }
    __threadfence();                                     // (the heads are written by a second launch, see the caller)
}
__global__ void k_unit_cone_heads(double *x, double *z, const int *cone_off, int n_soc) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_soc; i += gridDim.x * blockDim.x) { x[cone_off[i]] = 1.0; z[cone_off[i]] = 1.0; }
}

}  // namespace csb
