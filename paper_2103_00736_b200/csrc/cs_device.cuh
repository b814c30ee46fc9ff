// cs_device.cuh -- device-side building blocks of libcs.so (sm_100a, fp64).
//
// Everything here runs inside persistent COOPERATIVE kernels: one launch covers many phases that
// are separated by grid-wide barriers, so that the scalars of the inner CG (alpha, beta, residual
// norms) and its exit test never leave the device.  Citations P:<line> = /root/reference/PAPER.md.
#pragma once
#include <cooperative_groups.h>
#include <cstdint>

namespace cg = cooperative_groups;

namespace csd {

#ifndef CS_UN
#define CS_UN 8
#endif
#ifndef CS_MINB
#define CS_MINB 2
#endif
constexpr int kBlock = 512;          // threads per CTA (16 warps)
constexpr int kWarps = kBlock / 32;
constexpr int kMaxRed = 8;           // scalars per grid reduction
constexpr int kShortMax = 64;        // segments up to this many non-zeros are "short" (sub-warp groups)
constexpr int kChunk = 1024;         // long segments are cut into warp-sized chunks of this many non-zeros
constexpr int kConeLanes = 8;        // lanes cooperating on one Lorentz cone

// One sparse format (rows of the CSR-like copy or columns of the CSC-like copy), stored in two parts:
//  * ELL part: runs of consecutive short segments cut into slices of 32; slice s holds 32 x width
//    entries laid out [k][lane] so that lane l reads entry k of segment seg0+l at off + 32k + l
//    (fully coalesced, one thread per segment, no shuffles).  Padding entries have val = 0 and a valid
//    index.  Rows (and orthant columns) are physically sorted by length at cs_create, so padding is
//    negligible.
//  * long part: segments longer than kShortMax, cut into chunks of kChunk entries, one warp each;
//    segments spanning several chunks are finished from per-chunk partial sums in fixed order.
struct Sparse {
    int n_slice;
    const int4 *slices;     // {offset into e*, first segment id, segments in the slice | log2(T) << 8, width};
                            // T = lanes per segment (1,2,4,8): entry e of segment r sits at lane r*T + e%T, row e/T
    const int *eidx;
    double *eval;           // scaled values (D A O)
    const double *eval0;    // pristine values (A)
    int n_chunk;
    const int4 *chunks;     // {segment id, first entry in l*, length, slot}; slot < 0: chunk == whole segment
    const int *lidx;
    double *lval;
    const double *lval0;
    int n_multi;
    const int4 *multi;      // {segment id, first slot, number of slots, 0}
    double *partial;        // [slots][2]
};

struct Scalars {            // device-resident state scalars (read back only by cs_residuals)
    double resid[16];
    long long iter, cg_steps_total, cg_steps_cond;
    int cg_steps_last, n_cond, cg_hit_max, pad;
    double fp_res2;         // ||s_new - s||^2 of the last pass
    unsigned long long phase_ns[8];  // time spent per phase id (kPh*), measured by CTA 0 between grid barriers
};

enum { kPhCone = 0, kPhRhs = 1, kPhK1 = 2, kPhK2 = 3, kPhUpdate = 4, kPhReduce = 5, kPhCondition = 6, kPhResid = 7 };

struct Ctx {
    int m, n, n_lin, n_soc;
    const int *cone_off;    // [n_soc+1] absolute offsets of the Lorentz blocks (cone_off[0] = n_lin)
    const int *perm_r, *perm_c;  // internal index -> caller's index (rows / columns sorted by length)
    Sparse R, C;            // row-major (segments = rows) and column-major (segments = columns) copies of A
    // n-vectors
    double *s, *p, *g, *e, *u, *d, *chat, *O, *xb, *zb;
    const double *c;
    // m-vectors
    double *w, *r, *v, *wd, *D, *btil;
    const double *b;
    double *partials;       // [2][kMaxRed][gridDim]
    Scalars *sc;
    double mu, t, o_floor, cg_tol;
    int cg_max_iter;
    double norm_b, norm_c;
    int dbg;                // TEMP debug flags
    int hot_rows;           // leading (longest) rows whose r / w entries are cached in shared memory for the column passes
};

// ---------------------------------------------------------------------------------------------
// warp / group reductions (xor butterfly: every lane ends with the same bits)
// ---------------------------------------------------------------------------------------------
struct OpSum { __device__ static double f(double a, double b) { return a + b; } };
struct OpMax { __device__ static double f(double a, double b) { return fmax(a, b); } };

template <int W, class Op = OpSum>
__device__ __forceinline__ double group_reduce(double v) {
#pragma unroll
    for (int o = W / 2; o > 0; o >>= 1) v = Op::f(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

struct GridCtl {            // per-thread view of the grid barrier state (uniform over the grid)
    cg::grid_group grid;
    int parity;
    double *partials;
    double *smem;           // [kMaxRed * kWarps]
    unsigned long long t_last, ns[8];
    __device__ GridCtl(double *partials_, double *smem_) : grid(cg::this_grid()), parity(0), partials(partials_), smem(smem_) {
#pragma unroll
        for (int i = 0; i < 8; ++i) ns[i] = 0;
        t_last = now();
    }
    __device__ void sync() { grid.sync(); }
    __device__ static unsigned long long now() {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        return t;
    }
    // charge the time since the previous lap to phase `id` (only CTA 0 / thread 0 keeps the books)
    __device__ void lap(int id) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            const unsigned long long t = now();
            ns[id] += t - t_last;
            t_last = t;
        }
    }
    __device__ void flush(Scalars *sc) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
#pragma unroll
            for (int i = 0; i < 8; ++i) sc->phase_ns[i] += ns[i];
        }
    }
};

// Deterministic grid-wide reduction of NR per-thread values; includes ONE grid barrier.
// Every thread of every CTA returns the same bits.
template <int NR, class Op = OpSum>
__device__ void grid_reduce(double (&v)[NR], GridCtl &gc, double ident = 0.0) {
    static_assert(NR <= kMaxRed, "too many scalars");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < NR; ++i) {
        double x = group_reduce<32, Op>(v[i]);
        if (lane == 0) gc.smem[i * kWarps + warp] = x;
    }
    __syncthreads();
    double *buf = gc.partials + (size_t)gc.parity * kMaxRed * gridDim.x;
    if (threadIdx.x < NR) {
        double acc = gc.smem[threadIdx.x * kWarps];
        for (int w = 1; w < kWarps; ++w) acc = Op::f(acc, gc.smem[threadIdx.x * kWarps + w]);
        buf[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = acc;
    }
    gc.grid.sync();
    if (warp < NR) {
        double acc = ident;
        for (int b = lane; b < (int)gridDim.x; b += 32) acc = Op::f(acc, __ldcg(buf + (size_t)warp * gridDim.x + b));
        acc = group_reduce<32, Op>(acc);
        if (lane == 0) gc.smem[warp] = acc;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < NR; ++i) v[i] = gc.smem[i];
    __syncthreads();
    gc.parity ^= 1;
}

// ---------------------------------------------------------------------------------------------
// Segment traversals.  `term(a, j, acc)` adds the contribution of one entry (value a, minor index j)
// to acc[NV]; `epi(seg, sums)` is called once per segment with the complete sums.
// Long segments first (warp per chunk), then the ELL slices (thread per segment), then the segments
// that span several chunks (after a grid barrier, from their partial sums, in fixed order).
// The matrix streams use ld.global.cs (evict-first) so that the gathered vectors stay in L2.
// ---------------------------------------------------------------------------------------------
template <int NV, bool PRISTINE, class Term, class Epi>
__device__ __forceinline__ void seg_reduce(const Sparse &S, Term &term, Epi &epi, GridCtl &gc, int dbg = 0) {
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * kBlock + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * kBlock) >> 5;
    {
        const double *lv = PRISTINE ? S.lval0 : S.lval;
        for (int c = gwarp; c < ((dbg & 2) ? 0 : S.n_chunk); c += nwarps) {
            const int4 ch = __ldg(S.chunks + c);
            double acc[NV];
#pragma unroll
            for (int i = 0; i < NV; ++i) acc[i] = 0.0;
            const int end = ch.y + ch.z;
            constexpr int CU = 8;
            for (int k = ch.y + lane; k < end; k += 32 * CU) {
                double a[CU]; int j[CU];
#pragma unroll
                for (int q = 0; q < CU; ++q) {
                    const bool ok = k + 32 * q < end;
                    a[q] = ok ? __ldcs(lv + k + 32 * q) : 0.0;
                    j[q] = ok ? __ldcs(S.lidx + k + 32 * q) : -1;
                }
#pragma unroll
                for (int q = 0; q < CU; ++q) if (j[q] >= 0) term(a[q], j[q], acc);
            }
#pragma unroll
            for (int i = 0; i < NV; ++i) acc[i] = group_reduce<32>(acc[i]);
            if (lane == 0) {
                if (ch.w < 0) epi(ch.x, acc, epi.pre(ch.x));
                else {
#pragma unroll
                    for (int i = 0; i < NV; ++i) S.partial[(size_t)ch.w * 2 + i] = acc[i];
                }
            }
        }
    }
    {
        // ELL slices: one thread per segment.  All loads of a slice row-block are issued before the
        // first use (predicated 8-wide unroll), the operands of the epilogue are fetched up front
        // (epi.pre) and the next slice descriptor is prefetched, so that a warp keeps ~20 independent
        // loads in flight instead of a chain of dependent round trips.
        constexpr int UN = CS_UN;
        const double *ev = PRISTINE ? S.eval0 : S.eval;
        int s = gwarp;
        int4 sl = s < S.n_slice ? __ldg(S.slices + s) : make_int4(0, 0, 0, 0);
        if (dbg & 4) s = S.n_slice;
        while (s < S.n_slice) {
            const int sn = s + nwarps;
            const int4 nxt = sn < S.n_slice ? __ldg(S.slices + sn) : make_int4(0, 0, 0, 0);
            const double *vp = ev + sl.x + lane;
            const int *ip = S.eidx + sl.x + lane;
            const int lgT = sl.z >> 8, T = 1 << lgT;              // lanes per segment in this slice
            const int seg = sl.y + (lane >> lgT);
            const bool head = (lane >> lgT) < (sl.z & 255) && (lane & (T - 1)) == 0;
            typename Epi::Pre pre = epi.pre(head ? seg : sl.y);
            double acc[NV];
#pragma unroll
            for (int i = 0; i < NV; ++i) acc[i] = 0.0;
            for (int k = 0; k < sl.w; k += UN) {
                double a[UN]; int j[UN];
#pragma unroll
                for (int q = 0; q < UN; ++q) {
                    const bool ok = k + q < sl.w;
                    a[q] = ok ? __ldcs(vp + 32 * (k + q)) : 0.0;
                    j[q] = ok ? __ldcs(ip + 32 * (k + q)) : -1;
                }
#pragma unroll
                for (int q = 0; q < UN; ++q) if (j[q] >= 0) term(a[q], j[q], acc);
            }
            for (int o = T >> 1; o > 0; o >>= 1) {
#pragma unroll
                for (int i = 0; i < NV; ++i) acc[i] += __shfl_xor_sync(0xffffffffu, acc[i], o);
            }
            if (head) epi(seg, acc, pre);
            s = sn;
            sl = nxt;
        }
    }
    if (S.n_multi && !(dbg & 8)) {
        gc.sync();
        for (int r = gwarp; r < S.n_multi; r += nwarps) {
            const int4 mr = __ldg(S.multi + r);
            double acc[NV];
#pragma unroll
            for (int i = 0; i < NV; ++i) {
                double a = 0.0;
                const double *pp = S.partial + (size_t)mr.y * 2 + i;
                int k = lane;
                for (; k + 224 < mr.z; k += 256) {       // 8 independent loads in flight
                    double t[8];
#pragma unroll
                    for (int q = 0; q < 8; ++q) t[q] = __ldcg(pp + (size_t)(k + 32 * q) * 2);
#pragma unroll
                    for (int q = 0; q < 8; ++q) a += t[q];
                }
                for (; k < mr.z; k += 32) a += __ldcg(pp + (size_t)k * 2);
                acc[i] = group_reduce<32>(a);
            }
            if (lane == 0) epi(mr.x, acc, epi.pre(mr.x));
        }
    }
}

// Rewrite every stored entry: val = f(seg, val0, idx).  Same partition as seg_reduce.
template <class F>
__device__ __forceinline__ void seg_rescale(const Sparse &S, F &f) {
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * kBlock + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * kBlock) >> 5;
    for (int c = gwarp; c < S.n_chunk; c += nwarps) {
        const int4 ch = __ldg(S.chunks + c);
        for (int k = ch.y + lane; k < ch.y + ch.z; k += 32) S.lval[k] = f(ch.x, S.lval0[k], __ldg(S.lidx + k));
    }
    for (int s = gwarp; s < S.n_slice; s += nwarps) {
        const int4 sl = __ldg(S.slices + s);
        const int lgT = sl.z >> 8;
        if ((lane >> lgT) < (sl.z & 255)) {
            const int base = sl.x + lane, seg = sl.y + (lane >> lgT);
            for (int k = 0; k < sl.w; ++k) S.eval[base + 32 * k] = f(seg, S.eval0[base + 32 * k], __ldg(S.eidx + base + 32 * k));
        }
    }
}

}  // namespace csd
