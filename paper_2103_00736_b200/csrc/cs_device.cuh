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

constexpr int kBlock = 512;          // threads per CTA (16 warps)
constexpr int kWarps = kBlock / 32;
constexpr int kMaxRed = 8;           // scalars per grid reduction
constexpr int kShortMax = 64;        // segments up to this many non-zeros are "short" (sub-warp groups)
constexpr int kChunk = 1024;         // long segments are cut into warp-sized chunks of this many non-zeros
constexpr int kConeLanes = 8;        // lanes cooperating on one Lorentz cone

// Work partition of one sparse format (rows of the CSR copy or columns of the CSC copy).
struct Bins {
    int n_short;            // number of short segments
    const int *short_ids;   // their ids, or nullptr when every segment is short (identity)
    int G;                  // lanes per short segment: 4, 8, 16 or 32
    int n_chunk;            // chunks of long segments, one warp each
    const int4 *chunks;     // {segment id, first nnz, length, slot}; slot < 0: chunk == whole segment
    int n_multi;            // long segments spanning several chunks
    const int4 *multi;      // {segment id, first slot, number of slots, 0}
    double *partial;        // one partial sum per slot
};

struct Sparse {             // one compressed format: segment pointers, minor indices, values
    const int *ptr;
    const int *idx;
    double *val;            // scaled values  (D A O)
    const double *val0;     // pristine values (A)
    Bins bins;
};

struct Scalars {            // device-resident state scalars (read back only by cs_residuals)
    double resid[16];
    long long iter, cg_steps_total, cg_steps_cond;
    int cg_steps_last, n_cond, cg_hit_max, pad;
    double fp_res2;         // ||s_new - s||^2 of the last pass
};

struct Ctx {
    int m, n, n_lin, n_soc;
    const int *cone_off;    // [n_soc+1] absolute offsets of the Lorentz blocks (cone_off[0] = n_lin)
    Sparse R, C;            // CSR (segments = rows) and CSC (segments = columns) copies of A
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
    __device__ GridCtl(double *partials_, double *smem_) : grid(cg::this_grid()), parity(0), partials(partials_), smem(smem_) {}
    __device__ void sync() { grid.sync(); }
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
// Segment traversals.  `term(k, out)` adds the contribution of non-zero k to out[NV];
// `epi(seg, sums)` is called by ONE lane per segment with the complete sums.
// Long segments first (warp per chunk), then short segments (G lanes each), then the segments that
// span several chunks (after a grid barrier, from their per-chunk partial sums, in fixed order).
// ---------------------------------------------------------------------------------------------
template <int NV, int G, class Term, class Epi>
__device__ __forceinline__ void seg_reduce_G(const Sparse &S, Term &term, Epi &epi, GridCtl &gc) {
    const Bins &B = S.bins;
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * kBlock + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * kBlock) >> 5;
    for (int c = gwarp; c < B.n_chunk; c += nwarps) {
        const int4 ch = __ldg(B.chunks + c);
        double acc[NV];
#pragma unroll
        for (int i = 0; i < NV; ++i) acc[i] = 0.0;
        for (int k = ch.y + lane; k < ch.y + ch.z; k += 32) term(k, acc);
#pragma unroll
        for (int i = 0; i < NV; ++i) acc[i] = group_reduce<32>(acc[i]);
        if (lane == 0) {
            if (ch.w < 0) epi(ch.x, acc);
            else {
#pragma unroll
                for (int i = 0; i < NV; ++i) B.partial[(size_t)ch.w * NV + i] = acc[i];
            }
        }
    }
    constexpr int SPW = 32 / G;
    const int sub = lane / G, sl = lane % G;
    for (int base = gwarp * SPW; base < B.n_short; base += nwarps * SPW) {
        const int si = base + sub;
        int seg = -1;
        double acc[NV];
#pragma unroll
        for (int i = 0; i < NV; ++i) acc[i] = 0.0;
        if (si < B.n_short) {
            seg = B.short_ids ? __ldg(B.short_ids + si) : si;
            const int a = __ldg(S.ptr + seg), b = __ldg(S.ptr + seg + 1);
            for (int k = a + sl; k < b; k += G) term(k, acc);
        }
#pragma unroll
        for (int i = 0; i < NV; ++i) acc[i] = group_reduce<G>(acc[i]);
        if (seg >= 0 && sl == 0) epi(seg, acc);
    }
    if (B.n_multi) {
        gc.sync();
        for (int r = gwarp; r < B.n_multi; r += nwarps) {
            const int4 mr = __ldg(B.multi + r);
            double acc[NV];
#pragma unroll
            for (int i = 0; i < NV; ++i) {
                double a = 0.0;
                for (int k = lane; k < mr.z; k += 32) a += __ldcg(B.partial + (size_t)(mr.y + k) * NV + i);
                acc[i] = group_reduce<32>(a);
            }
            if (lane == 0) epi(mr.x, acc);
        }
    }
}

template <int NV, class Term, class Epi>
__device__ __forceinline__ void seg_reduce(const Sparse &S, Term &term, Epi &epi, GridCtl &gc) {
    switch (S.bins.G) {
        case 4: seg_reduce_G<NV, 4>(S, term, epi, gc); break;
        case 8: seg_reduce_G<NV, 8>(S, term, epi, gc); break;
        case 16: seg_reduce_G<NV, 16>(S, term, epi, gc); break;
        default: seg_reduce_G<NV, 32>(S, term, epi, gc); break;
    }
}

// Visit every non-zero once with its segment id: f(seg, k).  Same partition as seg_reduce.
template <class F>
__device__ __forceinline__ void seg_foreach(const Sparse &S, F &f) {
    const Bins &B = S.bins;
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * kBlock + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * kBlock) >> 5;
    for (int c = gwarp; c < B.n_chunk; c += nwarps) {
        const int4 ch = __ldg(B.chunks + c);
        for (int k = ch.y + lane; k < ch.y + ch.z; k += 32) f(ch.x, k);
    }
    const int G = B.G, SPW = 32 / G;
    const int sub = lane / G, sl = lane % G;
    for (int base = gwarp * SPW; base < B.n_short; base += nwarps * SPW) {
        const int si = base + sub;
        if (si < B.n_short) {
            const int seg = B.short_ids ? __ldg(B.short_ids + si) : si;
            const int a = __ldg(S.ptr + seg), b = __ldg(S.ptr + seg + 1);
            for (int k = a + sl; k < b; k += G) f(seg, k);
        }
    }
}

}  // namespace csd
