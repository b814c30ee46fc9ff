// cs_device.cuh -- device-side building blocks of libcs.so (sm_100a, fp64).
//
// Everything here runs inside persistent COOPERATIVE kernels: one launch covers many phases that
// are separated by grid-wide barriers, so that the scalars of the inner CG (alpha, beta, residual
// norms) and its exit test never leave the device.  Citations P:<line> = /root/reference/PAPER.md.
#pragma once
#include <cstdint>
#include <type_traits>

namespace csd {

#ifndef CS_MINB
#define CS_MINB 2
#endif
#ifndef CS_BLOCK
#define CS_BLOCK 512
#endif
constexpr int kBlock = CS_BLOCK;          // threads per CTA (16 warps)
constexpr int kWarps = kBlock / 32;
constexpr int kMaxRed = 8;           // scalars per grid reduction
#ifndef CS_SHORTMAX
#define CS_SHORTMAX 64
#endif
#ifndef CS_CHUNK
#define CS_CHUNK 1024
#endif
constexpr int kShortMax = CS_SHORTMAX;        // segments up to this many non-zeros are "short" (1-8 lanes each inside a slice)
constexpr int kChunk = CS_CHUNK;         // long segments are cut into warp-sized chunks of this many non-zeros
constexpr int kConeLanes = 8;        // lanes cooperating on one Lorentz cone
constexpr int kDenseMax = 256;       // largest m of the dense factor-apply path (cs_params.dense_m_threshold)
// Build-time alternative, measured and NOT the default (profiles/r01_ncu_notes.md, "TMA-staged stream"): with
// CS_TMA=1 the matrix stream of every traversal is staged through per-warp shared-memory rings by bulk async
// copies (cp.async.bulk + mbarrier) instead of ld.global.cs.  Parity-identical; config 4 307 vs 295 us per CG
// step: the rings take L1 capacity away from the gathers, and below ~90 KB of L1 per SM the gathers collapse
// (which is why that build uses batches of 4 rows and 2 stages: 48 KB per CTA).
#ifndef CS_TMA
#define CS_TMA 0
#endif
#ifndef CS_ROUNDK
#define CS_ROUNDK (CS_TMA ? 4 : 8)
#endif
#ifndef CS_STAGES
#define CS_STAGES 2
#endif
constexpr int kRoundK = CS_ROUNDK;   // slice rows per batch (8 values + 8 indices + 8 gathers in flight per lane)
constexpr int kStages = CS_STAGES;   // per-warp ring of staged batches
constexpr int kStageVal = kRoundK * 32 * 8, kStageIdx = kRoundK * 32 * 4, kStageBytes = kStageVal + kStageIdx;
// dynamic shared memory of every cooperative kernel: [warp][stage]{values, indices} then [warp][stage] mbarriers
constexpr int kDynSmem = CS_TMA ? kWarps * kStages * (kStageBytes + 8) : 0;

// One sparse format (rows of the row-major copy or columns of the column-major copy): a list of SLICES.
// A slice is 32 lanes x width entries stored [k][lane] (entry k of lane l at off + 32k + l), so that a
// warp reads it fully coalesced; the lanes of a slice are split over its segments T lanes at a time:
//   T = 1      32 short segments, one thread each (the bulk of every workload)
//   T = 2,4,8  fewer segments per slice, several lanes each: only when the problem is too small to
//              fill the machine with one thread per segment
//   T = 32     one CHUNK (<= kChunk entries) of a long segment; these slices come first, and chunk c
//              either completes its segment (chunk_slot[c] < 0) or writes a partial sum to a slot.
// Padding entries have val = 0 and a valid index.  Rows (and orthant columns) are physically sorted by
// length at cs_create, so padding is negligible.
struct Sparse {
    int n_slice;
    const int4 *slices;     // {off, first segment id, segments in the slice | log2(T) << 8, width}
    int n_chunk;            // slices [0, n_chunk) are chunks of long segments
    const int *chunk_slot;  // [n_chunk]
    const int *idx;
    double *val;            // scaled values (D A O)
    const double *val0;     // pristine values (A)
    int n_multi;
    const int4 *multi;      // long segments spanning several chunks: {segment id, first slot, number of slots, 0}
    double *partial;        // [slots][2]
};

// Plain compressed view of one copy (segment s = entries [ptr[s], ptr[s+1]), minor index idx[e], value
// val[pos[e]] in the slice storage).  Only the set-up of the FSAI preconditioner walks it.
struct Csr {
    const int *ptr, *idx, *pos;
};

struct Scalars {            // device-resident state scalars (read back only by cs_residuals)
    double resid[16];
    long long iter, cg_steps_total, cg_steps_cond;
    int cg_steps_last, n_cond, cg_hit_max, dense_ok;   // dense_ok: the Cholesky factor of the current scaling is usable
    double fp_res2;         // ||s_new - s||^2 of the last pass
    unsigned long long phase_ns[8];  // time spent per phase id (kPh*), measured by CTA 0 between grid barriers
};

enum { kPhCone = 0, kPhRhs = 1, kPhK1 = 2, kPhK2 = 3, kPhUpdate = 4, kPhReduce = 5, kPhPrecond = 6, kPhResid = 7 };

struct Ctx {
    int m, n, n_lin, n_soc;
    const int *cone_off;    // [n_soc+1] absolute offsets of the Lorentz blocks (cone_off[0] = n_lin)
    const int *perm_r, *perm_c;  // internal index -> caller's index (rows / columns sorted by length)
    Sparse R, C;            // row-major (segments = rows) and column-major (segments = columns) copies of A
    Csr Rc, Cc;             // plain compressed views of the same two copies
    // FSAI(1) preconditioner G = diag(gd) + strictly-lower part with one entry gm[i] at column partner[i]
    int fsai;               // 0: off (plain Jacobi-equilibrated CG)
    int *f_ctop;            // [n][3] strongest short rows of every column
    int *f_partner;         // [m] partner row (< i) or -1
    int *f_tptr, *f_tcur, *f_tidx, *f_blk;   // transposed lists: rows whose partner is k are f_tidx[f_tptr[k] .. f_tptr[k+1])
    double *f_gd, *f_gm;    // [m] during the build: g_ii and g_{i,partner}; afterwards the diagonal dd and the partner entry ee of G'G
    double *f_tc;           // [m] coefficients of the transposed-list entries of G'G
    double *z, *t1;         // [m] preconditioned residual; build scratch
    // dense factor-apply path (one-CTA problems with m <= dense_m_threshold, cs.h)
    int dense;              // 0: off
    double *dM;             // [m][m] row-major: lower triangle incl. diagonal = Cholesky factor L, strict upper = A~A~'
    double *dMd;            // [m] diagonal of A~A~'
    double *dv;             // [2m] scratch of the triangular solves
    // n-vectors
    double *s, *p, *g, *e, *u, *chat, *O, *xb, *zb;
    const double *c;
    // m-vectors
    double *w, *r, *v, *D, *btil;
    const double *b;
    double *partials;       // [2][kMaxRed][gridDim]
    unsigned int *bar;      // grid-barrier word
    Scalars *sc;
    double *partial_probe;  // scratch of cs_barrier_probe
    double mu, t, o_floor, cg_tol, cg_reduce;
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

// ---------------------------------------------------------------------------------------------
// Bulk asynchronous copies (TMA, cp.async.bulk) global -> shared with mbarrier completion, used by the
// CS_TMA=1 build only: the matrix stream (values + minor indices of a batch of slice rows) then never enters
// the LSU/L1TEX pipeline that bounds the gathers, needs no registers while in flight, and one
// lane issues a whole batch.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ unsigned long long policy_evict_first() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void tma_load(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar, unsigned long long pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
// generic-proxy writes to global memory that a later bulk copy will read (the rescaled matrix values)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

constexpr int kMaxGrid = 32 * 12;    // CTAs of a cooperative launch (148 SMs x 2 = 296 on B200)

// Grid-wide barrier + deterministic all-reduce.
//   barrier : one 32-bit word; every CTA adds 1 except CTA 0, which adds 2^31 - (grid-1), so the top
//             bit flips exactly when the last CTA has arrived; each CTA's thread 0 spins on that bit.
//             One atomic round trip plus the spin; the L2 atomic unit does the counting.
//   reduce  : every CTA stores its NR partial sums before arriving; after the barrier NR warps of every
//             CTA read all gridDim partials (<= 12 per lane, all loads in flight), add them in a fixed order
//             and butterfly: every CTA gets the same bits without a second barrier.
// Partials are double buffered (a fast CTA may already write the next reduction's partials while a slow
// one still reads this one's; it cannot get two barriers ahead).
// Measured on B200 (cs_barrier_probe): see profiles/r01_ncu_notes.md; a flag/mailbox barrier with a
// collector CTA was 6.4 us per barrier and is not used.
struct GridCtl {            // per-thread view of the grid barrier state (uniform over the grid)
    unsigned int *bar;
    int parity;
    double *partials;               // [2][kMaxRed][gridDim]
    double *smem;                   // [kMaxRed * kWarps]
    uint32_t ring, mbar, units;     // this warp's staging ring and mbarriers (shared-window addresses); batches consumed so far
    // phase clock of CTA 0 / thread 0: [0..7] ns per phase, [8] time of the previous lap (shared memory: no registers)
    __device__ static unsigned long long *clock() { __shared__ unsigned long long ns[9]; return ns; }
    __device__ GridCtl(double *partials_, double *smem_, unsigned int *bar_) : bar(bar_), parity(0), partials(partials_), smem(smem_) {
        if (threadIdx.x == 0) for (int i = 0; i < 8; ++i) clock()[i] = 0;
#if CS_TMA
        extern __shared__ __align__(128) unsigned char dyn_smem[];
        const int warp = threadIdx.x >> 5;
        ring = smem_u32(dyn_smem) + warp * kStages * kStageBytes;
        mbar = smem_u32(dyn_smem) + kWarps * kStages * kStageBytes + warp * kStages * 8;
        units = 0;
        if ((threadIdx.x & 31) == 0) {
            for (int i = 0; i < kStages; ++i) mbar_init(mbar + 8 * i, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            fence_proxy_async();
        }
        __syncthreads();
#endif
        if (threadIdx.x == 0) clock()[8] = now();
    }
    __device__ void sync() {
        __syncthreads();
        if (gridDim.x == 1) return;                            // tiny problems run on one CTA: no global traffic
        if (threadIdx.x == 0) {
            const unsigned int inc = blockIdx.x == 0 ? 0x80000000u - (gridDim.x - 1) : 1u;
            __threadfence();                                   // release the CTA's writes
            const unsigned int old = atomicAdd(bar, inc);
            unsigned int cur;
            do {
                asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(cur) : "l"(bar) : "memory");
            } while (((old ^ cur) & 0x80000000u) == 0);
            __threadfence();                                   // acquire everybody else's
        }
        __syncthreads();
    }
    __device__ static unsigned long long now() {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        return t;
    }
    // charge the time since the previous lap to phase `id` (only CTA 0 / thread 0 keeps the books)
    __device__ void lap(int id) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            const unsigned long long t = now();
            clock()[id] += t - clock()[8];
            clock()[8] = t;
        }
    }
    __device__ void flush(Scalars *sc) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
#pragma unroll
            for (int i = 0; i < 8; ++i) sc->phase_ns[i] += clock()[i];
        }
    }
};

// Deterministic grid-wide reduction of NR per-thread values; includes ONE grid barrier.
// Every thread of every CTA returns the same bits.
template <int NR, class Op = OpSum>
__device__ void grid_reduce(double (&v)[NR], GridCtl &gc, double ident = 0.0) {
    static_assert(NR <= kMaxRed && NR <= kWarps, "too many scalars");
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
        __stcg(buf + (size_t)threadIdx.x * gridDim.x + blockIdx.x, acc);
    }
    gc.sync();
    if (warp < NR) {
        double t[kMaxGrid / 32];
#pragma unroll
        for (int q = 0; q < kMaxGrid / 32; ++q) {
            const int b = lane + 32 * q;
            t[q] = b < (int)gridDim.x ? __ldcg(buf + (size_t)warp * gridDim.x + b) : ident;
        }
        double acc = t[0];
#pragma unroll
        for (int q = 1; q < kMaxGrid / 32; ++q) acc = Op::f(acc, t[q]);
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
// Segment traversal.  `g = term.fetch(j)` gathers the operand(s) of minor index j and
// `term.fma(a, g, acc)` adds the contribution of one entry of value a to acc[NV];
// `epi(seg, sums, pre)` is called once per segment with the complete sums, where
// `pre = epi.pre(seg)` holds whatever the epilogue reads from memory (fetched early).
//
// Every warp walks its slices (s = gwarp, gwarp + nwarps, ...).  Per slice, rows are consumed 8 at a
// time: 8 value + 8 index loads (ld.global.cs: streamed, evict-first, so that the gathered vectors stay
// in L2), then 8 gathers, then the FMAs -- all loads of a batch are in flight before the first use.
// The epilogue operands and the next slice descriptor are fetched before the batch loop.
// (A cp.async-staged variant of this loop was measured SLOWER on B200 -- the LDGSTS instructions add
// to the L1TEX load that already bounds the gathers; see profiles/r01_ncu_notes.md.)
// Long segments (chunks) leave partial sums; they are finished after a grid barrier in fixed order.
// ---------------------------------------------------------------------------------------------
template <int NV, bool PRISTINE, class Term, class Epi>
__device__ __forceinline__ void seg_reduce(const Sparse &S, Term &term, Epi &epi, GridCtl &gc) {
    const int lane = threadIdx.x & 31;
    // slice s goes to CTA s mod grid (then round-robin over its warps): every CTA -- hence every SM -- gets the
    // same number of slices (+-1) of every width class, also in the last, partial round
    const int gwarp = blockIdx.x + gridDim.x * (threadIdx.x >> 5);
    const int nwarps = (gridDim.x * kBlock) >> 5;
    const double *gval = PRISTINE ? S.val0 : S.val;
    constexpr int UN = NV == 1 ? kRoundK : kRoundK / 2;   // two-operand gathers: half the batch, same registers
    int s = gwarp;
    int4 sl = s < S.n_slice ? __ldg(S.slices + s) : make_int4(0, 0, 0, 0);
#if CS_TMA
    // Producer side of this warp's ring: the batches (<= kRoundK rows of one slice) are issued in the order
    // the loop below consumes them, kStages ahead; lane 0 issues, every lane keeps the (uniform) iterator.
    int is = s, ioff = sl.x, irem = sl.w;                    // slice, next entry offset, rows left in it
    while (is < S.n_slice && irem == 0) {
        is += nwarps;
        if (is < S.n_slice) { const int4 d = __ldg(S.slices + is); ioff = d.x; irem = d.w; }
    }
    auto issue = [&](uint32_t slot) {
        if (is >= S.n_slice) return;
        const int rows = min(kRoundK, irem);
        if (lane == 0) {
            const uint32_t dst = gc.ring + slot * kStageBytes, mb = gc.mbar + slot * 8;
            const unsigned long long pol = policy_evict_first();
            mbar_expect_tx(mb, (uint32_t)rows * 32u * 12u);
            tma_load(dst, gval + ioff, (uint32_t)rows * 256u, mb, pol);
            tma_load(dst + kStageVal, S.idx + ioff, (uint32_t)rows * 128u, mb, pol);
        }
        ioff += 32 * kRoundK;
        irem -= kRoundK;
        while (is < S.n_slice && irem <= 0) {
            is += nwarps;
            if (is < S.n_slice) { const int4 d = __ldg(S.slices + is); ioff = d.x; irem = d.w; }
        }
    };
    uint32_t units = gc.units;
#pragma unroll
    for (int i = 0; i < kStages; ++i) issue((units + i) % kStages);
    extern __shared__ __align__(128) unsigned char dyn_smem[];
    const unsigned char *my_ring = dyn_smem + (threadIdx.x >> 5) * kStages * kStageBytes;
#endif
    // The walk is instantiated twice: chunk slices (T = 32, one segment, partial-sum slot) and short-segment slices.
    auto walk = [&](auto chunk_tag, const int s_end) {
    constexpr bool CH = decltype(chunk_tag)::value;
    while (s < s_end) {
        const int sn = s + nwarps;
        const int4 nxt = sn < S.n_slice ? __ldg(S.slices + sn) : make_int4(0, 0, 0, 0);
        const int lgT = CH ? 5 : sl.z >> 8, T = 1 << lgT;     // lanes per segment in this slice
        const int seg = sl.y + (lane >> lgT);
        const bool head = (lane >> lgT) < (sl.z & 255) && (lane & (T - 1)) == 0;
        const int cslot = CH ? __ldg(S.chunk_slot + s) : -1;  // fetched early, like `pre` (warp-uniform address)
        typename Epi::Pre pre = epi.pre(head ? seg : sl.y);
        double acc[NV];
#pragma unroll
        for (int i = 0; i < NV; ++i) acc[i] = 0.0;
#if CS_TMA
        for (int k = 0; k < sl.w; k += kRoundK) {
            const uint32_t slot = units % kStages;
            mbar_wait(gc.mbar + slot * 8, (units / kStages) & 1);
            const double *sv = reinterpret_cast<const double *>(my_ring + slot * kStageBytes) + lane;
            const int *si = reinterpret_cast<const int *>(my_ring + slot * kStageBytes + kStageVal) + lane;
#pragma unroll
            for (int q0 = 0; q0 < kRoundK; q0 += UN) {
                int j[UN];
#pragma unroll
                for (int q = 0; q < UN; ++q) j[q] = k + q0 + q < sl.w ? si[32 * (q0 + q)] : -1;
                typename Term::G g[UN];
#pragma unroll
                for (int q = 0; q < UN; ++q) g[q] = term.fetch(j[q] >= 0 ? j[q] : 0);   // index 0: one broadcast wavefront
#pragma unroll
                for (int q = 0; q < UN; ++q) if (j[q] >= 0) term.fma(sv[32 * (q0 + q)], g[q], acc);
            }
            __syncwarp();                                    // every lane has consumed the stage
            issue(slot);
            ++units;
        }
#else
        const double *vp = gval + sl.x + lane;
        const int *ip = S.idx + sl.x + lane;
        for (int k = 0; k < sl.w; k += UN) {
            double a[UN]; int j[UN];
#pragma unroll
            for (int q = 0; q < UN; ++q) {                   // predicated: no traffic for rows past the end
                const bool ok = k + q < sl.w;
                a[q] = ok ? __ldcs(vp + 32 * (k + q)) : 0.0;
                j[q] = ok ? __ldcs(ip + 32 * (k + q)) : -1;
            }
            typename Term::G g[UN];
#pragma unroll
            for (int q = 0; q < UN; ++q) g[q] = term.fetch(j[q] >= 0 ? j[q] : 0);   // index 0: one broadcast wavefront
#pragma unroll
            for (int q = 0; q < UN; ++q) if (j[q] >= 0) term.fma(a[q], g[q], acc);
        }
#endif
        if (CH) {
#pragma unroll
            for (int i = 0; i < NV; ++i) acc[i] = group_reduce<32>(acc[i]);
        } else {
            for (int o = T >> 1; o > 0; o >>= 1) {
#pragma unroll
                for (int i = 0; i < NV; ++i) acc[i] += __shfl_xor_sync(0xffffffffu, acc[i], o);
            }
        }
        if (head) {
            if (cslot < 0) epi(seg, acc, pre);
            else {
#pragma unroll
                for (int i = 0; i < NV; ++i) S.partial[(size_t)cslot * 2 + i] = acc[i];
            }
        }
        s = sn;
        sl = nxt;
    }
    };
    walk(std::true_type{}, S.n_chunk);
    walk(std::false_type{}, S.n_slice);
#if CS_TMA
    gc.units = units;
#endif
    if (S.n_multi) {
        gc.sync();
        for (int r = gwarp; r < S.n_multi; r += nwarps) {
            const int4 mr = __ldg(S.multi + r);
            double tot[NV];
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
                tot[i] = group_reduce<32>(a);
            }
            if (lane == 0) epi(mr.x, tot, epi.pre(mr.x));
        }
    }
}

// Rewrite every stored entry: val = f(seg, val0, idx).
template <class F>
__device__ __forceinline__ void seg_rescale(const Sparse &S, F &f) {
    const int lane = threadIdx.x & 31;
    const int gwarp = (blockIdx.x * kBlock + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * kBlock) >> 5;
    for (int s = gwarp; s < S.n_slice; s += nwarps) {
        const int4 sl = __ldg(S.slices + s);
        const int lgT = sl.z >> 8;
        if ((lane >> lgT) < (sl.z & 255)) {
            const int base = sl.x + lane, seg = sl.y + (lane >> lgT);
            for (int k = 0; k < sl.w; ++k) S.val[base + 32 * k] = f(seg, S.val0[base + 32 * k], __ldg(S.idx + base + 32 * k));
        }
    }
#if CS_TMA
    fence_proxy_async();   // the next reader of S.val is a bulk async copy (after a grid barrier)
#endif
}

}  // namespace csd
