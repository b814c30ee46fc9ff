// cs_device.cuh -- device-side building blocks of libcs.so (sm_100a, fp64).
//
// Everything here runs inside persistent COOPERATIVE kernels: one launch covers many phases that
// are separated by grid-wide barriers, so that the scalars of the inner CG (alpha, beta, residual
// norms) and its exit test never leave the device.  Citations P:<line> = /root/reference/PAPER.md.
#pragma once
#include <cstdint>
#include <type_traits>

namespace csd {

// One CTA of 768 threads per SM: 80 registers per thread.  At 64 (2 x 512 threads) ptxas serialises the row pass's batch
// -- index load, gather, FMA one after the other -- to fit its live values; at 80 it keeps the 8 index loads and the
// gathers of a batch in flight together (config 4: row pass 138 -> 125 us; profiles/r02_ncu_notes.md).
#ifndef CS_MINB
#define CS_MINB 1
#endif
#ifndef CS_BLOCK
#define CS_BLOCK 768
#endif
constexpr int kBlock = CS_BLOCK;          // threads per CTA (24 warps)
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
constexpr int kConeLanes = 8;        // lanes cooperating on one SMALL Lorentz cone (<= kConeSmall entries); see cone_sweep
constexpr int kConeSmall = 64;       // up to here: sub-warp groups of kConeLanes lanes, 4 cones per warp
constexpr int kConeMedium = 4096;    // up to here: one warp per cone; beyond: one CTA per cone
constexpr int kDenseMax = 256;       // largest m of the dense factor-apply path (cs_params.dense_m_threshold)
#ifndef CS_ROUNDK
#define CS_ROUNDK 8
#endif
constexpr int kRoundK = CS_ROUNDK;   // slice rows per batch (8 values + 8 indices + 8 gathers in flight per lane)
// (A TMA-staged matrix stream -- per-warp shared-memory rings filled by cp.async.bulk + mbarrier -- was built and
//  measured in round 1: parity-identical, 307 vs 295 us per CG step at config 4, because the rings take L1 capacity
//  away from the gathers; profiles/r01_ncu_notes.md.  It is not in the tree any more.)

// Heavy-row fusion: the column pass K1 of a CG step holds a_ij and the fresh u_j of every entry in
// registers, so it can accumulate sum_j a_ij u_j for the few heaviest rows itself; those entries then leave the row
// pass K2, which would otherwise stream them a second time and gather u through L2.  The accumulators live in shared
// memory and are private, so that the sums have a fixed order (no atomics):
//   class A: the kFuseA longest rows -- one accumulator per THREAD and row (any number of lanes may hit the same
//            row in one instruction);
//   class B: the next kFuseB rows    -- one accumulator per WARP and row; cs_create marks an entry as fused only if
//            no lower lane of the same slice (32 columns) holds the same row, the others stay with K2.
// Which entries are fused is one byte per column of the column-major copy (Sparse::fmask), fetched with the slice's
// epilogue operands before the batch.
// Sizes: kFuseA * 6 KB + kFuseB * 192 B (one CTA of 768 threads per SM) must stay below ~96 KB, or the shared-memory
// carve-out moves from 100 KB to 132 KB per SM and the gathers lose the L1 capacity they need.
#ifndef CS_FUSE_A
#define CS_FUSE_A 4
#endif
#ifndef CS_FUSE_B
#define CS_FUSE_B 320
#endif
#ifndef CS_FUSE_MINLEN
#define CS_FUSE_MINLEN 4096
#endif
constexpr int kFuseA = CS_FUSE_A, kFuseB = CS_FUSE_B;
constexpr int kFuseMinLen = CS_FUSE_MINLEN;     // rows shorter than this are never fused
constexpr int kFuseSmem = (kFuseA * kBlock + kWarps * kFuseB) * 8;   // dynamic shared memory of k_iterate when rows are fused
#ifndef CS_FUSE_K
#define CS_FUSE_K 8
#endif
constexpr int kFuseK = CS_FUSE_K;          // only the first kFuseK entries of a column can be fused (the heavy rows come first)
static_assert(kFuseK % 4 == 0 && kFuseK <= CS_ROUNDK, "scatter works on groups of 4 of a batch's entries");
static_assert(kRoundK % 4 == 0 && kFuseA <= kMaxRed, "scatter works in groups of 4; fuse_flush borrows the reduction scratch");

// One sparse format (rows of the row-major copy or columns of the column-major copy): a list of SLICES.
// A slice is 32 lanes x width entries stored [k][lane] (entry k of lane l at off + 32k + l), so that a
// warp reads it fully coalesced; the lanes of a slice are split over its segments T lanes at a time:
//   T = 1      32 short segments, one thread each (the bulk of every workload)
//   T = 2,4,8  fewer segments per slice, several lanes each: only when the problem is too small to
//              fill the machine with one thread per segment
//   T = 32     one CHUNK (<= kChunk entries) of a long segment; these slices come first, and chunk c
//              either completes its segment (chunk_slot[c] < 0) or writes a partial sum to a slot.
// Slice descriptor: {offset, first segment id, segments | log2(T) << 8 | (has fused entries) << 16, width}.
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
    // K2 view of the row-major copy (heavy-row fusion): the chunk slices [0, n_chunk_k2) hold the entries the row pass
    // of a CG step still has to do; [n_chunk_k2, n_chunk) hold the fused entries (done by the column pass).  Fused
    // rows are always finished through multi_k2 = {segment id, first slot, number of slots, fused index + 1 or 0},
    // which adds the column pass's partial sums fpart[fused index][CTA] in CTA order.
    int n_chunk_k2, n_multi_k2;
    const int4 *multi_k2;
    const double *fpart;
    // column-major copy only: bit k of fmask[(s - n_chunk) * 32 + lane] = entry k of that lane's column in short slice s is fused
    const unsigned char *fmask;
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
    int dense_refine2;      // passes whose dense apply needed the second refinement step (grid dense path)
    unsigned long long phase_ns[8];  // time spent per phase id (kPh*), measured by CTA 0 between grid barriers
};

enum { kPhCone = 0, kPhRhs = 1, kPhK1 = 2, kPhK2 = 3, kPhUpdate = 4, kPhReduce = 5, kPhPrecond = 6, kPhResid = 7 };

struct Ctx {
    int m, n, n_lin, n_soc;
    const int *cone_off;    // [n_soc+1] absolute offsets of the Lorentz blocks (cone_off[0] = n_lin)
    const int *cone_cls;    // [n_soc] cone ids by size class: small, then medium, then large (cone_sweep, cs_kernels.cuh)
    int n_cone_small, n_cone_medium, n_cone_large;
    const int *perm_r, *perm_c;  // internal index -> caller's index (rows / columns sorted by length)
    Sparse R, C;            // row-major (segments = rows) and column-major (segments = columns) copies of A
    int n_fa, n_fb;         // heavy-row fusion: internal rows [0, n_fa) are class A, [n_fa, n_fa + n_fb) class B (0, 0: off)
    double *fpart;          // [n_fa + n_fb][gridDim]: the column pass's partial sums of the fused rows, per CTA
    Csr Rc, Cc;             // plain compressed views of the same two copies
    // FSAI(1) preconditioner G = diag(gd) + strictly-lower part with one entry gm[i] at column partner[i]
    int fsai;               // 0: off (plain Jacobi-equilibrated CG), 1: FSAI(1) below, 2: FSAI(P) (cs_fsaip.cuh)
    int *fp_ctop, *fp_idx, *fp_tptr, *fp_tcnt, *fp_trow;   // FSAI(P): [n][kFsTop], [kFsP][m], [m+1], [m], [kFsP*m]
    double *fp_val, *fp_tval;                               // FSAI(P): [kFsP+1][m], [kFsP*m]
    int n_long;             // internal rows [0, n_long) are longer than kShortMax: no FSAI partner, G = I there
    int *f_ctop;            // [n][3] strongest short rows of every column
    int *f_partner;         // [m] partner row (< i) or -1
    int *f_tptr, *f_tcur, *f_tidx, *f_blk;   // transposed lists: rows whose partner is k are f_tidx[f_tptr[k] .. f_tptr[k+1])
    double *f_gd, *f_gm;    // [m] during the build: g_ii and g_{i,partner}; afterwards the diagonal dd and the partner entry ee of G'G
    double *f_tc;           // [m] coefficients of the transposed-list entries of G'G
    double *z, *t1;         // [m] preconditioned residual; build scratch
    // dense factor-apply path (one-CTA problems with m <= dense_m_threshold, cs.h)
    int dense;              // 0: off, 1: one-CTA factor-apply below, 2: grid path (cs_dense.cuh): gM = A~A~', gMinv = its inverse
    double *gAd, *gM, *gL, *gZ, *gMinv;   // grid dense path: [m][n], then four [m][m] row-major matrices
    double *gDinv;          // inverses of L's 64 x 64 diagonal blocks (cs_dense.cuh)
    double *gpart;          // partial column sums of the dense update pass [row range][n] (cs_kernels.cuh dense_cols)
    int *g_ok;              // grid dense path: 0 if a Cholesky pivot failed (written by k_chol_diag)
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
    double *partial_probe;  // scratch of cs_diag_barrier_probe
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

constexpr int kMaxGrid = 32 * 6;     // CTAs of a cooperative launch (148 SMs x 1 on B200)

// Grid-wide barrier + deterministic all-reduce.
//   barrier : one 32-bit word; every CTA adds 1 except CTA 0, which adds 2^31 - (grid-1), so the top
//             bit flips exactly when the last CTA has arrived; each CTA's thread 0 spins on that bit.
//             One atomic round trip plus the spin; the L2 atomic unit does the counting.
//   reduce  : every CTA stores its NR partial sums before arriving; after the barrier NR warps of every
//             CTA read all gridDim partials (<= 6 per lane, all loads in flight), add them in a fixed order
//             and butterfly: every CTA gets the same bits without a second barrier.
// Partials are double buffered (a fast CTA may already write the next reduction's partials while a slow
// one still reads this one's; it cannot get two barriers ahead).
// Measured on B200 (cs_diag_barrier_probe): see profiles/r01_ncu_notes.md; a flag/mailbox barrier with a
// collector CTA was 6.4 us per barrier and is not used.
struct GridCtl {            // per-thread view of the grid barrier state (uniform over the grid)
    unsigned int *bar;
    int parity;
    double *partials;               // [2][kMaxRed][gridDim]
    double *smem;                   // [kMaxRed * kWarps]
    // phase clock of CTA 0 / thread 0: [0..7] ns per phase, [8] time of the previous lap (shared memory: no registers)
    __device__ static unsigned long long *clock() { __shared__ unsigned long long ns[9]; return ns; }
    __device__ GridCtl(double *partials_, double *smem_, unsigned int *bar_) : bar(bar_), parity(0), partials(partials_), smem(smem_) {
        if (threadIdx.x == 0) for (int i = 0; i < 8; ++i) clock()[i] = 0;
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
// Slice s of the walked range goes to CTA s mod grid (then round-robin over its warps): every CTA -- hence every
// SM -- gets the same number of slices (+-1) of every width class, also in the last, partial round.  Per slice,
// rows are consumed 8 at a time: 8 value + 8 index loads (ld.global.cs: streamed, evict-first, so that the
// gathered vectors stay in L2), then 8 gathers, then the FMAs -- all loads of a batch are in flight before the
// first use.  The epilogue operands and the next slice descriptor are fetched before the batch loop.
// (cp.async- and TMA-staged variants of this loop were measured SLOWER on B200, profiles/r01_ncu_notes.md; so was a
//  software prefetch of the warp's next slice into L2, profiles/r02_ncu_notes.md: the passes are bound by the SM's
//  L1TEX request path, not by DRAM latency.)
// Long segments (chunks) leave partial sums; they are finished after a grid barrier in fixed order.
//
// VIEW = 1 walks the K2 view of the copy (Sparse::n_chunk_k2, multi_k2): the entries the heavy-row fusion left.
// FUSE : the traversal is the column pass of a CG step and accumulates a_ij * (value returned by the epilogue of
//        column j) for every fused entry (Sparse::fmask) into the private shared-memory accumulators.
// ---------------------------------------------------------------------------------------------
struct NoFuse {
    static constexpr bool on = false;
    template <int N> __device__ __forceinline__ void flags(unsigned, bool (&)[N]) const {}
    template <int N> __device__ __forceinline__ void scatter(const double (&)[N], const int (&)[N], const bool (&)[N], double) const {}
};
// Shared-memory accumulators of the heavy-row fusion (see kFuseA / kFuseB above), in the dynamic shared memory of
// k_iterate:  A [kFuseA][kBlock]      class A, per thread
//             B [kWarps][kFuseB]      class B, per warp
constexpr int kFuseOffB = kFuseA * kBlock;
struct FuseAcc {
    static constexpr bool on = true;
    int n_fa;               // rows [0, n_fa) are class A, [n_fa, n_fa + n_fb) class B
    __device__ static double *smem() { extern __shared__ __align__(16) double fuse_smem[]; return fuse_smem; }
    // which of the first kFuseK entries of this lane's column are fused: bits of the byte fetched before the batch
    template <int N>
    __device__ __forceinline__ void flags(unsigned fb, bool (&f)[N]) const {
        static_assert(N == 8, "one byte per column");
#pragma unroll
        for (int q = 0; q < N; ++q) f[q] = q < kFuseK && ((fb >> q) & 1u);
    }
    // acc[row j[q]] += a[q] * uj for the fused entries (f[q]) among N entries of one column.  The read-modify-writes
    // are predicated, not branched around, and issued four at a time (loads, adds, stores), so that they overlap: the
    // rows of a column are distinct, and cs_create fuses a class-B row in at most one lane per slice, so no two of a
    // warp's read-modify-writes between two __syncwarp()s touch the same accumulator.
    template <int N>
    __device__ __forceinline__ void scatter(const double (&a)[N], const int (&j)[N], const bool (&f)[N], double uj) const {
        double *sm = smem();
        const int my_a = threadIdx.x, my_b = kFuseOffB + (threadIdx.x >> 5) * kFuseB - n_fa;
#pragma unroll
        for (int h = 0; h < kFuseK; h += 4) {
            int q[4];
            double v[4];
#pragma unroll
            for (int t = 0; t < 4; ++t) q[t] = j[h + t] < n_fa ? my_a + j[h + t] * kBlock : my_b + j[h + t];
#pragma unroll
            for (int t = 0; t < 4; ++t) v[t] = f[h + t] ? sm[q[t]] : 0.0;
#pragma unroll
            for (int t = 0; t < 4; ++t) if (f[h + t]) sm[q[t]] = v[t] + a[h + t] * uj;
        }
    }
};

// the epilogue of a fused column pass returns the value its column's fused entries are multiplied with
template <bool FUSED, class Epi, class Acc, class Pre>
__device__ __forceinline__ double call_epi(Epi &epi, int seg, const Acc &acc, const Pre &pre) {
    if constexpr (FUSED) return epi(seg, acc, pre);
    else { epi(seg, acc, pre); return 0.0; }
}

template <int NV, bool PRISTINE, int VIEW = 0, class Term, class Epi, class Fuse = NoFuse>
__device__ __forceinline__ void seg_reduce(const Sparse &S, Term &term, Epi &epi, GridCtl &gc, Fuse fuse = Fuse{}) {
    const int lane = threadIdx.x & 31;
    const int gwarp = blockIdx.x + gridDim.x * (threadIdx.x >> 5);
    const int nwarps = (gridDim.x * kBlock) >> 5;
    const double *gval = PRISTINE ? S.val0 : S.val;
    constexpr int UN = NV == 1 ? kRoundK : kRoundK / 2;   // two-operand gathers: half the batch, same registers
    const int chunk_end = VIEW ? S.n_chunk_k2 : S.n_chunk;
    // The walk is instantiated twice: chunk slices (T = 32, one segment, partial-sum slot) and short-segment slices.
    auto walk = [&](auto chunk_tag, int s, const int s_end) {
    constexpr bool CH = decltype(chunk_tag)::value;
    int4 sl = s < s_end ? __ldg(S.slices + s) : make_int4(0, 0, 0, 0);
    while (s < s_end) {
        const int sn = s + nwarps;
        const int4 nxt = sn < s_end ? __ldg(S.slices + sn) : make_int4(0, 0, 0, 0);
        const int lgT = CH ? 5 : (sl.z >> 8) & 7, T = 1 << lgT;     // lanes per segment in this slice
        const int seg = sl.y + (lane >> lgT);
        const bool head = (lane >> lgT) < (sl.z & 255) && (lane & (T - 1)) == 0;
        const int cslot = CH ? __ldg(S.chunk_slot + s) : -1;  // fetched early, like `pre` (warp-uniform address)
        typename Epi::Pre pre = epi.pre(head ? seg : sl.y);
        unsigned fb = 0;                                      // fused-entry bits of this lane's column (early, like `pre`)
        if constexpr (Fuse::on && !CH) { if (sl.z >> 16) fb = __ldg(S.fmask + (size_t)(s - S.n_chunk) * 32 + lane); }
        double acc[NV];
#pragma unroll
        for (int i = 0; i < NV; ++i) acc[i] = 0.0;
        const double *vp = gval + sl.x + lane;
        const int *ip = S.idx + sl.x + lane;
        // one batch: UN slice rows from row k on -- all value and index loads, then the gathers, then the FMAs
        auto batch = [&](int k, double (&a)[UN], int (&j)[UN]) {
#pragma unroll
            for (int q = 0; q < UN; ++q) {                   // predicated (warp-uniform): no traffic for rows past the end
                const bool ok = k + q < sl.w;
                a[q] = ok ? __ldcs(vp + 32 * (k + q)) : 0.0;
                j[q] = ok ? __ldcs(ip + 32 * (k + q)) : -1;
            }
            typename Term::G g[UN];
#pragma unroll
            for (int q = 0; q < UN; ++q) g[q] = term.fetch(j[q] >= 0 ? j[q] : 0);   // index 0: one broadcast wavefront
#pragma unroll
            for (int q = 0; q < UN; ++q) if (j[q] >= 0) term.fma(a[q], g[q], acc);
        };
        if constexpr (Fuse::on && !CH) {
            // Column pass of a CG step with heavy-row fusion.  Columns of at most UN entries (the bulk) are one batch
            // whose values and indices are still in registers when the epilogue has produced u_j.
            if (sl.w <= UN) {
                double a[UN]; int j[UN];
                batch(0, a, j);
                for (int o = T >> 1; o > 0; o >>= 1) acc[0] += __shfl_xor_sync(0xffffffffu, acc[0], o);
                double uj = 0.0;
                if (head) uj = call_epi<Fuse::on>(epi, seg, acc, pre);   // T = 1 whenever the slice has fused entries (cs_create)
                if (sl.z >> 16) {                            // warp-uniform: some entry of this slice is fused
                    bool f[UN];
                    fuse.flags(fb, f);
                    fuse.scatter(a, j, f, uj);
                    __syncwarp();                            // the warp's next slice may hit the same class-B accumulators from other lanes
                }
                s = sn;
                sl = nxt;
                continue;
            }
        }
        for (int k = 0; k < sl.w; k += UN) {
            double a[UN]; int j[UN];
            batch(k, a, j);
        }
        if (CH) {
#pragma unroll
            for (int i = 0; i < NV; ++i) acc[i] = group_reduce<32>(acc[i]);
        } else {
            for (int o = T >> 1; o > 0; o >>= 1) {
#pragma unroll
                for (int i = 0; i < NV; ++i) acc[i] += __shfl_xor_sync(0xffffffffu, acc[i], o);
            }
        }
        if constexpr (Fuse::on && !CH) {
            double uj = 0.0;
            if (head) uj = call_epi<Fuse::on>(epi, seg, acc, pre);
            if (sl.z >> 16) {                                // longer columns: their first entries come back from L1 / L2
                double a[UN]; int j[UN]; bool f[UN];
                fuse.flags(fb, f);
#pragma unroll
                for (int q = 0; q < UN; ++q) j[q] = f[q] ? __ldg(ip + 32 * q) : 0;
#pragma unroll
                for (int q = 0; q < UN; ++q) a[q] = f[q] ? __ldg(vp + 32 * q) : 0.0;
                fuse.scatter(a, j, f, uj);
                __syncwarp();
            }
        } else if (head) {
            if (cslot < 0) epi(seg, acc, pre);
            else {
#pragma unroll
                for (int i = 0; i < NV; ++i) S.partial[(size_t)cslot * 2 + i] = acc[i];
            }
        }
        s = sn;
        sl = nxt;
    }
    return s;
    };
    // the short-segment slices continue the deal where the chunk slices of this view left off: the chunk walk ends on
    // the warp's first slice number >= chunk_end, which is congruent to gwarp - chunk_end modulo nwarps past it
    const int s_short = walk(std::true_type{}, gwarp, chunk_end) - chunk_end + S.n_chunk;
    walk(std::false_type{}, s_short, S.n_slice);
    const int n_multi = VIEW ? S.n_multi_k2 : S.n_multi;
    if (n_multi) {
        const int4 *multi = VIEW ? S.multi_k2 : S.multi;
        gc.sync();
        for (int r = gwarp; r < n_multi; r += nwarps) {
            const int4 mr = __ldg(multi + r);
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
                if (VIEW && i == 0 && mr.w) {            // the column pass's share of a fused row, in CTA order
                    const double *fp = S.fpart + (size_t)(mr.w - 1) * gridDim.x;
                    double t[kMaxGrid / 32];
#pragma unroll
                    for (int q = 0; q < kMaxGrid / 32; ++q) t[q] = lane + 32 * q < (int)gridDim.x ? __ldcg(fp + lane + 32 * q) : 0.0;
#pragma unroll
                    for (int q = 0; q < kMaxGrid / 32; ++q) a += t[q];
                }
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
        const int lgT = (sl.z >> 8) & 7;
        if ((lane >> lgT) < (sl.z & 255)) {
            const int base = sl.x + lane, seg = sl.y + (lane >> lgT);
            for (int k = 0; k < sl.w; ++k) S.val[base + 32 * k] = f(seg, S.val0[base + 32 * k], __ldg(S.idx + base + 32 * k));
        }
    }
}

}  // namespace csd
