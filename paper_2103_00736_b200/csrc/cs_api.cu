// cs_api.cu -- host side of libcs.so: the C ABI of include/cs.h (diagnostics: include/cs_diag.h).
// Validation, the internal ordering, the CSR->CSC transposition, the slice layout and the heavy-row fusion plan are one-off
// host work at cs_create; every step of the iteration itself is a kernel in cs_kernels*.cuh, cs_fsaip.cuh, cs_dense.cuh.
// The handle-free, allocation-free entry point cs_cone_violation_static and its static scratch are at the end of the file.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <chrono>
#include <cstdlib>
#include <memory>
#include <mutex>
#include <new>
#include <string>
#include <thread>
#include <utility>
#include <vector>

#include "../../include/cs_diag.h"
#include "cs_kernels_cond.cuh"
#include "cs_build.cuh"

#ifndef CS_AUTO_FSAIP_MB
#define CS_AUTO_FSAIP_MB 100
#endif
#ifndef CS_STATIC_MAX_SOC
#define CS_STATIC_MAX_SOC 32768
#endif
#ifndef CS_FUSE_CARVEOUT
#define CS_FUSE_CARVEOUT 43
#endif

using namespace csd;

struct cs_solver {
    Ctx ctx{};
    cudaStream_t stream = nullptr;
    int device = 0;
    int grid = 0;
    int64_t nnz = 0;
    size_t dyn_smem = 0;       // bytes of dynamic shared memory of k_iterate (accumulators of the heavy-row fusion)
    std::vector<void *> allocs;
    cs_params prm{};
    bool dense_capable = false;   // dense-stored A on many CTAs with m <= kDenseGridMax: the grid dense path may be used (its buffers are allocated on first use)
    bool conditioned = false;  // the l=1 conditioning of step 4 has run
    bool xz_stale = false;     // xb, zb older than (p, s)
    bool started = false;      // some pass or conditioning has run (cs_set_point no longer allowed)
    int build_mode = 0;        // layout build: 0 automatic, 1 host, 2 device (cs_diag_create)
    size_t tot_r = 0, tot_c = 0;   // padded entries of the two sliced copies (cs_diag_layout_digest)
    int64_t launches = 0;
    int64_t iter = 0;          // passes done (Algorithm 2's l), mirrors Scalars::iter
    double stall_f = 0.0;      // cs_solve, stall rule: fixed-point residual sampled after pass stall_at (-1: none)
    int64_t stall_at = -1;
    std::string err;
};

namespace {

thread_local std::string g_create_err;
constexpr int kFuseCarveoutPct = CS_FUSE_CARVEOUT;   // percent of the SM's 228 KB of shared memory asked for when k_iterate fuses rows
constexpr double kAutoFsaiPMinBytes = 16e6;
constexpr double kAutoFsaiPBytes = CS_AUTO_FSAIP_MB * 1e6;   // precond = 0 selects FSAI(5) up to this many bytes of matrix copies (L2-resident), FSAI(1) beyond
constexpr int kDeviceBuildMinNnz = 100000;   // smaller problems are laid out on the host (a few ms either way)
constexpr int kOneCtaNnz = 8192;   // problems up to this many non-zeros run on ONE CTA

#define CS_CUDA(S, call)                                                                         \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            (S)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                       \
            return e_ == cudaErrorMemoryAllocation ? CS_ENOMEM : CS_ECUDA;                       \
        }                                                                                        \
    } while (0)

// A handle is bound to the device that was current at cs_create (cs.h): every entry point that takes a handle makes that
// device current for the duration of the call and restores the caller's on exit.
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const cs_solver *S) {
        if (S && cudaGetDevice(&prev) == cudaSuccess && prev != S->device) cudaSetDevice(S->device);
        else prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

template <class T>
cs_status dev_alloc(cs_solver *S, T **out, size_t count) {
    void *p = nullptr;
    CS_CUDA(S, cudaMalloc(&p, std::max<size_t>(count, 1) * sizeof(T)));
    S->allocs.push_back(p);
    *out = static_cast<T *>(p);
    return CS_OK;
}

template <class T>
cs_status dev_upload(cs_solver *S, T **out, const T *host, size_t count) {
    cs_status st = dev_alloc(S, out, count);
    if (st != CS_OK) return st;
    if (count) CS_CUDA(S, cudaMemcpyAsync(*out, host, count * sizeof(T), cudaMemcpyHostToDevice, S->stream));
    return CS_OK;
}

template <class T>
cs_status dev_zeros(cs_solver *S, T **out, size_t count) {
    cs_status st = dev_alloc(S, out, count);
    if (st != CS_OK) return st;
    CS_CUDA(S, cudaMemsetAsync(*out, 0, std::max<size_t>(count, 1) * sizeof(T), S->stream));
    return CS_OK;
}

// Fetch an input array to the host (inputs may live in device memory).
template <class T>
cs_status fetch(cs_solver *S, std::vector<T> &dst, const T *src, size_t count, cs_mem where) {
    dst.resize(count);
    if (!count) return CS_OK;
    if (where == CS_HOST) std::memcpy(dst.data(), src, count * sizeof(T));
    else CS_CUDA(S, cudaMemcpy(dst.data(), src, count * sizeof(T), cudaMemcpyDeviceToHost));
    return CS_OK;
}

// std::vector without value-initialisation: the big host arrays (hundreds of MB each) are written once, in parallel,
// by the code that fills them -- a serial zero-fill (and its page faults) would cost more than the fill itself.
template <class T>
struct NoInit : std::allocator<T> {
    template <class U> struct rebind { using other = NoInit<U>; };
    template <class U, class... Args>
    void construct(U *p, Args &&...args) {
        if constexpr (sizeof...(Args) == 0) ::new ((void *)p) U;
        else ::new ((void *)p) U(std::forward<Args>(args)...);
    }
};
template <class T> using uvec = std::vector<T, NoInit<T>>;

// Host image of one Sparse (cs_device.cuh): chunk slices of the long segments first, then the slices of
// the short ones, all in one pair of arrays.
struct HostSparse {
    std::vector<int4> slices, multi, multi_k2;
    std::vector<int> chunk_slot;
    uvec<int> idx;
    uvec<int> pos;                // compressed entry -> position in val/idx (for the plain compressed view, Csr in cs_device.cuh)
    uvec<double> val;
    std::vector<unsigned char> fmask;  // column-major copy with fused rows: [short slice][lane] bit k = entry k of the column is fused
    int n_chunk = 0, n_chunk_k2 = 0, n_slots = 0;
    std::vector<int> chunk_src, chunk_len;   // first source entry and length of every chunk slice (the fill needs them)
    size_t total = 0;             // padded entries
    bool too_big = false;         // padded storage would exceed 2^31 entries: nothing was filled
};

// Run f(block) for block = 0..n_blocks-1 on up to `nt` host threads (blocks are handed out dynamically).
// Nothing may throw across a thread boundary: an exception in a worker is recorded and rethrown by the caller's
// thread as std::bad_alloc (cs_create turns that into CS_ENOMEM).
template <class F>
void parallel_blocks(int n_blocks, int nt, F f) {
    nt = std::max(1, std::min(nt, n_blocks));
    if (nt == 1) { for (int b = 0; b < n_blocks; ++b) f(b); return; }
    std::atomic<int> next{0};
    std::atomic<bool> failed{false};
    std::vector<std::thread> th;
    auto body = [&] {
        try { for (int b = next.fetch_add(1); b < n_blocks && !failed.load(); b = next.fetch_add(1)) f(b); }
        catch (...) { failed.store(true); }
    };
    try { for (int t = 0; t < nt; ++t) th.emplace_back(body); }
    catch (...) { failed.store(true); }
    for (auto &t : th) t.join();
    if (failed.load()) throw std::bad_alloc();
}

int host_threads() { return (int)std::max(1u, std::min(16u, std::thread::hardware_concurrency())); }

// Heavy-row fusion plan (cs_device.cuh): internal rows [0, n_fa) are class A, [n_fa, n_fa + n_fb) class B.
struct FusePlan { int n_fa = 0, n_fb = 0; int rows() const { return n_fa + n_fb; } };

// ptr/idx/val: compressed segments in INTERNAL numbering (segment s = entries [ptr[s], ptr[s+1])).
// Two phases: a serial plan (slice descriptors and offsets, O(#segments)), then a parallel fill.
//   Column-major copy (fuse != nullptr, fused_out != nullptr): an entry of a one-thread-per-column slice whose row is a
//     fused row gets its lane's bit in the slice's masks (HostSparse::fmask) and fused_out[compressed position] = 1 --
//     class A always, class B only for the lowest lane of its slice that holds that row (the accumulators of class B
//     are per warp); only the first kFuseK entries of a column qualify.
//   Row-major copy (split != nullptr): the first split[s] entries of fused row s stay with the row pass of a CG step
//     (K2 view), the rest have been taken over by the column pass; each part gets its own chunk slices.
//   plan_only: stop after the plan (the device build fills the arrays with kernels, cs_build.cuh).
HostSparse make_sparse(const std::vector<int> &ptr, const uvec<int> &idx, const uvec<double> &val, int nt,
                       const FusePlan *fuse = nullptr, uvec<unsigned char> *fused_out = nullptr,
                       const std::vector<int> *split = nullptr, bool plan_only = false) {
    HostSparse h;
    std::vector<int> &chunk_src = h.chunk_src, &chunk_len = h.chunk_len;
    const int nseg = (int)ptr.size() - 1;
    // several lanes per segment only pay when there are too few segments to fill the machine (measured:
    // T>1 is slower once every warp has >= 2 thread-per-segment slices)
    const bool split_lanes = nseg < 300000;
    auto lg_lanes = [split_lanes](int len) { return (!split_lanes || len <= 8) ? 0 : len <= 16 ? 1 : len <= 32 ? 2 : 3; };  // T = 1,2,4,8 lanes
    size_t total = 0;
    auto plan_slice = [&](int seg0, int meta, int width) {
        h.slices.push_back(make_int4((int)std::min<size_t>(total, INT32_MAX), seg0, meta, width));
        total += 32u * (size_t)width;
    };
    // plan 1: chunks of the long segments (T = 32: entry e of the chunk at lane e%32, row e/32).  Pass 0 plans the part
    // every traversal walks (the K2 view), pass 1 the fused tails of the fused rows; slots are numbered per segment,
    // K2 part first, so that a chunk has the same slot in both views.
    const int n_split = split ? (int)split->size() : 0;
    std::vector<int> long_seg, first_slot;                 // the long segments (few) and the first slot of each (-1: none)
    for (int s = 0; s < nseg; ++s) {
        const int len = ptr[s + 1] - ptr[s];
        if (len <= kShortMax) continue;
        const int nu = s < n_split ? (*split)[s] : len, nf = len - nu;
        const int nch_u = (nu + kChunk - 1) / kChunk, nch_f = (nf + kChunk - 1) / kChunk;
        int fs = -1;
        if (nch_u + nch_f > 1 || nf > 0) { fs = h.n_slots; h.n_slots += nch_u + nch_f; }
        long_seg.push_back(s);
        first_slot.push_back(fs);
        if (nch_u + nch_f > 1) h.multi.push_back(make_int4(s, fs, nch_u + nch_f, 0));
        if (nf > 0) h.multi_k2.push_back(make_int4(s, fs, nch_u, s + 1));
        else if (nch_u > 1) h.multi_k2.push_back(make_int4(s, fs, nch_u, 0));
    }
    for (int pass = 0; pass < 2; ++pass) {
        for (size_t li = 0; li < long_seg.size(); ++li) {
            const int s = long_seg[li], len = ptr[s + 1] - ptr[s];
            const int nu = s < n_split ? (*split)[s] : len, nf = len - nu;
            const int nch_u = (nu + kChunk - 1) / kChunk;
            const int beg = pass ? ptr[s] + nu : ptr[s], cnt = pass ? nf : nu, nch = (cnt + kChunk - 1) / kChunk;
            const bool direct = nf == 0 && nch_u == 1;      // a single chunk that completes its segment
            for (int q = 0; q < nch; ++q) {
                const int a = beg + q * kChunk, clen = std::min(kChunk, beg + cnt - a);
                plan_slice(s, 1 | (5 << 8), (clen + 31) / 32);
                chunk_src.push_back(a);
                chunk_len.push_back(clen);
                int slot = direct ? -1 : first_slot[li] + (pass ? nch_u : 0) + q;
                if (pass && nu == 0 && nch == 1) slot = -1;  // all entries fused, one chunk: the full view completes it directly
                h.chunk_slot.push_back(slot);
            }
        }
        if (pass == 0) h.n_chunk_k2 = (int)h.slices.size();
    }
    h.n_chunk = (int)h.slices.size();
    // plan 2: runs of consecutive short segments -> slices of 32 lanes, T lanes per segment
    auto plan_run = [&](int a, int b) {
        int s0 = a;
        while (s0 < b) {
            const int lgT = lg_lanes(ptr[s0 + 1] - ptr[s0]), T = 1 << lgT, cap = 32 / T;
            int cnt = 1, maxlen = ptr[s0 + 1] - ptr[s0];
            while (cnt < cap && s0 + cnt < b && lg_lanes(ptr[s0 + cnt + 1] - ptr[s0 + cnt]) <= lgT) {
                maxlen = std::max(maxlen, ptr[s0 + cnt + 1] - ptr[s0 + cnt]);
                ++cnt;
            }
            plan_slice(s0, cnt | (lgT << 8), (maxlen + T - 1) / T);
            s0 += cnt;
        }
    };
    h.slices.reserve(h.slices.size() + (size_t)nseg / 32 + long_seg.size() + 2);
    int run = 0;
    for (int s : long_seg) {                                // the short segments between two long ones form a run
        plan_run(run, s);
        run = s + 1;
    }
    plan_run(run, nseg);
    h.total = total;
    if (total >= (size_t)INT32_MAX) { h.too_big = true; return h; }   // offsets are int32: refuse before anything is filled
    if (plan_only) return h;
    // fill (padding: val = 0, a valid index replicated)
    h.val.resize(total);          // no zero-fill: the fill below writes every slot (padding values = 0)
    h.idx.resize(total);
    h.pos.resize(idx.size());
    const int n_fuse = fuse ? fuse->rows() : 0, n_fa = fuse ? fuse->n_fa : 0;
    const int n_slice = (int)h.slices.size(), blk = 512;
    if (n_fuse) h.fmask.assign((size_t)(n_slice - h.n_chunk) * 32, (unsigned char)0);
    parallel_blocks((n_slice + blk - 1) / blk, nt, [&](int bi) {
        for (int si = bi * blk; si < std::min(n_slice, (bi + 1) * blk); ++si) {
            const int4 sl = h.slices[si];
            const size_t off = (size_t)sl.x;
            const int width = sl.w;
            if (si < h.n_chunk) {
                const int a = chunk_src[si], clen = chunk_len[si];
                for (int e = 0; e < 32 * width; ++e) {
                    h.idx[off + e] = idx[a + std::min(e, clen - 1)];
                    h.val[off + e] = e < clen ? val[a + e] : 0.0;
                    if (e < clen) h.pos[a + e] = (int)(off + e);
                }
                continue;
            }
            const int cnt = sl.z & 255, lgT = sl.z >> 8, T = 1 << lgT, s0 = sl.y;
            for (int lane = 0; lane < 32; ++lane) {
                const int seg = s0 + std::min(lane / T, cnt - 1);   // padding lanes replicate a valid index
                const int len = ptr[seg + 1] - ptr[seg], t = lane % T;
                for (int k = 0; k < width; ++k) {
                    const int e = k * T + t;
                    h.idx[off + 32u * k + lane] = len > 0 ? idx[ptr[seg] + std::min(e, len - 1)] : 0;  // empty segment: any valid index
                    const bool valid = lane / T < cnt && e < len;
                    h.val[off + 32u * k + lane] = valid ? val[ptr[seg] + e] : 0.0;
                    if (valid) h.pos[ptr[seg] + e] = (int)(off + 32u * k + lane);
                }
            }
            if (n_fuse && lgT == 0) {   // one thread per column: mark the entries the column pass takes over
                bool any_fused = false;
                int seen[kFuseB + 1], n_seen = 0;                    // class-B rows already fused in this slice (by a lower lane)
                for (int lane = 0; lane < cnt; ++lane) {
                    const int seg = s0 + lane, len = ptr[seg + 1] - ptr[seg];
                    for (int k = 0; k < std::min(len, kFuseK); ++k) {
                        const int i = idx[ptr[seg] + k];
                        if (i >= n_fuse) break;                      // rows ascend within a column
                        if (i >= n_fa) {                             // class B: one lane per row and slice
                            bool dup = false;
                            for (int q = 0; q < n_seen; ++q) dup |= seen[q] == i;
                            if (dup) continue;
                            seen[n_seen++] = i;
                        }
                        h.fmask[(size_t)(si - h.n_chunk) * 32 + lane] |= (unsigned char)(1u << k);
                        (*fused_out)[ptr[seg] + k] = 1;
                        any_fused = true;
                    }
                }
                if (any_fused) h.slices[si].z |= 1 << 16;
            }
        }
    });
    return h;
}

cs_status upload_sparse(cs_solver *S, const HostSparse &h, Sparse *out) {
    cs_status st;
    (out == &S->ctx.R ? S->tot_r : S->tot_c) = h.val.size();
    int4 *p4; int *pi; double *pd;
    if ((st = dev_upload(S, &p4, h.slices.data(), h.slices.size())) != CS_OK) return st; out->slices = p4;
    if ((st = dev_upload(S, &p4, h.multi.data(), h.multi.size())) != CS_OK) return st; out->multi = p4;
    if ((st = dev_upload(S, &p4, h.multi_k2.data(), h.multi_k2.size())) != CS_OK) return st; out->multi_k2 = p4;
    unsigned char *pu;
    if ((st = dev_upload(S, &pu, h.fmask.data(), h.fmask.size())) != CS_OK) return st; out->fmask = pu;
    if ((st = dev_upload(S, &pi, h.chunk_slot.data(), h.chunk_slot.size())) != CS_OK) return st; out->chunk_slot = pi;
    if ((st = dev_upload(S, &pi, h.idx.data(), h.idx.size())) != CS_OK) return st; out->idx = pi;
    if ((st = dev_upload(S, &pd, h.val.data(), h.val.size())) != CS_OK) return st; out->val0 = pd;
    if ((st = dev_alloc(S, &out->val, h.val.size())) != CS_OK) return st;      // scaled copy starts as the pristine one
    if (!h.val.empty()) CS_CUDA(S, cudaMemcpyAsync(out->val, pd, h.val.size() * sizeof(double), cudaMemcpyDeviceToDevice, S->stream));
    out->n_slice = (int)h.slices.size();
    out->n_chunk = h.n_chunk;
    out->n_chunk_k2 = h.n_chunk_k2;
    out->n_multi = (int)h.multi.size();
    out->n_multi_k2 = (int)h.multi_k2.size();
    return dev_zeros(S, &out->partial, (size_t)h.n_slots * 2);
}

// Stable sort of segment ids by decreasing length (counting sort); ids >= n_sort keep their place.
std::vector<int> order_by_length(const std::vector<int> &len, int n_sort) {
    const int n = (int)len.size();
    std::vector<int> perm(n);
    int maxlen = 0;
    for (int i = 0; i < n_sort; ++i) maxlen = std::max(maxlen, len[i]);
    std::vector<int> start((size_t)maxlen + 2, 0);
    for (int i = 0; i < n_sort; ++i) start[(size_t)(maxlen - len[i]) + 1]++;
    for (int q = 0; q <= maxlen; ++q) start[(size_t)q + 1] += start[q];
    for (int i = 0; i < n_sort; ++i) perm[start[maxlen - len[i]]++] = i;
    for (int i = n_sort; i < n; ++i) perm[i] = i;
    return perm;
}

// ---------------------------------------------------------------------------------------------------------------------
// cs_create on the device (cs_build.cuh): the O(nnz) work -- validation, the two ordered compressed copies (one radix sort
// each), the slice fill, the fusion marks, the fused rows' partition -- runs as kernels on the uploaded CSR; the host does
// the O(m + n) part (length ordering, prefix sums, slice plans).  Same layouts as the host build, bit for bit.
// ---------------------------------------------------------------------------------------------------------------------
int ew_blocks(int n) { return std::max(1, std::min((n + 255) / 256, 148 * 8)); }

struct DevTmp {                                   // scratch of the build: stream-ordered allocations, released on every path
    std::vector<void *> p;
    cudaStream_t stream = nullptr;
    ~DevTmp() { for (void *q : p) cudaFreeAsync(q, stream); }
    template <class T>
    cs_status alloc(cs_solver *S, T **out, size_t count, bool zero = false) {
        void *q = nullptr;
        stream = S->stream;
        CS_CUDA(S, cudaMallocAsync(&q, std::max<size_t>(count, 1) * sizeof(T), S->stream));
        p.push_back(q);
        *out = static_cast<T *>(q);
        if (zero) CS_CUDA(S, cudaMemsetAsync(q, 0, std::max<size_t>(count, 1) * sizeof(T), S->stream));
        return CS_OK;
    }
};

// plan -> device Sparse: uploads the descriptors, allocates the slice storage; chunk_src / chunk_len go to scratch
cs_status upload_plan(cs_solver *S, DevTmp &tmp, const HostSparse &h, Sparse *out, int4 **d_slices, int **d_csrc, int **d_clen, int **d_idx,
                      double **d_val0, bool with_fmask) {
    cs_status st;
    (out == &S->ctx.R ? S->tot_r : S->tot_c) = h.total;
    int4 *p4; int *pi;
    if ((st = dev_upload(S, d_slices, h.slices.data(), h.slices.size())) != CS_OK) return st; out->slices = *d_slices;
    if ((st = dev_upload(S, &p4, h.multi.data(), h.multi.size())) != CS_OK) return st; out->multi = p4;
    if ((st = dev_upload(S, &p4, h.multi_k2.data(), h.multi_k2.size())) != CS_OK) return st; out->multi_k2 = p4;
    if ((st = dev_upload(S, &pi, h.chunk_slot.data(), h.chunk_slot.size())) != CS_OK) return st; out->chunk_slot = pi;
    if ((st = tmp.alloc(S, d_csrc, h.chunk_src.size())) != CS_OK) return st;
    if ((st = tmp.alloc(S, d_clen, h.chunk_len.size())) != CS_OK) return st;
    if (!h.chunk_src.empty()) {
        CS_CUDA(S, cudaMemcpyAsync(*d_csrc, h.chunk_src.data(), sizeof(int) * h.chunk_src.size(), cudaMemcpyHostToDevice, S->stream));
        CS_CUDA(S, cudaMemcpyAsync(*d_clen, h.chunk_len.data(), sizeof(int) * h.chunk_len.size(), cudaMemcpyHostToDevice, S->stream));
    }
    if ((st = dev_alloc(S, d_idx, h.total)) != CS_OK) return st; out->idx = *d_idx;
    if ((st = dev_alloc(S, d_val0, h.total)) != CS_OK) return st; out->val0 = *d_val0;
    if ((st = dev_alloc(S, &out->val, h.total)) != CS_OK) return st;
    unsigned char *pu = nullptr;
    const size_t nmask = with_fmask ? (h.slices.size() - (size_t)h.n_chunk) * 32 : 0;
    if ((st = dev_zeros(S, &pu, nmask)) != CS_OK) return st; out->fmask = pu;
    out->n_slice = (int)h.slices.size();
    out->n_chunk = h.n_chunk;
    out->n_chunk_k2 = h.n_chunk_k2;
    out->n_multi = (int)h.multi.size();
    out->n_multi_k2 = (int)h.multi_k2.size();
    return dev_zeros(S, &out->partial, (size_t)h.n_slots * 2);
}

template <class LapFn>
cs_status layout_device(cs_solver *S, const cs_csr *A, const double *b, const double *c, cs_mem vec_where, const cs_cones *K, int m, int n,
                        int nnz, std::vector<int> &perm_r, std::vector<int> &perm_c, std::vector<double> &hb, std::vector<double> &hc,
                        double &nb, double &nc, LapFn lap) {
    DevTmp tmp;
    cs_status st;
    Ctx &x = S->ctx;
    const int grid = 148 * 8;
    // ---- the caller's CSR on the device
    const int *d_rptr = A->row_ptr, *d_cidx = A->col_idx;
    const double *d_val = A->val;
    std::vector<int> rptr_v;
    const int *rptr = A->row_ptr;
    if (A->where == CS_HOST) {
        int *q; double *qd;
        if ((st = tmp.alloc(S, &q, (size_t)m + 1)) != CS_OK) return st;
        CS_CUDA(S, cudaMemcpyAsync(q, A->row_ptr, sizeof(int) * ((size_t)m + 1), cudaMemcpyHostToDevice, S->stream)); d_rptr = q;
        if ((st = tmp.alloc(S, &q, (size_t)nnz)) != CS_OK) return st;
        CS_CUDA(S, cudaMemcpyAsync(q, A->col_idx, sizeof(int) * (size_t)nnz, cudaMemcpyHostToDevice, S->stream)); d_cidx = q;
        if ((st = tmp.alloc(S, &qd, (size_t)nnz)) != CS_OK) return st;
        CS_CUDA(S, cudaMemcpyAsync(qd, A->val, sizeof(double) * (size_t)nnz, cudaMemcpyHostToDevice, S->stream)); d_val = qd;
    } else {
        if ((st = fetch(S, rptr_v, A->row_ptr, (size_t)m + 1, A->where)) != CS_OK) return st;
        rptr = rptr_v.data();
    }
    // b, c: raw copies on the device (permuted there once the ordering is known); the host reads them for the norms
    const double *hb_p = b, *hc_p = c, *d_braw = b, *d_craw = c;
    if (vec_where == CS_HOST) {
        double *qd;
        if ((st = tmp.alloc(S, &qd, (size_t)m)) != CS_OK) return st;
        CS_CUDA(S, cudaMemcpyAsync(qd, b, sizeof(double) * (size_t)m, cudaMemcpyHostToDevice, S->stream)); d_braw = qd;
        if ((st = tmp.alloc(S, &qd, (size_t)n)) != CS_OK) return st;
        CS_CUDA(S, cudaMemcpyAsync(qd, c, sizeof(double) * (size_t)n, cudaMemcpyHostToDevice, S->stream)); d_craw = qd;
    } else {
        if ((st = fetch(S, hb, b, (size_t)m, vec_where)) != CS_OK) return st;
        if ((st = fetch(S, hc, c, (size_t)n, vec_where)) != CS_OK) return st;
        hb_p = hb.data(); hc_p = hc.data();
    }
    if (rptr[0] != 0 || rptr[m] != nnz) { S->err = "row_ptr[0] != 0 or row_ptr[m] != nnz"; return CS_EINVAL; }
    std::vector<int> long_rows;                                       // validated by one CTA each
    for (int i = 0; i < m; ++i) {
        if (rptr[i + 1] <= rptr[i]) { S->err = "row_ptr not increasing (empty rows are not allowed)"; return CS_EINVAL; }
        if (rptr[i + 1] > nnz) { S->err = "row_ptr out of range"; return CS_EINVAL; }
        if (rptr[i + 1] - rptr[i] > csb::kValidateLong) long_rows.push_back(i);
    }
    // ---- validation + column counts (device)
    int *d_clen, *d_status;
    if ((st = tmp.alloc(S, &d_clen, (size_t)n, true)) != CS_OK) return st;
    if ((st = tmp.alloc(S, &d_status, 1, true)) != CS_OK) return st;
    csb::k_validate<<<grid, 256, 0, S->stream>>>(d_rptr, d_cidx, d_val, m, n, d_clen, d_status);
    if (!long_rows.empty()) {
        int *d_long;
        if ((st = tmp.alloc(S, &d_long, long_rows.size())) != CS_OK) return st;
        CS_CUDA(S, cudaMemcpyAsync(d_long, long_rows.data(), sizeof(int) * long_rows.size(), cudaMemcpyHostToDevice, S->stream));
        csb::k_validate_long<<<std::min((int)long_rows.size(), grid), 256, 0, S->stream>>>(d_rptr, d_cidx, d_val, d_long, (int)long_rows.size(), n,
                                                                                       d_clen, d_status);
    }
    int status = 0;
    CS_CUDA(S, cudaMemcpyAsync(&status, d_status, sizeof(int), cudaMemcpyDeviceToHost, S->stream));
    nb = 0.0; nc = 0.0;                                                // meanwhile on the host: b, c
    for (int i = 0; i < m; ++i) { if (!std::isfinite(hb_p[i])) { S->err = "non-finite b"; return CS_EINVAL; } nb += hb_p[i] * hb_p[i]; }
    for (int j = 0; j < n; ++j) { if (!std::isfinite(hc_p[j])) { S->err = "non-finite c"; return CS_EINVAL; } nc += hc_p[j] * hc_p[j]; }
    CS_CUDA(S, cudaStreamSynchronize(S->stream));
    S->launches += 1;
    if (status & csb::kBadIndex) { S->err = "col_idx out of range, unsorted or duplicated within a row"; return CS_EINVAL; }
    if (status & csb::kBadValue) { S->err = "non-finite matrix entry"; return CS_EINVAL; }
    if (status & csb::kZeroRow) { S->err = "a row of A has zero norm (all stored entries are 0 or underflow when squared)"; return CS_EINVAL; }
    lap("upload + validate (device)");
    // ---- internal ordering: stable sorts by decreasing length (rows; the orthant columns), inverse permutations, new pointers
    const int n_lin = (int)K->n_lin, nmax = std::max(m, n);
    unsigned *lk, *lk_s, *io;
    int *d_perm_r, *d_perm_c, *d_inv_r, *d_inv_c, *d_rp2, *d_cp2, *d_len;
    if ((st = tmp.alloc(S, &lk, (size_t)nmax)) != CS_OK) return st;
    if ((st = tmp.alloc(S, &lk_s, (size_t)nmax)) != CS_OK) return st;
    if ((st = tmp.alloc(S, &io, (size_t)nmax)) != CS_OK) return st;
    if ((st = tmp.alloc(S, &d_len, (size_t)nmax + 1)) != CS_OK) return st;
    if ((st = tmp.alloc(S, &d_inv_r, (size_t)m)) != CS_OK) return st;
    if ((st = tmp.alloc(S, &d_inv_c, (size_t)n)) != CS_OK) return st;
    if ((st = dev_alloc(S, &d_perm_r, (size_t)m)) != CS_OK) return st; x.perm_r = d_perm_r;
    if ((st = dev_alloc(S, &d_perm_c, (size_t)n)) != CS_OK) return st; x.perm_c = d_perm_c;
    if ((st = dev_alloc(S, &d_rp2, (size_t)m + 1)) != CS_OK) return st; x.Rc.ptr = d_rp2;
    if ((st = dev_alloc(S, &d_cp2, (size_t)n + 1)) != CS_OK) return st; x.Cc.ptr = d_cp2;
    size_t ob1 = 0, ob2 = 0;
    CS_CUDA(S, cub::DeviceRadixSort::SortPairs(nullptr, ob1, lk, lk_s, io, reinterpret_cast<unsigned *>(d_perm_r), nmax, 0, 32, S->stream));
    CS_CUDA(S, cub::DeviceScan::ExclusiveSum(nullptr, ob2, d_len, d_rp2, nmax + 1, S->stream));
    unsigned char *otmp;
    const size_t ob = std::max(ob1, ob2) + 16;
    if ((st = tmp.alloc(S, &otmp, ob)) != CS_OK) return st;
    size_t obq = ob;
    csb::k_len_keys<<<grid, 256, 0, S->stream>>>(d_rptr, 1, m, lk, io);
    CS_CUDA(S, cub::DeviceRadixSort::SortPairs(otmp, obq, lk, lk_s, io, reinterpret_cast<unsigned *>(d_perm_r), m, 0, 32, S->stream));
    csb::k_invert_and_len<<<grid, 256, 0, S->stream>>>(d_perm_r, d_rptr, 1, m, d_inv_r, d_len);
    obq = ob;
    CS_CUDA(S, cub::DeviceScan::ExclusiveSum(otmp, obq, d_len, d_rp2, m + 1, S->stream));
    if (n_lin > 0) {
        csb::k_len_keys<<<grid, 256, 0, S->stream>>>(d_clen, 0, n_lin, lk, io);
        obq = ob;
        CS_CUDA(S, cub::DeviceRadixSort::SortPairs(otmp, obq, lk, lk_s, io, reinterpret_cast<unsigned *>(d_perm_c), n_lin, 0, 32, S->stream));
    }
    csb::k_iota_tail<<<grid, 256, 0, S->stream>>>(d_perm_c, n_lin, n);
    csb::k_invert_and_len<<<grid, 256, 0, S->stream>>>(d_perm_c, d_clen, 0, n, d_inv_c, d_len);
    obq = ob;
    CS_CUDA(S, cub::DeviceScan::ExclusiveSum(otmp, obq, d_len, d_cp2, n + 1, S->stream));
    // b, c in internal order
    double *d_b, *d_c;
    if ((st = dev_alloc(S, &d_b, (size_t)m)) != CS_OK) return st; x.b = d_b;
    if ((st = dev_alloc(S, &d_c, (size_t)n)) != CS_OK) return st; x.c = d_c;
    k_gather_perm<<<ew_blocks(m), 256, 0, S->stream>>>(d_b, d_braw, d_perm_r, m);
    k_gather_perm<<<ew_blocks(n), 256, 0, S->stream>>>(d_c, d_craw, d_perm_c, n);
    std::vector<int> rp2((size_t)m + 1), cp2((size_t)n + 1);        // the slice plans are made on the host
    CS_CUDA(S, cudaMemcpyAsync(rp2.data(), d_rp2, sizeof(int) * ((size_t)m + 1), cudaMemcpyDeviceToHost, S->stream));
    CS_CUDA(S, cudaMemcpyAsync(cp2.data(), d_cp2, sizeof(int) * ((size_t)n + 1), cudaMemcpyDeviceToHost, S->stream));
    CS_CUDA(S, cudaStreamSynchronize(S->stream));
    S->launches += 9;
    for (int i = 0; i < m && rp2[(size_t)i + 1] - rp2[i] > kShortMax; ++i) x.n_long = i + 1;
    lap("row/column ordering");
    // ---- the two compressed copies: one radix sort each
    unsigned long long *key_c, *key_r, *key_s;
    unsigned int *pay, *pay_s;
    if ((st = tmp.alloc(S, &key_c, (size_t)nnz)) != CS_OK) return st;
    if ((st = tmp.alloc(S, &key_r, (size_t)nnz)) != CS_OK) return st;
    if ((st = tmp.alloc(S, &key_s, (size_t)nnz)) != CS_OK) return st;
    if ((st = tmp.alloc(S, &pay, (size_t)nnz)) != CS_OK) return st;
    if ((st = tmp.alloc(S, &pay_s, (size_t)nnz)) != CS_OK) return st;
    csb::k_keys<<<grid, 256, 0, S->stream>>>(d_rptr, d_cidx, m, d_inv_r, d_inv_c, key_c, key_r, pay);
    auto bits = [](int v) { int b = 1; while ((1ll << b) < (long long)v) ++b; return b; };
    const int end_c = 32 + bits(n), end_r = 32 + bits(m);       // the high word holds an internal column / row number
    size_t cub_bytes = 0;
    CS_CUDA(S, cub::DeviceRadixSort::SortPairs(nullptr, cub_bytes, key_c, key_s, pay, pay_s, nnz, 0, 64, S->stream));
    unsigned char *cub_tmp;
    if ((st = tmp.alloc(S, &cub_tmp, cub_bytes + 16)) != CS_OK) return st;
    int *ri2, *ci2;
    double *cv2, *va2;
    if ((st = dev_alloc(S, &ri2, (size_t)nnz)) != CS_OK) return st; x.Cc.idx = ri2;
    if ((st = dev_alloc(S, &ci2, (size_t)nnz)) != CS_OK) return st; x.Rc.idx = ci2;
    if ((st = tmp.alloc(S, &cv2, (size_t)nnz)) != CS_OK) return st;
    if ((st = tmp.alloc(S, &va2, (size_t)nnz)) != CS_OK) return st;
    CS_CUDA(S, cub::DeviceRadixSort::SortPairs(cub_tmp, cub_bytes, key_c, key_s, pay, pay_s, nnz, 0, end_c, S->stream));
    csb::k_gather_c<<<grid, 256, 0, S->stream>>>(key_s, pay_s, d_val, nnz, ri2, cv2);
    CS_CUDA(S, cub::DeviceRadixSort::SortPairs(cub_tmp, cub_bytes, key_r, key_s, pay, pay_s, nnz, 0, end_r, S->stream));
    csb::k_gather_r<<<grid, 256, 0, S->stream>>>(pay_s, d_cidx, d_val, d_inv_c, nnz, ci2, va2);
    S->launches += 5;
    CS_CUDA(S, cudaGetLastError());
    lap("compressed copies (2 radix sorts)");
    // ---- column-major copy: plan (host), fill + fusion marks (device)
    const int nt = host_threads();
    const uvec<int> no_idx;
    const uvec<double> no_val;
    FusePlan fuse;
    if (nnz > kOneCtaNnz)
        for (int i = 0; i < std::min(m, kFuseA + kFuseB) && rp2[(size_t)i + 1] - rp2[i] >= kFuseMinLen; ++i)
            (i < kFuseA ? fuse.n_fa : fuse.n_fb) += 1;
    const HostSparse hc2 = make_sparse(cp2, no_idx, no_val, nt, nullptr, nullptr, nullptr, true);
    lap("  column-major plan (host)");
    if (hc2.too_big) { S->err = "padded slice storage exceeds 2^31 entries"; return CS_EINVAL; }
    int4 *d_sl; int *d_csrc, *d_clen2, *d_idx, *d_pos;
    double *d_val0;
    if ((st = upload_plan(S, tmp, hc2, &x.C, &d_sl, &d_csrc, &d_clen2, &d_idx, &d_val0, fuse.rows() > 0)) != CS_OK) return st;
    if ((st = dev_alloc(S, &d_pos, (size_t)nnz)) != CS_OK) return st; x.Cc.pos = d_pos;
    lap("  column-major allocations + plan upload");
    unsigned char *fused_c;
    if ((st = tmp.alloc(S, &fused_c, (size_t)nnz, fuse.rows() > 0)) != CS_OK) return st;
    csb::k_fill_slices<<<grid, 256, 0, S->stream>>>(d_sl, x.C.n_slice, x.C.n_chunk, d_csrc, d_clen2, d_cp2, ri2, cv2, d_idx, d_val0, d_pos,
                                                    fuse.rows(), fuse.n_fa, const_cast<unsigned char *>(x.C.fmask), fused_c);
    CS_CUDA(S, cudaMemcpyAsync(x.C.val, d_val0, sizeof(double) * hc2.total, cudaMemcpyDeviceToDevice, S->stream));
    S->launches += 1;
    // ---- fused rows of the row-major copy: unfused entries first
    std::vector<int> split((size_t)fuse.rows());
    if (fuse.rows()) {
        const int nf = fuse.rows(), region = rp2[nf];
        int *flag, *sc, *ci2_o, *d_split;
        double *va2_o;
        if ((st = tmp.alloc(S, &flag, (size_t)region + 1)) != CS_OK) return st;
        if ((st = tmp.alloc(S, &sc, (size_t)region + 1)) != CS_OK) return st;
        if ((st = tmp.alloc(S, &ci2_o, (size_t)region)) != CS_OK) return st;
        if ((st = tmp.alloc(S, &va2_o, (size_t)region)) != CS_OK) return st;
        if ((st = tmp.alloc(S, &d_split, (size_t)nf)) != CS_OK) return st;
        csb::k_fused_flags<<<grid, 256, 0, S->stream>>>(d_rp2, ci2, d_cp2, ri2, fused_c, nf, flag);
        size_t scan_bytes = 0;
        CS_CUDA(S, cub::DeviceScan::ExclusiveSum(nullptr, scan_bytes, flag, sc, region + 1, S->stream));
        unsigned char *scan_tmp;
        if ((st = tmp.alloc(S, &scan_tmp, scan_bytes + 16)) != CS_OK) return st;
        CS_CUDA(S, cub::DeviceScan::ExclusiveSum(scan_tmp, scan_bytes, flag, sc, region + 1, S->stream));
        csb::k_fused_partition<<<grid, 256, 0, S->stream>>>(d_rp2, flag, sc, nf, ci2, va2, ci2_o, va2_o, d_split);
        CS_CUDA(S, cudaMemcpyAsync(ci2, ci2_o, sizeof(int) * (size_t)region, cudaMemcpyDeviceToDevice, S->stream));
        CS_CUDA(S, cudaMemcpyAsync(va2, va2_o, sizeof(double) * (size_t)region, cudaMemcpyDeviceToDevice, S->stream));
        CS_CUDA(S, cudaMemcpyAsync(split.data(), d_split, sizeof(int) * (size_t)nf, cudaMemcpyDeviceToHost, S->stream));
        CS_CUDA(S, cudaStreamSynchronize(S->stream));
        S->launches += 3;
        x.n_fa = fuse.n_fa;
        x.n_fb = fuse.n_fb;
    }
    lap("column-major slices + fused rows");
    // ---- row-major copy: plan (host, needs the split), fill (device)
    const HostSparse hr = make_sparse(rp2, no_idx, no_val, nt, nullptr, nullptr, fuse.rows() ? &split : nullptr, true);
    if (hr.too_big) { S->err = "padded slice storage exceeds 2^31 entries"; return CS_EINVAL; }
    if ((st = upload_plan(S, tmp, hr, &x.R, &d_sl, &d_csrc, &d_clen2, &d_idx, &d_val0, false)) != CS_OK) return st;
    if ((st = dev_alloc(S, &d_pos, (size_t)nnz)) != CS_OK) return st; x.Rc.pos = d_pos;
    csb::k_fill_slices<<<grid, 256, 0, S->stream>>>(d_sl, x.R.n_slice, x.R.n_chunk, d_csrc, d_clen2, d_rp2, ci2, va2, d_idx, d_val0, d_pos, 0, 0,
                                                    nullptr, nullptr);
    CS_CUDA(S, cudaMemcpyAsync(x.R.val, d_val0, sizeof(double) * hr.total, cudaMemcpyDeviceToDevice, S->stream));
    S->launches += 1;
    CS_CUDA(S, cudaGetLastError());
    CS_CUDA(S, cudaStreamSynchronize(S->stream));    // the scratch (DevTmp) is freed on return
    lap("row-major slices");
    return CS_OK;
}

cs_status launch_coop(cs_solver *S, const void *fn, void **args) {
    // k_iterate_dense runs the same CG (fused column pass included) when a Cholesky pivot fails, so it gets the same shared memory
    const bool iter = fn == (const void *)k_iterate || fn == (const void *)k_iterate_dense;
    const size_t dyn = iter ? S->dyn_smem : 0;
    // the shared-memory carve-out is a property of the FUNCTION, shared by every handle of the process: a handle without
    // fused rows must not inherit the 100 KB another handle asked for (its gathers would lose 100 KB of L1)
    if (iter)
        CS_CUDA(S, cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, dyn ? kFuseCarveoutPct : (int)cudaSharedmemCarveoutDefault));
    CS_CUDA(S, cudaLaunchCooperativeKernel(fn, dim3(S->grid), dim3(kBlock), args, dyn, S->stream));
    S->launches += 1;
    return CS_OK;
}

cs_status ensure_xz(cs_solver *S) {
    if (!S->xz_stale) return CS_OK;
    k_materialize_xz<<<std::max(1, std::min((S->ctx.n + 255) / 256, 148 * 8)), 256, 0, S->stream>>>(S->ctx);
    CS_CUDA(S, cudaGetLastError());
    S->launches += 1;
    S->xz_stale = false;
    return CS_OK;
}

void sync_params(cs_solver *S) {
    S->ctx.cg_tol = S->prm.cg_tol;
    S->ctx.cg_reduce = S->prm.cg_reduce;
    S->ctx.cg_max_iter = S->prm.cg_max_iter;
}

// Grid dense path: M = A~A~', its blocked Cholesky factor and the explicit inverse, from the values k_condition has
// just rescaled (cs_dense.cuh).  Ordinary kernel launches on the handle's stream, no host synchronisation.
cs_status dense_grid_factor(cs_solver *S) {
    const Ctx &c = S->ctx;
    const int m = c.m, n = c.n;
    const size_t mm = (size_t)m * m;
    const int tiles = (m + kGemmT - 1) / kGemmT, n_tri = tiles * (tiles + 1) / 2, one = 1;
    CS_CUDA(S, cudaMemsetAsync(c.gAd, 0, sizeof(double) * (size_t)m * n, S->stream));
    CS_CUDA(S, cudaMemsetAsync(c.gZ, 0, sizeof(double) * mm, S->stream));
    CS_CUDA(S, cudaMemcpyAsync(c.g_ok, &one, sizeof(int), cudaMemcpyHostToDevice, S->stream));
    k_dense_scatter<<<148 * 4, 256, 0, S->stream>>>(c, c.gAd);
    k_dense_aat<<<n_tri, 256, 0, S->stream>>>(c.gAd, m, n, c.gM, 0);
    CS_CUDA(S, cudaMemcpyAsync(c.gL, c.gM, sizeof(double) * mm, cudaMemcpyDeviceToDevice, S->stream));
    S->launches += 2;
    for (int pb = 0; pb < m; pb += kCholPanel) {
        const int pend = std::min(pb + kCholPanel, m);
        for (int kb = pb; kb < pend; kb += kCholNB) {
            k_chol_diag<<<1, kCholNB * kCholNB, 0, S->stream>>>(c.gL, m, kb, c.g_ok);
            S->launches += 1;
            const int rest = m - kb - kCholNB;
            if (rest <= 0) break;
            k_chol_panel<<<std::min(148 * 4, (rest + 7) / 8), 256, 0, S->stream>>>(c.gL, m, kb);
            S->launches += 1;
            if (kb + kCholNB < pend) {                           // the panel's remaining columns
                k_chol_update<<<dim3((rest + 63) / 64, (pend - kb - kCholNB + 63) / 64), 256, 0, S->stream>>>(c.gL, m, kb, pend);
                S->launches += 1;
            }
        }
        if (pend < m) {                                          // everything behind the panel, rank 128
            const int t = (m - pend + kGemmT - 1) / kGemmT;
            k_chol_update_panel<<<t * (t + 1) / 2, 256, 0, S->stream>>>(c.gL, m, pb, pend);
            S->launches += 1;
        }
    }
    // Z = L^-T by column groups (inverses of the diagonal blocks first), then Minv = Z Z'
    k_dense_diag_inv<<<(m + kTriNB - 1) / kTriNB, kTriNB, 0, S->stream>>>(c.gL, m, c.gDinv);
    {   // the widest column group that still gives every SM two CTAs (cs_dense.cuh)
        auto run = [&](auto tag) -> cs_status {
            constexpr int CW = decltype(tag)::value;
            CS_CUDA(S, cudaFuncSetAttribute((const void *)k_dense_trinv_blk<CW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TrinvSmem<CW>)));
            k_dense_trinv_blk<CW><<<(m + CW - 1) / CW, kTriThreads, sizeof(TrinvSmem<CW>), S->stream>>>(c.gL, c.gDinv, m, c.gZ);
            return CS_OK;
        };
        const int sms2 = 2 * 148;
        cs_status st = m >= 32 * sms2 ? run(std::integral_constant<int, 32>{}) : m >= 16 * sms2 ? run(std::integral_constant<int, 16>{})
                                                                                                : run(std::integral_constant<int, 8>{});
        if (st != CS_OK) return st;
    }
    k_dense_aat<<<n_tri, 256, 0, S->stream>>>(c.gZ, m, m, c.gMinv, 1);
    S->launches += 3;
    CS_CUDA(S, cudaGetLastError());
    return CS_OK;
}

cs_status do_condition(cs_solver *S, int use_rule) {
    cs_status st = ensure_xz(S);
    if (st != CS_OK) return st;
    // automatic: FSAI(1) pays when the conditioning may spread O^2 over many decades (t = 9.2 for LPs);
    // with the SOCP setting t = 1.7 it saves ~10 % of the CG steps and costs 18 % per step (measured)
    if (S->dense_capable && !S->ctx.gM && S->ctx.m <= S->prm.dense_m_threshold) {
        // buffers of the grid dense path, on first use: Ad [m][n], four [m][m] matrices (24 GB at the paper's largest LP,
        // n = 30000).  If the device cannot hold them the solve stays with CG: not an error.
        Ctx &x = S->ctx;
        const size_t m = (size_t)x.m, mm = m * m, nd = ((m + kTriNB - 1) / kTriNB) * kTriNB * kTriNB;
        const size_t npart = std::max<size_t>((size_t)x.n, (size_t)kMaxGrid * (kBlock / 32) * 64);   // [row ranges][n], ranges * n <= warps * 64
        const size_t counts[] = {m * (size_t)x.n, mm, mm, mm, mm, nd, 4 * m, npart};
        double **ptrs[] = {&x.gAd, &x.gM, &x.gL, &x.gZ, &x.gMinv, &x.gDinv, &x.dv, &x.gpart};
        constexpr int NB = 8;
        void *got[NB] = {};
        bool ok = true;
        for (int q = 0; q < NB && ok; ++q) ok = cudaMalloc(&got[q], counts[q] * sizeof(double)) == cudaSuccess;
        if (ok) ok = cudaMalloc((void **)&x.g_ok, sizeof(int)) == cudaSuccess;
        if (!ok) {
            cudaGetLastError();                                  // clear the allocation error
            for (void *q : got) if (q) cudaFree(q);
            x.g_ok = nullptr;
            S->dense_capable = false;
        } else {
            for (int q = 0; q < NB; ++q) { *ptrs[q] = static_cast<double *>(got[q]); S->allocs.push_back(got[q]); }
            S->allocs.push_back(x.g_ok);
            CS_CUDA(S, cudaMemsetAsync(x.dv, 0, 4 * m * sizeof(double), S->stream));
        }
    }
    S->ctx.dense = (S->grid == 1 && S->ctx.dM && S->ctx.m <= std::min(S->prm.dense_m_threshold, kDenseMax)) ? 1
                 : (S->grid > 1 && S->ctx.gM && S->ctx.m <= S->prm.dense_m_threshold) ? 2 : 0;
    // automatic: FSAI pays when the conditioning may spread O^2 over many decades (t = 9.2 for LPs); FSAI(5) where the
    // matrix copies are L2-resident but the passes not yet latency-bound (config 2: 1.22x faster per pass; config 1: its two
    // dependent gather passes and the heavier build cost what the saved steps gain; config 4: slower), FSAI(1) otherwise
    const double mat_bytes = 24.0 * (double)S->nnz;
    const int auto_fsai = mat_bytes >= kAutoFsaiPMinBytes && mat_bytes <= kAutoFsaiPBytes ? 2 : 1;
    S->ctx.fsai = S->ctx.dense ? 0 : S->prm.precond == 3 ? 2 : S->prm.precond == 2 ? 1 : (S->prm.precond == 0 && S->prm.t >= 4.0) ? auto_fsai : 0;
    if (S->ctx.fsai == 2 && !S->ctx.fp_ctop) {   // the tables of FSAI(5) (~76 bytes per row + 24 per column) are allocated on first use
        Ctx &x = S->ctx;
        const size_t m = (size_t)x.m, n = (size_t)x.n;
        if ((st = dev_zeros(S, &x.fp_idx, kFsP * m)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.fp_tptr, m + 1)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.fp_tcnt, m)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.fp_trow, kFsP * m)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.fp_val, (kFsP + 1) * m)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.fp_tval, kFsP * m)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.fp_ctop, kFsTop * n)) != CS_OK) return st;
    }
    S->ctx.mu = S->prm.mu;  // mu, t, o_floor, precond take effect here (cs.h)
    S->ctx.t = S->prm.t;
    S->ctx.o_floor = S->prm.o_floor;
    sync_params(S);
    void *args[] = {&S->ctx, &use_rule};
    st = launch_coop(S, (const void *)k_condition, args);
    if (st != CS_OK) return st;
    if (S->ctx.dense == 2 && (st = dense_grid_factor(S)) != CS_OK) return st;
    S->conditioned = true;
    S->started = true;
    S->stall_at = -1;          // residuals of the old scaling do not compare with the new one's
    return CS_OK;
}


// caller's n-vector (host or device) -> internal order, into dst (device)
cs_status import_cols(cs_solver *S, double *dst, const double *src, cs_mem where) {
    const Ctx &c = S->ctx;
    const double *dsrc = src;
    if (where == CS_HOST) {
        CS_CUDA(S, cudaMemcpyAsync(c.e, src, sizeof(double) * c.n, cudaMemcpyHostToDevice, S->stream));  // e = scratch
        dsrc = c.e;
    }
    k_gather_perm<<<ew_blocks(c.n), 256, 0, S->stream>>>(dst, dsrc, c.perm_c, c.n);
    CS_CUDA(S, cudaGetLastError());
    S->launches += 1;
    if (where == CS_HOST) CS_CUDA(S, cudaStreamSynchronize(S->stream));
    return CS_OK;
}

// internal n-vector -> caller's order and memory space
cs_status export_cols(cs_solver *S, double *dst, const double *src, cs_mem where) {
    const Ctx &c = S->ctx;
    double *ddst = where == CS_HOST ? c.e : dst;
    k_scatter_perm<<<ew_blocks(c.n), 256, 0, S->stream>>>(ddst, src, c.perm_c, c.n);
    CS_CUDA(S, cudaGetLastError());
    S->launches += 1;
    if (where == CS_HOST) CS_CUDA(S, cudaMemcpyAsync(dst, c.e, sizeof(double) * c.n, cudaMemcpyDeviceToHost, S->stream));
    return CS_OK;
}

}  // namespace

// =================================================================================================
extern "C" {

const char *cs_last_error(const cs_solver *S) { return S ? S->err.c_str() : g_create_err.c_str(); }

void cs_destroy(cs_solver *S) {
    if (!S) return;
    DeviceGuard guard(S);
    cudaStreamSynchronize(S->stream);
    for (void *p : S->allocs) cudaFree(p);
    delete S;
}

int64_t cs_kernel_launches(const cs_solver *S) { return S ? S->launches : 0; }

static cs_status create_impl(cs_solver *S, const cs_csr *A, const double *b, const double *c, cs_mem vec_where,
                             const cs_cones *K) {
    const bool verbose = getenv("CS_VERBOSE") != nullptr;      // stage timings of cs_create on stderr
    auto t_prev = std::chrono::steady_clock::now();
    auto lap = [&](const char *what) {
        if (!verbose) return;
        const auto t = std::chrono::steady_clock::now();
        fprintf(stderr, "[cs_create] %-28s %8.1f ms\n", what, std::chrono::duration<double, std::milli>(t - t_prev).count());
        t_prev = t;
    };
    const int64_t m64 = A->m, n64 = A->n, nnz64 = A->nnz;
    if (m64 <= 0 || n64 <= 0 || nnz64 <= 0 || m64 >= INT32_MAX || n64 >= INT32_MAX || nnz64 >= INT32_MAX) {
        S->err = "sizes must be positive and below 2^31";
        return CS_EINVAL;
    }
    const int m = (int)m64, n = (int)n64, nnz = (int)nnz64;
    // ---- cones
    if (K->n_lin < 0 || K->n_soc < 0 || (K->n_soc > 0 && !K->soc_size)) { S->err = "bad cone spec"; return CS_EINVAL; }
    std::vector<int> cone_off((size_t)K->n_soc + 1);
    int64_t off = K->n_lin;
    for (int64_t i = 0; i < K->n_soc; ++i) {
        if (K->soc_size[i] < 1) { S->err = "soc_size entries must be >= 1"; return CS_EINVAL; }
        cone_off[i] = (int)off;
        off += K->soc_size[i];
        if (off > n64) break;
    }
    if (off != n64) { S->err = "n_lin + sum(soc_size) != n"; return CS_EINVAL; }
    cone_off[K->n_soc] = n;
    // ---- the layout: internal ordering, the two sliced copies, the fusion plan -- built on the device (cs_build.cuh) for
    //      all but small problems, on the host otherwise (and on request: cs_diag_create, for the layout-identity test)
    cs_status st;
    std::vector<int> perm_r, perm_c;
    std::vector<double> hb, hc;
    double nb = 0.0, nc = 0.0;
    const bool device_build = S->build_mode == 2 || (S->build_mode == 0 && nnz >= kDeviceBuildMinNnz);
    if (device_build) {
        if ((st = layout_device(S, A, b, c, vec_where, K, m, n, nnz, perm_r, perm_c, hb, hc, nb, nc, lap)) != CS_OK) return st;
    } else {
        // ---- fetch and validate A
        std::vector<int> rptr_v, cidx_v;
        std::vector<double> val_v;
        const int *rptr = A->row_ptr, *cidx = A->col_idx;      // host inputs are read in place (they are only read)
        const double *val = A->val;
        if (A->where != CS_HOST) {
            if ((st = fetch(S, rptr_v, A->row_ptr, (size_t)m + 1, A->where)) != CS_OK) return st;
            if ((st = fetch(S, cidx_v, A->col_idx, (size_t)nnz, A->where)) != CS_OK) return st;
            if ((st = fetch(S, val_v, A->val, (size_t)nnz, A->where)) != CS_OK) return st;
            rptr = rptr_v.data(); cidx = cidx_v.data(); val = val_v.data();
        }
        if ((st = fetch(S, hb, b, (size_t)m, vec_where)) != CS_OK) return st;
        if ((st = fetch(S, hc, c, (size_t)n, vec_where)) != CS_OK) return st;
        if (rptr[0] != 0 || rptr[m] != nnz) { S->err = "row_ptr[0] != 0 or row_ptr[m] != nnz"; return CS_EINVAL; }
        for (int i = 0; i < m; ++i) {
            if (rptr[i + 1] <= rptr[i]) { S->err = "row_ptr not increasing (empty rows are not allowed)"; return CS_EINVAL; }
            if (rptr[i + 1] > nnz) { S->err = "row_ptr out of range"; return CS_EINVAL; }
        }
        {
            std::atomic<int> bad{0};
            const int blk = 16384;
            parallel_blocks((m + blk - 1) / blk, host_threads(), [&](int bi) {
                for (int i = bi * blk; i < std::min(m, (bi + 1) * blk); ++i) {
                    double ss = 0.0;
                    for (int k = rptr[i]; k < rptr[i + 1]; ++k) {
                        if (cidx[k] < 0 || cidx[k] >= n || (k > rptr[i] && cidx[k] <= cidx[k - 1])) bad.store(1);
                        else if (!std::isfinite(val[k])) bad.store(2);
                        ss += val[k] * val[k];
                    }
                    if (!(ss > 0.0) && !bad.load()) bad.store(3);       // a row of stored zeros: A is not of full row rank
                }
            });
            if (bad.load() == 1) { S->err = "col_idx out of range, unsorted or duplicated within a row"; return CS_EINVAL; }
            if (bad.load() == 2) { S->err = "non-finite matrix entry"; return CS_EINVAL; }
            if (bad.load() == 3) { S->err = "a row of A has zero norm (all stored entries are 0 or underflow when squared)"; return CS_EINVAL; }
        }
        nb = 0.0; nc = 0.0;
        for (int i = 0; i < m; ++i) { if (!std::isfinite(hb[i])) { S->err = "non-finite b"; return CS_EINVAL; } nb += hb[i] * hb[i]; }
        for (int j = 0; j < n; ++j) { if (!std::isfinite(hc[j])) { S->err = "non-finite c"; return CS_EINVAL; } nc += hc[j] * hc[j]; }
        lap("fetch + validate");
        // ---- internal ordering: rows sorted by decreasing length, orthant columns likewise (Lorentz blocks
        //      keep their place so that cones stay contiguous).  perm[internal] = caller's index.
        std::vector<int> rlen((size_t)m), clen((size_t)n, 0);
        for (int i = 0; i < m; ++i) rlen[i] = rptr[i + 1] - rptr[i];
        {
            const int blk = 1 << 20;
            parallel_blocks((nnz + blk - 1) / blk, host_threads(), [&](int bi) {
                for (int k = bi * blk; k < std::min(nnz, (bi + 1) * blk); ++k) __atomic_fetch_add(&clen[cidx[k]], 1, __ATOMIC_RELAXED);
            });
        }
        perm_r = order_by_length(rlen, m);
        for (int i = 0; i < m && rlen[perm_r[i]] > kShortMax; ++i) S->ctx.n_long = i + 1;
        // (A lexicographic ordering of the columns by the heavy rows they touch was tried so that those rows'
        //  gathers run over contiguous stretches; it cost 3.4 s at config 4 and changed nothing measurable.)
        perm_c = order_by_length(clen, (int)K->n_lin);
        std::vector<int> inv_c((size_t)n);
        for (int j = 0; j < n; ++j) inv_c[perm_c[j]] = j;
        lap("row/column ordering");
        // row-major copy in internal numbering (entries of a row sorted by internal column)
        std::vector<int> rp2((size_t)m + 1, 0);
        uvec<int> ci2((size_t)nnz);
        uvec<double> va2((size_t)nnz);
        for (int i = 0; i < m; ++i) rp2[(size_t)i + 1] = rp2[i] + rlen[perm_r[i]];
        {
            auto fill_rows = [&](int i0, int i1) {
                std::vector<std::pair<int, double>> tmp;
                for (int i = i0; i < i1; ++i) {
                    const int src = perm_r[i], a0 = rptr[src], len = rlen[src], dst = rp2[i];
                    if (len <= kShortMax) {     // order inside a short row is irrelevant
                        for (int k = 0; k < len; ++k) { ci2[dst + k] = inv_c[cidx[a0 + k]]; va2[dst + k] = val[a0 + k]; }
                        continue;
                    }
                    if (len > n / 16) {         // nearly dense row: bucket by internal column instead of sorting (O(n))
                        std::vector<double> dense((size_t)n, 0.0);
                        std::vector<unsigned char> mark((size_t)n, 0);
                        for (int k = 0; k < len; ++k) { const int j = inv_c[cidx[a0 + k]]; dense[j] = val[a0 + k]; mark[j] = 1; }
                        int q = dst;
                        for (int j = 0; j < n; ++j) if (mark[j]) { ci2[q] = j; va2[q] = dense[j]; ++q; }
                        continue;
                    }
                    tmp.resize(len);            // long rows: ascending internal column, so their gathers stay as local as they were
                    for (int k = 0; k < len; ++k) tmp[k] = {inv_c[cidx[a0 + k]], val[a0 + k]};
                    std::sort(tmp.begin(), tmp.end(), [](const std::pair<int, double> &u, const std::pair<int, double> &v) { return u.first < v.first; });
                    for (int k = 0; k < len; ++k) { ci2[dst + k] = tmp[k].first; va2[dst + k] = tmp[k].second; }
                }
            };
            // blocks of rows with at most ~256k entries (the heavy rows come first and get blocks of their own)
            std::vector<int> cut{0};
            for (int i = 0, acc = 0; i < m; ++i) {
                acc += rlen[perm_r[i]];
                if (acc >= (1 << 18) || i + 1 == m) { cut.push_back(i + 1); acc = 0; }
            }
            parallel_blocks((int)cut.size() - 1, host_threads(), [&](int bi) { fill_rows(cut[bi], cut[bi + 1]); });
        }
        lap("row-major copy");
        // column-major copy (counting sort by internal column; rows come out sorted within a column)
        HostSparse hr, hc2;
        std::vector<int> cp2((size_t)n + 1, 0);
        uvec<int> ri2((size_t)nnz);
        const int nt = host_threads();
        {
            uvec<double> cv2((size_t)nnz);
            for (int j = 0; j < n; ++j) cp2[(size_t)j + 1] = cp2[j] + clen[perm_c[j]];   // internal column j = caller's perm_c[j]
            std::vector<int> fill(cp2.begin(), cp2.end() - 1);
            // every helper scans all entries in row order but places only those of its own column range:
            // sequential reads, writes confined to the range, order within a column = row order (deterministic)
            const int parts = std::max(1, nt);
            parallel_blocks(parts, parts, [&](int part) {
                const int j0 = (int)((long long)n * part / parts), j1 = (int)((long long)n * (part + 1) / parts);
                for (int i = 0; i < m; ++i)
                    for (int k = rp2[i]; k < rp2[i + 1]; ++k) {
                        const int j = ci2[k];
                        if (j < j0 || j >= j1) continue;
                        const int q = fill[j]++;
                        ri2[q] = i;
                        cv2[q] = va2[k];
                    }
            });
            lap("column-major copy");
            // Heavy-row fusion plan: the longest rows (internal rows come sorted by decreasing length), if they are long
            // enough to be worth it and the problem runs on more than one CTA.
            FusePlan fuse;
            if (nnz > kOneCtaNnz)
                for (int i = 0; i < std::min(m, kFuseA + kFuseB) && rp2[(size_t)i + 1] - rp2[i] >= kFuseMinLen; ++i)
                    (i < kFuseA ? fuse.n_fa : fuse.n_fb) += 1;
            uvec<unsigned char> fused;
            if (fuse.rows()) {
                fused.resize((size_t)nnz);
                std::memset(fused.data(), 0, (size_t)nnz);
            }
            hc2 = make_sparse(cp2, ri2, cv2, nt, fuse.rows() ? &fuse : nullptr, fuse.rows() ? &fused : nullptr);
            lap("column-major slices");
            // fused rows: entries that stay with the row pass first, the fused ones after them (each part keeps its
            // ascending column order); split[s] = size of the first part.  The rows are rebuilt from the column-major copy
            // by two sequential scans over the columns (count, then place): the fused rows are the first entries of a
            // column (rows ascend), so a column is left as soon as a row >= fuse.rows() shows up -- no searching.
            std::vector<int> split((size_t)fuse.rows());
            if (fuse.rows() && !hc2.too_big) {
                const int nf = fuse.rows(), cblk = 1 << 16, nblk = (n + cblk - 1) / cblk;
                std::vector<int> cnt((size_t)nblk * nf * 2, 0);      // [block][row][unfused, fused]
                parallel_blocks(nblk, nt, [&](int bi) {
                    int *c = cnt.data() + (size_t)bi * nf * 2;
                    for (int j = bi * cblk; j < std::min(n, (bi + 1) * cblk); ++j)
                        for (int e = cp2[j]; e < cp2[(size_t)j + 1] && ri2[e] < nf; ++e) c[2 * ri2[e] + fused[e]] += 1;
                });
                std::vector<int> off((size_t)nblk * nf * 2);
                for (int r = 0; r < nf; ++r) {
                    int u = rp2[r];
                    for (int bi = 0; bi < nblk; ++bi) { off[((size_t)bi * nf + r) * 2] = u; u += cnt[((size_t)bi * nf + r) * 2]; }
                    split[r] = u - rp2[r];
                    for (int bi = 0; bi < nblk; ++bi) { off[((size_t)bi * nf + r) * 2 + 1] = u; u += cnt[((size_t)bi * nf + r) * 2 + 1]; }
                }
                parallel_blocks(nblk, nt, [&](int bi) {
                    int *o = off.data() + (size_t)bi * nf * 2;
                    for (int j = bi * cblk; j < std::min(n, (bi + 1) * cblk); ++j)
                        for (int e = cp2[j]; e < cp2[(size_t)j + 1] && ri2[e] < nf; ++e) {
                            const int q = o[2 * ri2[e] + fused[e]]++;
                            ci2[q] = j;
                            va2[q] = cv2[e];
                        }
                });
                S->ctx.n_fa = fuse.n_fa;
                S->ctx.n_fb = fuse.n_fb;
                lap("fused rows: partition");
            }
            hr = make_sparse(rp2, ci2, va2, nt, nullptr, nullptr, fuse.rows() ? &split : nullptr);
        }
        lap("row-major slices");
        if (hr.too_big || hc2.too_big) {
            S->err = "padded slice storage exceeds 2^31 entries";
            return CS_EINVAL;
        }
        {
            int *q;
            if ((st = upload_sparse(S, hr, &S->ctx.R)) != CS_OK) return st;
            if ((st = dev_upload(S, &q, rp2.data(), rp2.size())) != CS_OK) return st; S->ctx.Rc.ptr = q;
            if ((st = dev_upload(S, &q, ci2.data(), ci2.size())) != CS_OK) return st; S->ctx.Rc.idx = q;
            if ((st = dev_upload(S, &q, hr.pos.data(), hr.pos.size())) != CS_OK) return st; S->ctx.Rc.pos = q;
        }
        {   // b, c in internal order
            std::vector<double> t((size_t)std::max(m, n));
            for (int i = 0; i < m; ++i) t[i] = hb[perm_r[i]];
            std::copy(t.begin(), t.begin() + m, hb.begin());
            for (int j = 0; j < n; ++j) t[j] = hc[perm_c[j]];
            std::copy(t.begin(), t.begin() + n, hc.begin());
        }
        {   // the column-major copy and the plain compressed views of the same entries (the FSAI build and the dense path walk them)
            int *q;
            if ((st = upload_sparse(S, hc2, &S->ctx.C)) != CS_OK) return st;
            if ((st = dev_upload(S, &q, cp2.data(), cp2.size())) != CS_OK) return st; S->ctx.Cc.ptr = q;
            if ((st = dev_upload(S, &q, ri2.data(), ri2.size())) != CS_OK) return st; S->ctx.Cc.idx = q;
            if ((st = dev_upload(S, &q, hc2.pos.data(), hc2.pos.size())) != CS_OK) return st; S->ctx.Cc.pos = q;
            CS_CUDA(S, cudaStreamSynchronize(S->stream));   // the host images die at the end of this block
        }
    }
    // ---- device state
    Ctx &x = S->ctx;
    x.m = m; x.n = n; x.n_lin = (int)K->n_lin; x.n_soc = (int)K->n_soc;
    x.norm_b = std::sqrt(nb); x.norm_c = std::sqrt(nc);
    int *ip; double *dp;
    if ((st = dev_upload(S, &ip, cone_off.data(), cone_off.size())) != CS_OK) return st; x.cone_off = ip;
    {   // Lorentz blocks by size class (cone_sweep, cs_kernels.cuh): small (sub-warp), medium (warp), large (CTA)
        std::vector<int> cls[3];
        for (int i = 0; i < (int)K->n_soc; ++i) cls[K->soc_size[i] <= kConeSmall ? 0 : K->soc_size[i] <= kConeMedium ? 1 : 2].push_back(i);
        x.n_cone_small = (int)cls[0].size(); x.n_cone_medium = (int)cls[1].size(); x.n_cone_large = (int)cls[2].size();
        cls[0].insert(cls[0].end(), cls[1].begin(), cls[1].end());
        cls[0].insert(cls[0].end(), cls[2].begin(), cls[2].end());
        if ((st = dev_upload(S, &ip, cls[0].data(), cls[0].size())) != CS_OK) return st; x.cone_cls = ip;
        CS_CUDA(S, cudaStreamSynchronize(S->stream));   // the staging vectors die here
    }
    if (!x.perm_r) {   // (the device build has made them on the device)
        if ((st = dev_upload(S, &ip, perm_r.data(), perm_r.size())) != CS_OK) return st; x.perm_r = ip;
        if ((st = dev_upload(S, &ip, perm_c.data(), perm_c.size())) != CS_OK) return st; x.perm_c = ip;
    }
    if ((st = dev_zeros(S, &x.fpart, (size_t)(x.n_fa + x.n_fb) * kMaxGrid)) != CS_OK) return st;
    x.R.fpart = x.fpart;
    {   // scratch of the FSAI builds
        if ((st = dev_zeros(S, &x.f_ctop, (size_t)3 * n)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.f_partner, (size_t)m)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.f_tptr, (size_t)m + 1)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.f_tcur, (size_t)m)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.f_tidx, (size_t)m)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.f_blk, (size_t)kMaxGrid)) != CS_OK) return st;
        double **fv[] = {&x.f_gd, &x.f_gm, &x.f_tc, &x.z, &x.t1};
        for (double **q2 : fv) if ((st = dev_zeros(S, q2, (size_t)m)) != CS_OK) return st;
    }
    CS_CUDA(S, cudaStreamSynchronize(S->stream));
    lap("upload");
    if (!x.b) {   // (the device build has already permuted b, c on the device)
        if ((st = dev_upload(S, &dp, hb.data(), hb.size())) != CS_OK) return st; x.b = dp;
        if ((st = dev_upload(S, &dp, hc.data(), hc.size())) != CS_OK) return st; x.c = dp;
    }
    double **nv[] = {&x.s, &x.p, &x.g, &x.e, &x.u, &x.chat};
    for (double **q : nv) if ((st = dev_zeros(S, q, (size_t)n)) != CS_OK) return st;
    double **mv[] = {&x.w, &x.r, &x.v, &x.btil};
    for (double **q : mv) if ((st = dev_zeros(S, q, (size_t)m)) != CS_OK) return st;
    {   // O = 1, D = 1, x = z = e_K
        if ((st = dev_alloc(S, &x.O, (size_t)n)) != CS_OK) return st;
        if ((st = dev_alloc(S, &x.D, (size_t)m)) != CS_OK) return st;
        if ((st = dev_alloc(S, &x.xb, (size_t)n)) != CS_OK) return st;
        if ((st = dev_alloc(S, &x.zb, (size_t)n)) != CS_OK) return st;
        csb::k_fill<<<ew_blocks(n), 256, 0, S->stream>>>(x.O, n, 1.0);
        csb::k_fill<<<ew_blocks(m), 256, 0, S->stream>>>(x.D, m, 1.0);
        csb::k_unit_cone_point<<<ew_blocks(n), 256, 0, S->stream>>>(x.xb, x.zb, n, x.n_lin, x.cone_off, x.n_soc);
        if (x.n_soc) csb::k_unit_cone_heads<<<ew_blocks(x.n_soc), 256, 0, S->stream>>>(x.xb, x.zb, x.cone_off, x.n_soc);
        CS_CUDA(S, cudaGetLastError());
        S->launches += 4;
    }
    if ((st = dev_zeros(S, &x.sc, 1)) != CS_OK) return st;
    if ((st = dev_zeros(S, &x.partial_probe, 1)) != CS_OK) return st;
    lap("vectors");
    // ---- cooperative grid: as many CTAs as can be co-resident (k_iterate carries the fusion accumulators in dynamic
    //      shared memory when some rows are fused)
    int sms = 0, occ = 0, occ_min = 1 << 30;
    CS_CUDA(S, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, S->device));
    const void *kernels[] = {(const void *)k_iterate, (const void *)k_iterate_dense, (const void *)k_condition, (const void *)k_residuals,
                             (const void *)k_equilibrate, (const void *)k_barrier_probe};
    S->dyn_smem = x.n_fa + x.n_fb > 0 ? (size_t)kFuseSmem : 0;
    for (const void *k : kernels) {
        const size_t dyn = k == (const void *)k_iterate || k == (const void *)k_iterate_dense ? S->dyn_smem : 0;
        if (dyn) {
            CS_CUDA(S, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
            // < 96 KB: ask for the 100 KB carve-out, so that the gathers keep ~128 KB of L1 (they collapse below ~90 KB,
            // DESIGN.md 8); left to itself the driver picked 132 KB for 2 x 49 KB in an earlier build
            CS_CUDA(S, cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, kFuseCarveoutPct));
        }
        CS_CUDA(S, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, kBlock, dyn));
        occ_min = std::min(occ_min, occ);
    }
    if (occ_min < 1) { S->err = "kernel does not fit on an SM"; return CS_ECUDA; }
    S->grid = std::min(sms * occ_min, kMaxGrid);
    if (verbose) fprintf(stderr, "cs_create: %d SMs x %d CTAs of %d threads, %zu B dynamic shared memory in k_iterate, fused rows %d + %d\n",
                         sms, occ_min, kBlock, S->dyn_smem, x.n_fa, x.n_fb);
    if (nnz <= kOneCtaNnz) S->grid = 1;   // tiny problem (config 0): one CTA, barriers are __syncthreads (cs_device.cuh)
    if (S->grid == 1 && m <= kDenseMax) {   // scratch of the dense factor-apply path (cs_params.dense_m_threshold)
        if ((st = dev_zeros(S, &x.dM, (size_t)m * m)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.dMd, (size_t)m)) != CS_OK) return st;
        if ((st = dev_zeros(S, &x.dv, (size_t)2 * m)) != CS_OK) return st;
    }
    // grid dense path (cs_dense.cuh): only for a dense-stored A (at least half of the m x n entries present) on many CTAs
    S->dense_capable = S->grid > 1 && m <= kDenseGridMax && (double)nnz >= 0.5 * (double)m * (double)n;
    if ((st = dev_zeros(S, &x.bar, 1)) != CS_OK) return st;
    if ((st = dev_zeros(S, &x.partials, (size_t)2 * kMaxRed * kMaxGrid)) != CS_OK) return st;
    // ---- defaults (cs.h)
    S->prm.mu = 1.0;
    S->prm.t = K->n_soc > 0 ? 1.7 : 9.2;
    S->prm.o_floor = 1e-16;
    S->prm.cg_tol = 2.220446049250313e-16;   // DBL_EPSILON: the recurrence residual below one ulp of the right-hand side (cs.h)
    S->prm.cg_reduce = 0.0;
    S->prm.cg_max_iter = 20000;
    S->prm.precond = 0;
    S->prm.dense_m_threshold = S->dense_capable ? kDenseGridMax : 128;   // dense-stored input: the dense path is the default (cs.h)
    S->prm.reserved = 0;
    S->nnz = nnz;
    x.mu = S->prm.mu; x.t = S->prm.t; x.o_floor = S->prm.o_floor;
    sync_params(S);
    CS_CUDA(S, cudaStreamSynchronize(S->stream));
    lap("grid + parameters");
    return CS_OK;
}

static cs_status create_common(cs_solver **out, const cs_csr *A, const double *b, const double *c, cs_mem vec_where,
                               const cs_cones *K, void *cuda_stream, int build_mode) {
    if (!out) return CS_EINVAL;
    *out = nullptr;
    if (!A || !b || !c || !K || !A->row_ptr || !A->col_idx || !A->val) { g_create_err = "NULL argument"; return CS_EINVAL; }
    cs_solver *S = new (std::nothrow) cs_solver;
    if (!S) return CS_ENOMEM;
    S->stream = static_cast<cudaStream_t>(cuda_stream);
    S->build_mode = build_mode;
    cs_status st = CS_OK;
    if (cudaGetDevice(&S->device) != cudaSuccess) { S->err = "no CUDA device"; st = CS_ECUDA; }
    if (st == CS_OK) {
        try { st = create_impl(S, A, b, c, vec_where, K); }
        catch (const std::bad_alloc &) { S->err = "host allocation failed"; st = CS_ENOMEM; }
    }
    if (st != CS_OK) { g_create_err = S->err; cs_destroy(S); return st; }
    *out = S;
    return CS_OK;
}

cs_status cs_create(cs_solver **out, const cs_csr *A, const double *b, const double *c, cs_mem vec_where,
                    const cs_cones *K, void *cuda_stream) {
    return create_common(out, A, b, c, vec_where, K, cuda_stream, 0);
}

cs_status cs_diag_create(cs_solver **out, const cs_csr *A, const double *b, const double *c, cs_mem vec_where,
                         const cs_cones *K, void *cuda_stream, int32_t build_mode) {
    if (build_mode < 0 || build_mode > 2) return CS_EINVAL;
    return create_common(out, A, b, c, vec_where, K, cuda_stream, build_mode);
}

cs_status cs_diag_layout_digest(cs_solver *S, uint64_t out[32]) {
    if (!S || !out) return CS_EINVAL;
    DeviceGuard guard(S);
    const Ctx &c = S->ctx;
    std::vector<unsigned char> h;
    int k = 0;
    auto digest = [&](const void *dev, size_t bytes) -> cs_status {       // FNV-1a over a device array
        h.resize(bytes);
        if (bytes) CS_CUDA(S, cudaMemcpy(h.data(), dev, bytes, cudaMemcpyDeviceToHost));
        uint64_t f = 1469598103934665603ull;
        for (size_t i = 0; i < bytes; ++i) { f ^= h[i]; f *= 1099511628211ull; }
        out[k++] = f;
        return CS_OK;
    };
    CS_CUDA(S, cudaStreamSynchronize(S->stream));
    cs_status st;
    const Sparse *sp[2] = {&c.R, &c.C};
    const Csr *cv[2] = {&c.Rc, &c.Cc};
    const size_t tot[2] = {S->tot_r, S->tot_c};
    const int nseg[2] = {c.m, c.n};
    for (int q = 0; q < 2; ++q) {
        if ((st = digest(sp[q]->slices, sizeof(int4) * (size_t)sp[q]->n_slice)) != CS_OK) return st;
        if ((st = digest(sp[q]->idx, sizeof(int) * tot[q])) != CS_OK) return st;
        if ((st = digest(sp[q]->val0, sizeof(double) * tot[q])) != CS_OK) return st;
        if ((st = digest(sp[q]->chunk_slot, sizeof(int) * (size_t)sp[q]->n_chunk)) != CS_OK) return st;
        if ((st = digest(sp[q]->multi, sizeof(int4) * (size_t)sp[q]->n_multi)) != CS_OK) return st;
        if ((st = digest(sp[q]->multi_k2, sizeof(int4) * (size_t)sp[q]->n_multi_k2)) != CS_OK) return st;
        if ((st = digest(cv[q]->ptr, sizeof(int) * ((size_t)nseg[q] + 1))) != CS_OK) return st;
        if ((st = digest(cv[q]->idx, sizeof(int) * (size_t)S->nnz)) != CS_OK) return st;
        if ((st = digest(cv[q]->pos, sizeof(int) * (size_t)S->nnz)) != CS_OK) return st;
    }
    if ((st = digest(c.C.fmask, c.n_fa + c.n_fb ? (size_t)(c.C.n_slice - c.C.n_chunk) * 32 : 0)) != CS_OK) return st;
    if ((st = digest(c.perm_r, sizeof(int) * (size_t)c.m)) != CS_OK) return st;
    if ((st = digest(c.perm_c, sizeof(int) * (size_t)c.n)) != CS_OK) return st;
    if ((st = digest(c.b, sizeof(double) * (size_t)c.m)) != CS_OK) return st;
    if ((st = digest(c.c, sizeof(double) * (size_t)c.n)) != CS_OK) return st;
    out[k++] = ((uint64_t)(unsigned)c.R.n_chunk_k2 << 32) | (unsigned)c.R.n_chunk;
    out[k++] = ((uint64_t)(unsigned)c.n_fa << 40) | ((uint64_t)(unsigned)c.n_fb << 20) | (unsigned)c.n_long;
    while (k < 32) out[k++] = 0;
    return CS_OK;
}

cs_status cs_set_params(cs_solver *S, const cs_params *p) {
    if (!S || !p) return CS_EINVAL;
    if (!(p->mu > 0.0) || !(p->t > 0.0) || !(p->o_floor > 0.0) || !(p->cg_tol >= 0.0) || !(p->cg_reduce >= 0.0 && p->cg_reduce < 1.0) || p->cg_max_iter < 1 ||
        p->precond < 0 || p->precond > 3 || p->dense_m_threshold < 0 || p->dense_m_threshold > kDenseGridMax) {
        S->err = "mu, t, o_floor must be > 0, cg_tol >= 0, 0 <= cg_reduce < 1, cg_max_iter >= 1, precond in {0,1,2,3}, dense_m_threshold in [0,24576]";
        return CS_EINVAL;
    }
    S->prm = *p;
    sync_params(S);
    return CS_OK;
}

cs_status cs_get_params(const cs_solver *S, cs_params *p) {
    if (!S || !p) return CS_EINVAL;
    *p = S->prm;
    return CS_OK;
}

cs_status cs_set_point(cs_solver *S, const double *x, const double *z, cs_mem where) {
    if (!S || !x || !z) return CS_EINVAL;
    DeviceGuard guard(S);
    if (S->started) { S->err = "cs_set_point after the iteration has started"; return CS_ESTATE; }
    cs_status st;
    if ((st = import_cols(S, S->ctx.xb, x, where)) != CS_OK) return st;
    return import_cols(S, S->ctx.zb, z, where);
}

cs_status cs_set_dual(cs_solver *S, const double *y, cs_mem where) {
    if (!S || !y) return CS_EINVAL;
    DeviceGuard guard(S);
    if (S->started) { S->err = "cs_set_dual after the iteration has started"; return CS_ESTATE; }
    const Ctx &c = S->ctx;
    const double *dy = y;
    if (where == CS_HOST) {                                      // r is scratch until the first pass
        CS_CUDA(S, cudaMemcpyAsync(c.r, y, sizeof(double) * c.m, cudaMemcpyHostToDevice, S->stream));
        dy = c.r;
    }
    k_w_from_y<<<ew_blocks(c.m), 256, 0, S->stream>>>(c, dy, S->prm.mu);
    CS_CUDA(S, cudaGetLastError());
    S->launches += 1;
    if (where == CS_HOST) CS_CUDA(S, cudaStreamSynchronize(S->stream));   // the caller's buffer is free on return
    return CS_OK;
}

cs_status cs_condition(cs_solver *S) {
    if (!S) return CS_EINVAL;
    DeviceGuard guard(S);
    return do_condition(S, 1);
}

cs_status cs_set_scaling(cs_solver *S, const double *O, cs_mem where) {
    if (!S || !O) return CS_EINVAL;
    DeviceGuard guard(S);
    cs_status st = ensure_xz(S);  // x,z of the OLD scaling, before O is overwritten
    if (st != CS_OK) return st;
    if ((st = import_cols(S, S->ctx.O, O, where)) != CS_OK) return st;
    return do_condition(S, 0);
}

cs_status cs_iterate(cs_solver *S, int64_t k) {
    if (!S || k < 0) return CS_EINVAL;
    DeviceGuard guard(S);
    if (k == 0) return CS_OK;
    cs_status st;
    if (!S->conditioned && (st = do_condition(S, 1)) != CS_OK) return st;  // step 4: l = 1
    sync_params(S);
    long long kk = k;
    void *args[] = {&S->ctx, &kk};
    if ((st = launch_coop(S, S->ctx.dense ? (const void *)k_iterate_dense : (const void *)k_iterate, args)) != CS_OK) return st;
    S->xz_stale = true;
    S->started = true;
    S->iter += k;
    return CS_OK;
}

cs_status cs_residuals(cs_solver *S, cs_resid *out) {
    if (!S || !out) return CS_EINVAL;
    DeviceGuard guard(S);
    cs_status st;
    if (!S->conditioned && (st = do_condition(S, 1)) != CS_OK) return st;
    if ((st = ensure_xz(S)) != CS_OK) return st;
    void *args[] = {&S->ctx};
    if ((st = launch_coop(S, (const void *)k_residuals, args)) != CS_OK) return st;
    Scalars h;
    CS_CUDA(S, cudaMemcpyAsync(&h, S->ctx.sc, sizeof(h), cudaMemcpyDeviceToHost, S->stream));
    CS_CUDA(S, cudaMemsetAsync(&S->ctx.sc->cg_hit_max, 0, sizeof(int), S->stream));
    CS_CUDA(S, cudaStreamSynchronize(S->stream));
    out->iter = h.iter; out->cg_steps_total = h.cg_steps_total; out->cg_steps_cond = h.cg_steps_cond; out->cg_steps_last = h.cg_steps_last;
    out->n_conditionings = h.n_cond; out->cg_hit_max = h.cg_hit_max; out->dense_refine2 = h.dense_refine2;
    out->pres_abs = h.resid[0]; out->pres_rel = h.resid[1]; out->dres_abs = h.resid[2]; out->dres_rel = h.resid[3];
    out->gap_abs = h.resid[4]; out->gap_rel = h.resid[5]; out->cone_viol_rel = h.resid[6]; out->kkt_rel = h.resid[7];
    out->pobj = h.resid[8]; out->dobj = h.resid[9]; out->fp_res = h.resid[10];
    if (!std::isfinite(out->kkt_rel)) {
        S->err = "non-finite KKT residual: the iteration has diverged or a scaling over/underflowed (t too large for this data?)";
        return CS_ESTATE;
    }
    return h.cg_hit_max ? CS_ECGMAX : CS_OK;
}

cs_status cs_equilibrate(cs_solver *S, int32_t n_sweeps) {
    if (!S || n_sweeps < 0) return CS_EINVAL;
    DeviceGuard guard(S);
    cs_status st = ensure_xz(S);  // x,z of the OLD scaling, before O is overwritten
    if (st != CS_OK) return st;
    int ns = n_sweeps;
    void *args[] = {&S->ctx, &ns};
    if ((st = launch_coop(S, (const void *)k_equilibrate, args)) != CS_OK) return st;
    return do_condition(S, 0);
}

namespace {
cs_status fetch_fp_res(cs_solver *S, double *f) {
    double f2 = 0.0;
    CS_CUDA(S, cudaMemcpyAsync(&f2, &S->ctx.sc->fp_res2, sizeof(double), cudaMemcpyDeviceToHost, S->stream));
    CS_CUDA(S, cudaStreamSynchronize(S->stream));
    *f = std::sqrt(f2);
    return CS_OK;
}
int64_t next_multiple(int64_t l, int64_t q) { return (l / q + 1) * q; }   // smallest multiple of q above l
}  // namespace

cs_status cs_solve(cs_solver *S, const cs_schedule *sch, cs_resid *out, int64_t *cond_iters, int64_t cond_cap,
                   int64_t *n_cond) {
    if (!S || !sch || !out || sch->max_iter < 0 || sch->check_every < 0 || cond_cap < 0) return CS_EINVAL;
    DeviceGuard guard(S);
    const bool stall = sch->rule == CS_RULE_STALL;
    if (sch->rule != CS_RULE_SET && !stall) { S->err = "cs_solve: unknown rule"; return CS_EINVAL; }
    if (stall && (sch->window < 2 || sch->lag < 1 || sch->lag >= sch->window || !(sch->ratio >= 0.0))) {
        S->err = "cs_solve: the stall rule needs window >= 2, 1 <= lag < window, ratio >= 0";
        return CS_EINVAL;
    }
    const int64_t kInf = INT64_MAX / 2;
    const int64_t start = S->iter, end = start + sch->max_iter;
    int64_t nc = 0;
    auto note = [&](int64_t l) { if (cond_iters && nc < cond_cap) cond_iters[nc] = l; ++nc; };
    auto in_L = [&](int64_t l) {   // CS_RULE_SET membership
        if (sch->first <= 0 || l < sch->first) return false;
        return l == sch->first || (sch->every > 0 && (l - sch->first) % sch->every == 0);
    };
    cs_status st, sticky = CS_OK;
    bool have_resid = false;
    if (!S->conditioned && S->iter == 0 && sch->max_iter > 0) note(1);   // cs_iterate runs the l = 1 conditioning
    while (true) {
        const int64_t l = S->iter;   // passes done; the next iteration is l + 1
        have_resid = false;
        if (sch->check_every > 0 && l > start && l % sch->check_every == 0 && sch->tol > 0.0) {
            st = cs_residuals(S, out);
            if (st == CS_ECGMAX) sticky = st; else if (st != CS_OK) return st;
            have_resid = true;
            if (out->kkt_rel <= sch->tol) break;
        }
        if (l >= end) break;
        if (stall && l > 0) {
            if ((l + sch->lag) % sch->window == 0) {
                if ((st = fetch_fp_res(S, &S->stall_f)) != CS_OK) return st;
                S->stall_at = l;
            }
            if (l % sch->window == 0 && S->stall_at == l - sch->lag) {
                double f_now;
                if ((st = fetch_fp_res(S, &f_now)) != CS_OK) return st;
                if (f_now > sch->ratio * S->stall_f && f_now > sch->f_floor) {
                    if ((st = do_condition(S, 1)) != CS_OK) return st;
                    note(l + 1);
                }
            }
        } else if (!stall && l > 0 && in_L(l + 1)) {
            if ((st = do_condition(S, 1)) != CS_OK) return st;
            note(l + 1);
        }
        int64_t nxt = end;
        if (sch->check_every > 0 && sch->tol > 0.0) nxt = std::min(nxt, next_multiple(l, sch->check_every));
        if (stall) {
            nxt = std::min(nxt, next_multiple(l, sch->window));
            nxt = std::min(nxt, next_multiple(l + sch->lag, sch->window) - sch->lag);
        } else if (sch->first > 0) {
            int64_t c = kInf;   // smallest member of L above l + 1
            if (l + 1 < sch->first) c = sch->first;
            else if (sch->every > 0) c = sch->first + ((l + 1 - sch->first) / sch->every + 1) * sch->every;
            nxt = std::min(nxt, c - 1);
        }
        if ((st = cs_iterate(S, nxt - l)) != CS_OK) return st;
    }
    if (!have_resid) {
        st = cs_residuals(S, out);
        if (st == CS_ECGMAX) sticky = st; else if (st != CS_OK) return st;
    }
    if (n_cond) *n_cond = nc;
    return sticky;
}

cs_status cs_diag_phase_times(cs_solver *S, double out[8]) {
    if (!S || !out) return CS_EINVAL;
    DeviceGuard guard(S);
    Scalars h;
    CS_CUDA(S, cudaMemcpyAsync(&h, S->ctx.sc, sizeof(h), cudaMemcpyDeviceToHost, S->stream));
    CS_CUDA(S, cudaStreamSynchronize(S->stream));
    for (int i = 0; i < 8; ++i) out[i] = (double)h.phase_ns[i];
    return CS_OK;
}

cs_status cs_diag_gather_probe(int64_t n_vec, int64_t n_idx, double *us_gather, double *us_stream_only) {
    if (n_vec < 1 || n_idx < 1 || n_vec >= INT32_MAX || n_idx >= INT32_MAX || !us_gather || !us_stream_only) return CS_EINVAL;
    int *idx = nullptr; double *x = nullptr, *out = nullptr;
    int sms = 0, dev = 0;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cs_status st = CS_ECUDA;
    do {
        if (cudaGetDevice(&dev) != cudaSuccess) break;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) break;
        const int grid = sms * 2;
        if (cudaMalloc(&idx, sizeof(int) * n_idx) != cudaSuccess || cudaMalloc(&x, sizeof(double) * n_vec) != cudaSuccess ||
            cudaMalloc(&out, sizeof(double) * (size_t)grid * kBlock) != cudaSuccess) { st = CS_ENOMEM; break; }
        if (cudaMemset(x, 0, sizeof(double) * n_vec) != cudaSuccess) break;
        k_probe_indices<<<sms * 8, 256>>>(idx, (int)n_idx, (int)n_vec);
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) break;
        double us[2] = {0.0, 0.0};
        bool ok = true;
        for (int mode = 0; mode < 2 && ok; ++mode)
            for (int rep = 0; rep < 3 && ok; ++rep) {           // keep the last of three
                cudaEventRecord(e0);
                k_gather_probe<<<grid, kBlock>>>(idx, x, out, (int)n_idx, 1 - mode);
                cudaEventRecord(e1);
                float ms = 0.f;
                ok = cudaEventSynchronize(e1) == cudaSuccess && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess;
                us[mode] = 1e3 * ms;
            }
        if (!ok) break;
        *us_gather = us[0];
        *us_stream_only = us[1];
        st = CS_OK;
    } while (false);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(idx); cudaFree(x); cudaFree(out);
    return st;
}

cs_status cs_diag_l2_probe(int64_t bytes, int32_t reps, double *gbs) {
    if (bytes < 4096 || bytes > ((int64_t)1 << 32) || reps < 1 || !gbs) return CS_EINVAL;
    double2 *buf = nullptr; double *out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cs_status st = CS_ECUDA;
    int sms = 0, dev = 0;
    do {
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) break;
        const long long n16 = bytes / 16;
        if (cudaMalloc(&buf, (size_t)n16 * 16) != cudaSuccess || cudaMalloc(&out, 8) != cudaSuccess) { st = CS_ENOMEM; break; }
        if (cudaMemset(buf, 0, (size_t)n16 * 16) != cudaSuccess) break;
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) break;
        double best = 0.0;
        bool ok = true;
        for (int rep = 0; rep < 4 && ok; ++rep) {                // the first launch also warms L2; keep the best
            cudaEventRecord(e0);
            k_l2_probe<<<sms * 4, 512>>>(buf, n16, reps, out);
            cudaEventRecord(e1);
            float ms = 0.f;
            ok = cudaEventSynchronize(e1) == cudaSuccess && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess;
            if (ok && ms > 0.f) best = std::max(best, (double)n16 * 16.0 * reps / (ms * 1e-3) / 1e9);
        }
        if (!ok) break;
        *gbs = best;
        st = CS_OK;
    } while (false);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf); cudaFree(out);
    return st;
}

cs_status cs_diag_barrier_probe(cs_solver *S, int32_t n, double *us_per_barrier) {
    if (!S || n < 1 || !us_per_barrier) return CS_EINVAL;
    DeviceGuard guard(S);
    cudaEvent_t e0, e1;
    CS_CUDA(S, cudaEventCreate(&e0));
    CS_CUDA(S, cudaEventCreate(&e1));
    double *out = S->ctx.partial_probe;
    int nn = n;
    void *args[] = {&S->ctx, &nn, &out};
    cs_status st = launch_coop(S, (const void *)k_barrier_probe, args);   // warm-up
    if (st != CS_OK) return st;
    CS_CUDA(S, cudaEventRecord(e0, S->stream));
    if ((st = launch_coop(S, (const void *)k_barrier_probe, args)) != CS_OK) return st;
    CS_CUDA(S, cudaEventRecord(e1, S->stream));
    CS_CUDA(S, cudaEventSynchronize(e1));
    float ms = 0.f;
    CS_CUDA(S, cudaEventElapsedTime(&ms, e0, e1));
    double total = 0.0;
    CS_CUDA(S, cudaMemcpy(&total, out, sizeof(double), cudaMemcpyDeviceToHost));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (total != (double)n * S->grid * kBlock) { S->err = "barrier probe: wrong all-reduce result"; return CS_ECUDA; }
    *us_per_barrier = 1e3 * ms / n;
    return CS_OK;
}

cs_status cs_solution(cs_solver *S, double *x, double *z, double *y, double *s, double *O, cs_mem where) {
    if (!S) return CS_EINVAL;
    DeviceGuard guard(S);
    cs_status st;
    if ((st = ensure_xz(S)) != CS_OK) return st;
    const Ctx &c = S->ctx;
    const cudaMemcpyKind kind = where == CS_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    if (x && (st = export_cols(S, x, c.xb, where)) != CS_OK) return st;
    if (z && (st = export_cols(S, z, c.zb, where)) != CS_OK) return st;
    if (s && (st = export_cols(S, s, c.s, where)) != CS_OK) return st;
    if (O && (st = export_cols(S, O, c.O, where)) != CS_OK) return st;
    if (y) {
        double *ydev = where == CS_DEVICE ? y : c.r;  // r is scratch between solves
        k_dual_y<<<ew_blocks(c.m), 256, 0, S->stream>>>(c, ydev);
        CS_CUDA(S, cudaGetLastError());
        S->launches += 1;
        if (where == CS_HOST) CS_CUDA(S, cudaMemcpyAsync(y, ydev, sizeof(double) * c.m, kind, S->stream));
    }
    if (where == CS_HOST) CS_CUDA(S, cudaStreamSynchronize(S->stream));
    return CS_OK;
}

}  // extern "C"

// =================================================================================================
// cs_cone_violation_static -- the ONE entry point of the library that allocates nothing (cs.h): for callers that
// cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it).  It is the cone
// part of k_residuals (distance of x and z to K, their norms) as a handle-free kernel whose scratch -- the cone
// offsets, the per-CTA partial sums, the arrival ticket and the result -- lives in a file-scope device array of
// fixed size.  Every GPU that loads libcs.so holds these kStaticBytes until the process exits.
// In host code `g_static_scratch` is only a stand-in for the symbol; the device address comes from
// cudaGetSymbolAddress, once per device, with that device current (static_scratch_address).
// All calls share the array: calls that overlap on the GPU (different streams, different host threads) RACE.
// =================================================================================================
namespace {
constexpr int kStaticMaxSoc = CS_STATIC_MAX_SOC;     // largest n_soc the entry point accepts
constexpr int kStaticMaxGrid = 512;                  // CTAs of its launch (<= 2 per SM)
constexpr int kStaticThreads = 256;
constexpr size_t kStaticOffPartials = ((size_t)(kStaticMaxSoc + 1) * sizeof(int) + 255) / 256 * 256;
constexpr size_t kStaticOffTicket = kStaticOffPartials + (size_t)4 * kStaticMaxGrid * sizeof(double);
constexpr size_t kStaticOffOut = kStaticOffTicket + 256;
constexpr size_t kStaticBytes = kStaticOffOut + 256;   // 128 KB of offsets + 16 KB of partials + ticket + result
}  // namespace

static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

namespace {
// x, z [n] in the caller's order (orthant coordinates first, then the Lorentz blocks at off[0..n_soc]); out[5] =
// {||x - proj_K x||, ||z - proj_K z||, ||x||, ||z||, cone_viol_rel}.  One launch: every CTA leaves its four partial
// sums in the scratch, the last one to arrive (ticket) adds them in CTA order -- deterministic.
__global__ void __launch_bounds__(kStaticThreads) k_cone_violation_static(const double *x, const double *z, int n_lin, int n_soc,
                                                                          unsigned char *scratch, double *out) {
    const int *off = reinterpret_cast<const int *>(scratch);
    double *partials = reinterpret_cast<double *>(scratch + kStaticOffPartials);     // [4][gridDim]
    unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch + kStaticOffTicket);
    __shared__ double sm[4][kStaticThreads / 32];
    __shared__ bool last;
    const int tid = blockIdx.x * kStaticThreads + threadIdx.x, nth = gridDim.x * kStaticThreads;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double v[4] = {0.0, 0.0, 0.0, 0.0};                      // dist2(x), dist2(z), ||x||^2, ||z||^2
    for (int j = tid; j < n_lin; j += nth) {
        const double a = x[j], b = z[j], am = fmin(a, 0.0), bm = fmin(b, 0.0);
        v[0] += am * am; v[1] += bm * bm; v[2] += a * a; v[3] += b * b;
    }
    {   // Lorentz blocks: kConeLanes lanes per block, as in k_residuals
        const int sub = lane / kConeLanes, sl = lane % kConeLanes;
        constexpr int CPW = 32 / kConeLanes;
        const int gwarp = tid >> 5, nwarps = nth >> 5;
        for (int base = gwarp * CPW; base < n_soc; base += nwarps * CPW) {
            const int ci = base + sub;
            const bool act = ci < n_soc;
            const int a = act ? off[ci] : 0, b = act ? off[ci + 1] : 0;
            double nx = 0.0, nz = 0.0;
            for (int j = a + 1 + sl; j < b; j += kConeLanes) { nx += x[j] * x[j]; nz += z[j] * z[j]; }
            nx = group_reduce<kConeLanes>(nx);
            nz = group_reduce<kConeLanes>(nz);
            if (act && sl == 0) {
                v[0] += soc_dist2(x[a], nx); v[1] += soc_dist2(z[a], nz);
                v[2] += x[a] * x[a] + nx;    v[3] += z[a] * z[a] + nz;
            }
        }
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const double r = group_reduce<32>(v[q]);
        if (lane == 0) sm[q][warp] = r;
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double acc = sm[threadIdx.x][0];
        for (int w = 1; w < kStaticThreads / 32; ++w) acc += sm[threadIdx.x][w];
        __stcg(partials + (size_t)threadIdx.x * gridDim.x + blockIdx.x, acc);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!last) return;
    __threadfence();
    if (warp < 4) {                                          // warp q adds the partials of sum q in CTA order
        double acc = 0.0;
        for (int b = lane; b < (int)gridDim.x; b += 32) acc += __ldcg(partials + (size_t)warp * gridDim.x + b);
        acc = group_reduce<32>(acc);
        if (lane == 0) sm[warp][0] = sqrt(acc);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        out[0] = sm[0][0]; out[1] = sm[1][0]; out[2] = sm[2][0]; out[3] = sm[3][0];
        out[4] = (sm[0][0] + sm[1][0]) / (1.0 + sm[2][0] + sm[3][0]);
        *ticket = 0u;                                        // leave the ticket at zero for the next call
    }
}

// device address of g_static_scratch on the CURRENT device, resolved once per device (cudaGetSymbolAddress)
cs_status static_scratch_address(unsigned char **out, std::string *err) {
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static unsigned char *addr[kMaxDev] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDev) { *err = "no CUDA device"; return CS_ECUDA; }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        unsigned char *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_static_scratch);
        if (e != cudaSuccess || !p) { *err = std::string("cudaGetSymbolAddress(g_static_scratch): ") + cudaGetErrorString(e); return CS_ECUDA; }
        addr[dev] = p;
    }
    *out = addr[dev];
    return CS_OK;
}
}  // namespace

extern "C" cs_status cs_cone_violation_static(const double *x_dev, const double *z_dev, int64_t n, const cs_cones *K,
                                              double *out, cs_mem out_where, void *cuda_stream) {
    std::string &err = g_create_err;                         // no handle: the text goes where cs_create's goes (cs_last_error(NULL))
    if (!x_dev || !z_dev || !K || !out || n <= 0 || n >= INT32_MAX || K->n_lin < 0 || K->n_soc < 0 || (K->n_soc > 0 && !K->soc_size)) {
        err = "cs_cone_violation_static: NULL argument or bad sizes";
        return CS_EINVAL;
    }
    if (K->n_soc > kStaticMaxSoc) {
        err = "cs_cone_violation_static: n_soc = " + std::to_string(K->n_soc) + " exceeds the static scratch (at most " +
              std::to_string(kStaticMaxSoc) + " Lorentz cones); use cs_create + cs_residuals";
        return CS_EINVAL;
    }
    static thread_local int h_off[kStaticMaxSoc + 1];        // host staging of the offsets: no heap either
    int64_t off = K->n_lin;
    for (int64_t i = 0; i < K->n_soc; ++i) {
        if (K->soc_size[i] < 1) { err = "cs_cone_violation_static: soc_size entries must be >= 1"; return CS_EINVAL; }
        h_off[i] = (int)off;
        off += K->soc_size[i];
        if (off > n) break;
    }
    if (off != n) { err = "cs_cone_violation_static: n_lin + sum(soc_size) != n"; return CS_EINVAL; }
    h_off[K->n_soc] = (int)n;
    unsigned char *scratch = nullptr;
    cs_status st = static_scratch_address(&scratch, &err);
    if (st != CS_OK) return st;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // the array keeps the previous call's contents: the offsets are overwritten, the ticket must start at zero
    if (e == cudaSuccess) e = cudaMemcpyAsync(scratch, h_off, sizeof(int) * (size_t)(K->n_soc + 1), cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(scratch + kStaticOffTicket, 0, sizeof(unsigned int), stream);
    if (e == cudaSuccess) {
        const int64_t want = (n + kStaticThreads - 1) / kStaticThreads;
        const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(want, std::min(2 * sms, kStaticMaxGrid)));
        double *out_dev = out_where == CS_DEVICE ? out : reinterpret_cast<double *>(scratch + kStaticOffOut);
        k_cone_violation_static<<<grid, kStaticThreads, 0, stream>>>(x_dev, z_dev, (int)K->n_lin, (int)K->n_soc, scratch, out_dev);
        e = cudaGetLastError();
        if (e == cudaSuccess && out_where == CS_HOST) {
            e = cudaMemcpyAsync(out, out_dev, 5 * sizeof(double), cudaMemcpyDeviceToHost, stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
        }
    }
    // h_off is reused by the next call of this thread: the H2D copy from pageable memory has been staged when
    // cudaMemcpyAsync returns (CUDA runtime semantics for pageable host memory)
    if (e != cudaSuccess) { err = std::string("cs_cone_violation_static: ") + cudaGetErrorString(e); return CS_ECUDA; }
    return CS_OK;
}
