// A3 for LARGE candidate sets: stark_beam_topk with every SM of the GPU on it (topk_grid_kernel).
//
// Same definition as topk.cu (Eq. 1: beam score = sum of log-probabilities; PAPER.md:257,
// 263, 306: keep the top-W paths per level; readings R4 / R6):
//   key[i*C + c] = fl32(score[i] + logp[i, c]);  keep the W_out first in (key descending, flat index ascending).
// At the paper's own shape (C = 8192, widths 512 / 512 / 1024; B = 1, 8) a
// user has 4.2 M candidates (16.8 MB) per level.  One thread-block cluster per user (topk.cu) leaves most of the
// GPU idle there (16 SMs at B = 1, 64 at B = 8), so here a user is spread over S = capacity / B CTAs of a plain
// grid that is launched COOPERATIVELY (all CTAs co-resident), which makes a per-user barrier legal:
//
//   1. Every CTA owns the 2048-key chunks s, s + S, s + 2S, ... of its user (interleaved: parents arrive sorted
//      by score, so every CTA sees a sample of the best beams first).  It loads its first batch (8 chunks, 16 K
//      keys, all loads in flight at once), parks the keys in shared memory and reduces them to G group maxima
//      (group = the keys of 512 / G neighbouring threads).
//   2. It publishes the G maxima in the user's slice of the workspace and arrives at the user's barrier (the
//      next batch's loads are already in flight).  The LAST CTA to arrive reads all M = S * G maxima, takes
//      their K-th largest (K = W_out) as the user's bound L and releases the others: M disjoint groups, K of
//      them with a key >= L, hence at least K keys >= L, hence the K-th best key is >= L and NO key below L can
//      be selected.  With M ~ 4-8 K the number of keys >= L is 1.1-2 K.
//   3. The parked batch is filtered against L (which frees the key cache), then the rest of the slice is streamed
//      ONCE against L (one fp32 add and one compare per key): through a ring of 8 sixteen-byte slots per thread in
//      the key cache, filled by cp.async, so that 7-8 loads of every thread are in flight all the time; survivors
//      (a handful per CTA) go to a shared-memory list.  Unsorted parents make L loose: when the list fills up, the CTA re-tightens its
//      own bound from the list (its K-th largest entry is again a valid bound) and compacts -- a streaming top-K.
//   4. Every CTA writes its survivors, as composites (~ord(key) . index), and their count to its own segment of
//      the user's list in the workspace and arrives at the user's second barrier.  Then EVERY CTA copies the
//      whole list (1-2 K composites) into shared memory and ranks its OWN survivors against it, a warp per
//      survivor: the composites are all distinct, so the order "key descending, index ascending" is their plain
//      ascending order, rank = number of smaller composites, and the survivors of rank < K write their (score,
//      parent, code) row directly -- no sort, no serial tail, a result independent of arrival order.
//      Exceptional cases are finished by the last CTA to arrive alone: more than 8192 survivors (cut down by
//      exact radix passes, then ranked by bucketing), or a CTA that lost survivors (list overflow: K keys of
//      -inf, all keys equal, ...): the same exact selection over ALL keys of the user, read again by that one
//      CTA: slow, never wrong.
//   5. The last CTA to finish zeroes the user's workspace state, so the workspace only has to be zero ONCE, before its
//      first use (include/stark.h).
// Algorithmic HBM bytes: 4 per candidate (read once) + 4 per input beam + 12 per selected beam.
#include "common.cuh"

namespace stark {

namespace {

constexpr int kThreads = 512;
constexpr int kWarps = kThreads / 32;
constexpr int kUnroll = 8;                        // 16-byte loads per thread per batch
constexpr int kChunk = kThreads * 4;              // 2048 keys: one 16-byte load per thread
constexpr int kBatch = kChunk * kUnroll;          // 16384 keys parked in shared memory
constexpr int kBins = 2048;                       // 11-bit digits
constexpr int kCoarse = 64;
constexpr int kSvCap = 4096;                      // survivor list entries per CTA
constexpr int kEmitMax = 2048;                    // a CTA emits at most this many survivors
constexpr int kSortCap = 4096;                    // composites the last CTA ranks in shared memory (exceptional path)
constexpr int kRankCap = 8192;                    // survivors of a user every CTA ranks against (fills the key cache)
constexpr int kBucketMax = 192;                   // largest bucket ranked by counting (beyond: massive ties, sort)
constexpr int kMaxK = 1024;                       // W_out served by this path (kSvCap / 2 >= K for the re-tightening)
constexpr int kPubPerThread = 16;                 // published maxima a thread reads
constexpr int kMaxGroups = kPubPerThread * kThreads;   // published maxima per user at most (8192)
constexpr uint32_t kOverflow = 0x00400000u;       // added to a user's count by a CTA that lost survivors (> any real count; 512 of them do not wrap)
#ifndef STARK_GRID_MIN_N
#define STARK_GRID_MIN_N 131072
#endif
constexpr long long kGridMinN = STARK_GRID_MIN_N;  // candidates per user from which this path is tried (measured)
constexpr int kGridMaxCtas = 512;                 // CTAs of one launch at most (workspace sizing; 2 x 148 on B200)

#ifdef STARK_TOPK_PROF   // phase probes of scratch builds (never defined in the product build)
__device__ unsigned long long g_topk_prof[1024 * 16];
#define PROF(i)                                                                                            \
    do {                                                                                                   \
        if (threadIdx.x == 0) {                                                                            \
            unsigned long long t_;                                                                         \
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                                         \
            g_topk_prof[((blockIdx.y * gridDim.x + blockIdx.x) & 1023) * 16 + (i)] = t_;                   \
        }                                                                                                  \
    } while (0)
#define PROF_VAL(i, v) g_topk_prof[((blockIdx.y * gridDim.x + blockIdx.x) & 1023) * 16 + (i)] = (v)
#else
#define PROF(i) do {} while (0)
#define PROF_VAL(i, v) do {} while (0)
#endif

// Per-user counters, each on a cache line of its own (zero before the launch, zero after it).  The release words
// are NOT here: hundreds of CTAs polling one address saturate that L2 slice and delay the very atomics they wait
// for (measured: 5 us per barrier), so every CTA polls a slot of its own (RelSlot), which the releasing CTA writes.
struct UserState {
    uint32_t arrived_a, pad0[31];
    uint32_t arrived_b, pad1[31];
    uint32_t done, pad2[31];
    uint32_t count, pad3[31];                     // survivors appended to the user's list (+ kOverflow if any were lost)
};
static_assert(sizeof(UserState) == 512, "workspace layout");
struct RelSlot {                                  // one per CTA, 64 bytes apart
    unsigned long long a;                         // (1 << 32) | bound: written by the user's last CTA at barrier A
    unsigned long long b;                         // (1 << 63) | mode << 32 | survivors: ... at barrier B
    unsigned long long pad[6];
};
static_assert(sizeof(RelSlot) == 64, "workspace layout");

struct Shared {
    uint32_t hist[kBins];
    uint32_t coarse[kCoarse];                     // (directly behind hist: zeroed together)
    uint32_t wmax[kWarps], wmin[kWarps], wcnt[kWarps];
    unsigned long long w64a[kWarps], w64b[kWarps];
    uint32_t sel_bin, sel_rem, sel_cnt;
    uint32_t sv_count, sv_count2, bound, flag, cursor;
};

// dynamic shared memory: Shared | cache: kBatch keys (the last CTA: kSortCap composites + kSortCap bucketed) |
// sv: kSvCap survivors (the last CTA: bucket bases [kBins + 1] and segment offsets [kGridMaxCtas + 1])
constexpr size_t kSharedBytes = ((sizeof(Shared) + 15) / 16) * 16;
constexpr size_t kSmemBytes = kSharedBytes + (size_t)kBatch * 4 + (size_t)kSvCap * 8;
static_assert((size_t)kBatch * 4 >= (size_t)kSortCap * 16, "the key cache holds the last CTA's two composite arrays");
static_assert((size_t)kBatch * 4 >= (size_t)kRankCap * 8, "the key cache holds the user's whole survivor list");
static_assert((size_t)kSvCap * 8 >= (size_t)(kBins + 1 + kThreads) * 4, "bucket bases + scan words");

__device__ __forceinline__ uint32_t ord_of(float key) {
    uint32_t b = __float_as_uint(key);
    if (b == 0x80000000u) b = 0u;                 // -0.0 == +0.0 (IEEE comparison, reading R6)
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
// the float whose ord is `o` (o > 0); keys compare against it with the plain IEEE >=
__device__ __forceinline__ float ord_inv(uint32_t o) {
    return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}
__device__ __forceinline__ unsigned long long ld_acquire(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t ld_acquire32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// arrive at a counter: release this CTA's writes (ordered before by the CTA barrier), acquire the others'
__device__ __forceinline__ uint32_t atom_add_acq_rel(uint32_t* p, uint32_t v) {
    uint32_t old;
    asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], %2;" : "=r"(old) : "l"(p), "r"(v) : "memory");
    return old;
}
__device__ __forceinline__ void st_release(unsigned long long* p, unsigned long long v) {
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// One warp: descending-bin suffix scan over 32 per-lane counts c.  Finds the highest bin with
// sum_{b' >= b} c(b') >= rem; returns (bin 0..31, rem minus the counts above it, count inside it).
__device__ __forceinline__ void warp_select32(uint32_t c, uint32_t rem, int& bin, uint32_t& rem_out, uint32_t& cnt) {
    const int lane = threadIdx.x & 31;
    uint32_t inc = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_down_sync(0xffffffffu, inc, o);
        if (lane + o < 32) inc += t;
    }
    const uint32_t above = inc - c;
    const bool hit = above < rem && rem <= inc;
    const uint32_t bal = __ballot_sync(0xffffffffu, hit);
    const int src = bal ? __ffs(bal) - 1 : 0;     // bal == 0 only on inconsistent (NaN-poisoned) counts
    bin = src;
    rem_out = __shfl_sync(0xffffffffu, rem - above, src);
    cnt = __shfl_sync(0xffffffffu, c, src);
}

// warp 0: highest bin of sh.hist (coarse sums in sh.coarse) with suffix count >= rem (total >= rem required)
__device__ __forceinline__ void block_select(Shared& sh, uint32_t rem) {
    const int lane = threadIdx.x & 31;
    const uint32_t cu = sh.coarse[32 + lane], cl = sh.coarse[lane];
    const uint32_t tot_u = __reduce_add_sync(0xffffffffu, cu);
    int g, b;
    uint32_t r2, c2, r3, c3;
    if (tot_u >= rem) { warp_select32(cu, rem, g, r2, c2); g += 32; }
    else warp_select32(cl, rem - tot_u, g, r2, c2);
    warp_select32(sh.hist[32 * g + lane], r2, b, r3, c3);
    if (lane == 0) { sh.sel_bin = (uint32_t)(32 * g + b); sh.sel_rem = r3; sh.sel_cnt = c3; }
}

__device__ __forceinline__ void zero_hist(Shared& sh) {
    for (int b = threadIdx.x; b < kBins + kCoarse; b += kThreads) sh.hist[b] = 0;
}

// Code size matters here: every phase after the first batch runs once per CTA (or once per USER, in its last
// CTA), i.e. on a cold instruction cache -- straight-line unrolled code cost several microseconds of instruction
// fetch per phase.  Hence rolled loops over shared memory and __noinline__ helpers for everything rare.

// per-user view of the inputs
struct Keys {
    const float* __restrict__ lp;     // [N] log-probs (or raw logits) of the user
    const float* __restrict__ sc;     // [W_in] parent scores (or offsets), nullptr = zeros
    uint32_t N;
    int C, c_shift;
    __device__ __forceinline__ int row_of(uint32_t idx) const {
        return c_shift >= 0 ? (int)(idx >> c_shift) : (int)(idx / (uint32_t)C);
    }
    __device__ __forceinline__ float score_of(int row) const { return sc ? __ldg(sc + row) : 0.f; }
};

// coarse[g] = sum of the 32 fine bins of group g (8 threads x 4 bins); call between two barriers
__device__ __forceinline__ void coarse_from_hist(Shared& sh) {
    const int tid = threadIdx.x, lane = tid & 31;
    const uint4 v = reinterpret_cast<const uint4*>(sh.hist)[tid];
    uint32_t c4 = v.x + v.y + v.z + v.w;
    c4 += __shfl_xor_sync(0xffffffffu, c4, 1);
    c4 += __shfl_xor_sync(0xffffffffu, c4, 2);
    c4 += __shfl_xor_sync(0xffffffffu, c4, 4);
    if ((lane & 7) == 0) sh.coarse[tid >> 3] = c4;
}

// A value L such that at least K of the NON-ZERO values among the block's kNV * kThreads register-held values `v`
// (0 = absent) are >= L, within 2^-11 of their range of the K-th largest; 0 if there are fewer than K non-zero
// values.  Bisection on the value, counting by warp votes: shared-memory atomics cost ~2 cycles per VALUE on this
// machine (a 2048-bin histogram of 4.7 K values took 3 us), a bisection step ~0.06 us.  Block-uniform result.
template <int kNV>
__device__ __forceinline__ uint32_t kth_largest(Shared& sh, const uint32_t (&v)[kNV], uint32_t K) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t vmax = 0u, vmin = 0xffffffffu, cnt = 0u;
#pragma unroll
    for (int x = 0; x < kNV; ++x)
        if (v[x]) { vmax = max(vmax, v[x]); vmin = min(vmin, v[x]); ++cnt; }
    vmax = __reduce_max_sync(0xffffffffu, vmax);
    vmin = __reduce_min_sync(0xffffffffu, vmin);
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    if (lane == 0) { sh.wmax[warp] = vmax; sh.wmin[warp] = vmin; sh.wcnt[warp] = cnt; }
    __syncthreads();
    vmax = __reduce_max_sync(0xffffffffu, lane < kWarps ? sh.wmax[lane] : 0u);
    vmin = __reduce_min_sync(0xffffffffu, lane < kWarps ? sh.wmin[lane] : 0xffffffffu);
    cnt = __reduce_add_sync(0xffffffffu, lane < kWarps ? sh.wcnt[lane] : 0u);
    __syncthreads();
    if (cnt < K) return 0u;
    // invariant: count(v >= lo) >= K, count(v >= hi) < K  (hi = vmax + 1 conceptually: count 0 < K)
    uint32_t lo = vmin, hi = vmax;                // hi is tested with ">" below so that vmax itself stays eligible
    uint32_t n_lo = cnt;
#pragma unroll 1
    for (int it = 0; it < 11 && hi - lo > 1u && n_lo > K + (K >> 5); ++it) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        uint32_t c = 0;
#pragma unroll
        for (int x = 0; x < kNV; ++x) c += __popc(__ballot_sync(0xffffffffu, v[x] >= mid));   // (0 < mid always)
        if (lane == 0) sh.hist[(it & 1) * kWarps + warp] = c;
        __syncthreads();
        c = __reduce_add_sync(0xffffffffu, lane < kWarps ? sh.hist[(it & 1) * kWarps + lane] : 0u);
        if (c >= K) { lo = mid; n_lo = c; } else hi = mid;
    }
    __syncthreads();
    return lo;
}

// block-wide (max, min) of one 64-bit value per thread; ends with a barrier
__device__ __forceinline__ void block_minmax64(Shared& sh, unsigned long long& hi, unsigned long long& lo) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    }
    if (lane == 0) { sh.w64a[warp] = hi; sh.w64b[warp] = lo; }
    __syncthreads();
    hi = sh.w64a[0]; lo = sh.w64b[0];
#pragma unroll 1
    for (int w = 1; w < kWarps; ++w) { hi = max(hi, sh.w64a[w]); lo = min(lo, sh.w64b[w]); }
    __syncthreads();
}

// Ascending sort of the n <= 32 * kWarps * E composites in sel[0..n) (distinct; capacity 32 * kWarps * E in both
// sel and tmp).  Every warp bitonic-sorts a run of 32 * E in registers (strides >= 32 are thread-local, smaller
// ones exchange by shuffle: no barrier), then every element finds its final position by ranking: its position
// in its own run plus its lower bounds in the other runs (binary searches over shared memory).  Fallback of
// rank_emit (massive exact ties only).
template <int E>
__device__ __noinline__ void sort_runs(unsigned long long* sel, unsigned long long* tmp, int n) {
    constexpr int RUN = 32 * E;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_runs = (n + RUN - 1) / RUN;
    for (int i = n + tid; i < n_runs * RUN; i += kThreads) sel[i] = ~0ull;
    __syncthreads();
    unsigned long long v[E];
    if (warp < n_runs) {
#pragma unroll
        for (int x = 0; x < E; ++x) v[x] = sel[warp * RUN + x * 32 + lane];
#pragma unroll
        for (int k = 2; k <= RUN; k <<= 1) {
#pragma unroll
            for (int j = k >> 1; j > 0; j >>= 1) {
                if (j >= 32) {
                    const int dx = j >> 5;
#pragma unroll
                    for (int x = 0; x < E; ++x) {
                        if ((x & dx) == 0) {
                            const bool up = ((x << 5) & k) == 0;   // (k > j >= 32: bit k of the position is in x)
                            const unsigned long long a = v[x], b = v[x | dx];
                            if ((a > b) == up) { v[x] = b; v[x | dx] = a; }
                        }
                    }
                } else {
#pragma unroll
                    for (int x = 0; x < E; ++x) {
                        const unsigned long long pv = __shfl_xor_sync(0xffffffffu, v[x], j);
                        const bool lower = (lane & j) == 0, up = (((x << 5) | lane) & k) == 0;
                        v[x] = (lower == up) ? min(v[x], pv) : max(v[x], pv);
                    }
                }
            }
        }
#pragma unroll
        for (int x = 0; x < E; ++x) sel[warp * RUN + x * 32 + lane] = v[x];
    }
    __syncthreads();
    if (warp < n_runs) {
        int rk[E];
#pragma unroll
        for (int x = 0; x < E; ++x) rk[x] = x * 32 + lane;
#pragma unroll 1
        for (int w2 = 0; w2 < n_runs; ++w2) {
            if (w2 == warp) continue;
            const unsigned long long* run = sel + w2 * RUN;
            int lo[E];
#pragma unroll
            for (int x = 0; x < E; ++x) lo[x] = 0;
#pragma unroll 1
            for (int st = RUN / 2; st > 0; st >>= 1) {
#pragma unroll
                for (int x = 0; x < E; ++x)
                    if (run[lo[x] + st - 1] < v[x]) lo[x] += st;
            }
#pragma unroll
            for (int x = 0; x < E; ++x) rk[x] += lo[x] + (run[lo[x]] < v[x] ? 1 : 0);
        }
#pragma unroll
        for (int x = 0; x < E; ++x)
            if (v[x] != ~0ull) tmp[rk[x]] = v[x];          // (padding is never read back)
    }
    __syncthreads();
    for (int i = tid; i < n; i += kThreads) sel[i] = tmp[i];
    __syncthreads();
}

// (score, parent, code) row `rr` of user `u` from composite c
struct Out {
    float* __restrict__ score; int32_t* __restrict__ parent; int32_t* __restrict__ code;
    size_t row0;                                   // u * W_out
    __device__ __forceinline__ void put(const Keys& ks, uint32_t rr, unsigned long long c) const {
        const uint32_t idx = min((uint32_t)c, ks.N - 1);       // (clamp: memory safety on NaN-poisoned input)
        const int row = ks.row_of(idx);
        // the key is the composite's upper half (order-preserving map inverted); only a zero may be -0.0 or
        // +0.0 (both map to one ord): that one is recomputed
        const uint32_t o = ~(uint32_t)(c >> 32);
        score[row0 + rr] = o != 0x80000000u ? ord_inv(o) : __fadd_rn(ks.score_of(row), __ldg(ks.lp + idx));
        parent[row0 + rr] = row;
        code[row0 + rr] = (int)idx - row * ks.C;
    }
};

// Ranks the n <= kSortCap DISTINCT composites ent[0..n) ascending; those of rank < K write their result row.
// Counting sort on the top 11 bits of (c - min c), then every entry counts the smaller entries of its own
// bucket: a handful of barriers, no sorting network.  A bucket beyond kBucketMax entries (massive exact ties:
// the composites then differ in their index bits only) takes the register/merge sort instead.
// bucketed: kSortCap composites; base: kBins + 1 words; part: kThreads words.
__device__ __noinline__ void rank_emit(Shared& sh, unsigned long long* ent, unsigned long long* bucketed,
                                       uint32_t* base, uint32_t* part, int n, uint32_t K, const Keys& ks,
                                       const Out& out) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned long long hi = 0ull, lo = ~0ull;
#pragma unroll 4
    for (int i = tid; i < n; i += kThreads) { const unsigned long long c = ent[i]; hi = max(hi, c); lo = min(lo, c); }
    zero_hist(sh);
    if (tid == 0) sh.sel_cnt = 0;                     // (largest bucket, by atomicMax)
    block_minmax64(sh, hi, lo);
    const unsigned long long span = hi - lo;
    const int nb = span ? 64 - __clzll((long long)span) : 0;
    const int shift = max(nb - 11, 0);
    PROF(10);
#pragma unroll 4
    for (int i = tid; i < n; i += kThreads) atomicAdd(&sh.hist[(uint32_t)((ent[i] - lo) >> shift)], 1u);
    __syncthreads();
    PROF(11);
    // exclusive prefix over the 2048 buckets (4 per thread) + the largest bucket: per-thread sums to shared
    // memory, warp 0 scans the 512 sums (16 per lane), every thread adds its offset
    const uint4 h = reinterpret_cast<const uint4*>(sh.hist)[tid];
    part[tid] = h.x + h.y + h.z + h.w;
    uint32_t bmax = __reduce_max_sync(0xffffffffu, max(max(h.x, h.y), max(h.z, h.w)));
    if (lane == 0) atomicMax(&sh.sel_cnt, bmax);
    __syncthreads();
    if (warp == 0) {
        uint32_t tot = 0;
#pragma unroll 4
        for (int x = 0; x < kThreads / 32; ++x) tot += part[lane * (kThreads / 32) + x];
        uint32_t inc = tot;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        uint32_t run = inc - tot;
#pragma unroll 4
        for (int x = 0; x < kThreads / 32; ++x) {
            const uint32_t t = part[lane * (kThreads / 32) + x];
            part[lane * (kThreads / 32) + x] = run;
            run += t;
        }
    }
    __syncthreads();
    {
        const uint32_t b0 = part[tid];
        base[4 * tid] = b0; base[4 * tid + 1] = b0 + h.x; base[4 * tid + 2] = b0 + h.x + h.y;
        base[4 * tid + 3] = b0 + h.x + h.y + h.z;
        if (tid == kThreads - 1) base[kBins] = (uint32_t)n;
    }
    bmax = sh.sel_cnt;
    __syncthreads();
    PROF(12);
    PROF_VAL(15, bmax);
    if (bmax > (uint32_t)kBucketMax) {               // (block-uniform)
        sort_runs<kSortCap / kThreads>(ent, bucketed, n);
        for (uint32_t r = tid; r < K; r += kThreads) out.put(ks, r, ent[r]);
        return;
    }
    // scatter into the buckets (any order inside one), from the bucket's end
#pragma unroll 4
    for (int i = tid; i < n; i += kThreads) {
        const unsigned long long c = ent[i];
        const uint32_t b = (uint32_t)((c - lo) >> shift);
        bucketed[base[b] + atomicSub(&sh.hist[b], 1u) - 1u] = c;
    }
    __syncthreads();
    PROF(13);
    // rank = entries in lower buckets + smaller entries of the own bucket
#pragma unroll 1
    for (int i = tid; i < n; i += kThreads) {
        const unsigned long long c = bucketed[i];
        const uint32_t b = (uint32_t)((c - lo) >> shift);
        const uint32_t r0 = base[b], r1 = base[b + 1];
        if (r0 >= K) continue;
        uint32_t rk = r0;
#pragma unroll 1
        for (uint32_t q = r0; q < r1; q += 4) {       // 4 loads in flight
            const unsigned long long a0 = bucketed[q], a1 = q + 1 < r1 ? bucketed[q + 1] : ~0ull,
                                     a2 = q + 2 < r1 ? bucketed[q + 2] : ~0ull, a3 = q + 3 < r1 ? bucketed[q + 3] : ~0ull;
            rk += (a0 < c) + (a1 < c) + (a2 < c) + (a3 < c);
        }
        if (rk < K) out.put(ks, rk, c);
    }
}

// A superset (<= kSortCap entries, gathered into sel) of the K smallest of the n DISTINCT 64-bit composites
// `each` enumerates (n > kSortCap, n >= K).  `each(fn)` must enumerate the same multiset at every call,
// block-strided.  Exact radix select on (hi - c) from the top bits until the candidates fit.  Returns the count.
template <class Each>
__device__ int select_gather(Shared& sh, unsigned long long* sel, Each&& each, uint32_t n, uint32_t K) {
    const int tid = threadIdx.x, warp = tid >> 5;
    unsigned long long hi = 0ull, lo = ~0ull;
    each([&](unsigned long long c) { hi = max(hi, c); lo = min(lo, c); });
    block_minmax64(sh, hi, lo);
    const unsigned long long span = hi - lo;
    uint32_t rem = K, cb = n;
    unsigned long long pref = 0ull;
    int r = span ? 64 - __clzll((long long)span) : 0;    // unresolved low bits of y = hi - c
    bool first = true;                                   // nothing resolved: every entry is a candidate
#pragma unroll 1
    while ((K - rem) + cb > (uint32_t)kSortCap && r > 0) {
        const int w = min(11, r), shift = r - w;
        const uint32_t mask = (1u << w) - 1u;
        zero_hist(sh);
        __syncthreads();
        each([&](unsigned long long c) {
            const unsigned long long y = hi - c;
            if (first || (y >> r) == pref) atomicAdd(&sh.hist[(uint32_t)(y >> shift) & mask], 1u);
        });
        __syncthreads();
        coarse_from_hist(sh);
        __syncthreads();
        if (warp == 0) block_select(sh, rem);
        __syncthreads();
        pref = (first ? 0ull : (pref << w)) | (unsigned long long)sh.sel_bin;
        rem = sh.sel_rem;
        cb = sh.sel_cnt;
        r = shift;
        first = false;
        __syncthreads();
    }
    // gather: everything above the boundary bin plus the bin itself ((K - rem) + cb <= kSortCap entries)
    if (tid == 0) sh.cursor = 0;
    __syncthreads();
    each([&](unsigned long long c) {
        if (first || ((hi - c) >> r) >= pref) {
            const uint32_t pos = atomicAdd(&sh.cursor, 1u);
            if (pos < (uint32_t)kSortCap) sel[pos] = c;
        }
    });
    __syncthreads();
    return (int)min(sh.cursor, (uint32_t)kSortCap);
}

// rare path of the stream: the vector holds at least one key at or above the bound
__device__ __noinline__ void append4(Shared& sh, uint2* sv, float thr, float4 k, uint32_t idx) {
    const float kk[4] = {k.x, k.y, k.z, k.w};
#pragma unroll
    for (int e = 0; e < 4; ++e)
        if (kk[e] >= thr) {
            const uint32_t pos = atomicAdd(&sh.sv_count, 1u);
            if (pos < (uint32_t)kSvCap) sv[pos] = make_uint2(ord_of(kk[e]), idx + e);
        }
}

// The survivor list is more than half full (cnt entries): its K-th largest entry is a valid (tighter) bound;
// raise `bound` and compact the list.  Returns the new length.
__device__ __noinline__ uint32_t retighten(Shared& sh, uint2* sv, uint32_t cnt, uint32_t& bound, uint32_t K) {
    const int tid = threadIdx.x;
    uint2 mine[kSvCap / kThreads];
    uint32_t ov[kSvCap / kThreads];
#pragma unroll
    for (int x = 0; x < kSvCap / kThreads; ++x) {
        const uint32_t e = tid + x * kThreads;
        mine[x] = e < cnt ? sv[e] : make_uint2(0u, 0u);       // (ord of a real key is never 0)
        ov[x] = mine[x].x;
    }
    bound = max(bound, kth_largest<kSvCap / kThreads>(sh, ov, K));
    __syncthreads();
#pragma unroll
    for (int x = 0; x < kSvCap / kThreads; ++x)
        if (ov[x] && ov[x] >= bound) sv[atomicAdd(&sh.sv_count2, 1u)] = mine[x];
    __syncthreads();
    const uint32_t c2 = sh.sv_count2;
    __syncthreads();
    if (tid == 0) { sh.sv_count = c2; sh.sv_count2 = 0; }
    __syncthreads();
    return c2;
}

// The user's last CTA: rank the survivors of all S segments, write the result, leave the workspace zeroed.
__device__ __noinline__ void finish_user(Shared& sh, unsigned long long* ent, uint32_t* words, const Keys& ks,
                                         const Out& out, uint32_t K, uint32_t n_list, bool lost, int S, int G,
                                         UserState* st, uint32_t* upub, const unsigned long long* ulist, RelSlot* urel) {
    const int tid = threadIdx.x;
    unsigned long long* bucketed = ent + kSortCap;                            // kSortCap composites
    uint32_t* base = words;                                                   // kBins + 1 bucket bases
    uint32_t* part = base + kBins + 1;                                        // kThreads scan words
    int n_g;
    if (!lost && n_list >= K && n_list <= (uint32_t)kSortCap) {
#pragma unroll 4
        for (uint32_t i = tid; i < n_list; i += kThreads) ent[i] = __ldcg(ulist + i);
        n_g = (int)n_list;
        __syncthreads();
    } else if (!lost && n_list >= K) {
        n_g = select_gather(sh, ent, [&](auto&& put) {
#pragma unroll 4
            for (uint32_t i = tid; i < n_list; i += kThreads) put(__ldcg(ulist + i));
        }, n_list, K);
    } else {
        // a CTA lost survivors: the same exact selection over ALL keys of the user, read again by this CTA
        auto all_keys = [&](auto&& put) {
#pragma unroll 2
            for (uint32_t i = (uint32_t)tid * 4u; i < ks.N; i += kThreads * 4u) {
                const float4 v = __ldg(reinterpret_cast<const float4*>(ks.lp + i));
                const float sx = ks.score_of(ks.row_of(i));
                put(((unsigned long long)(~ord_of(__fadd_rn(sx, v.x))) << 32) | i);
                put(((unsigned long long)(~ord_of(__fadd_rn(sx, v.y))) << 32) | (i + 1));
                put(((unsigned long long)(~ord_of(__fadd_rn(sx, v.z))) << 32) | (i + 2));
                put(((unsigned long long)(~ord_of(__fadd_rn(sx, v.w))) << 32) | (i + 3));
            }
        };
        if (ks.N > (uint32_t)kSortCap) n_g = select_gather(sh, ent, all_keys, ks.N, K);
        else {
            if (tid == 0) sh.cursor = 0;
            __syncthreads();
            all_keys([&](unsigned long long c) { ent[atomicAdd(&sh.cursor, 1u)] = c; });
            __syncthreads();
            n_g = (int)ks.N;
        }
    }
    rank_emit(sh, ent, bucketed, base, part, n_g, K, ks, out);
    // leave the workspace zeroed
    for (int i = tid; i < S * G; i += kThreads) upub[i] = 0u;
    if (tid < S) { urel[tid].a = 0ull; urel[tid].b = 0ull; }
    if (tid < (int)(sizeof(UserState) / 4)) reinterpret_cast<uint32_t*>(st)[tid] = 0u;
}

__global__ void __launch_bounds__(kThreads, 2)
topk_grid_kernel(const float* __restrict__ logp, const float* __restrict__ score, int W_in, int C, int c_shift,
                 int W_out, float* __restrict__ out_score, int32_t* __restrict__ out_parent,
                 int32_t* __restrict__ out_code, int S, int G, UserState* __restrict__ state,
                 uint32_t* __restrict__ pub, unsigned long long* __restrict__ list, RelSlot* __restrict__ rel) {
    const int s = blockIdx.x, u = blockIdx.y;
    const int tid = threadIdx.x;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Shared& sh = *reinterpret_cast<Shared*>(smem_raw);
    float* cache = reinterpret_cast<float*>(smem_raw + kSharedBytes);                        // [kBatch] keys
    uint2* sv = reinterpret_cast<uint2*>(cache + kBatch);                                    // [kSvCap] (ord, idx)

    Keys ks;
    ks.N = (uint32_t)((long long)W_in * C);                    // < 2^31, N % 4 == 0 (C % 4 == 0)
    ks.lp = logp + (size_t)u * ks.N;
    ks.sc = score ? score + (size_t)u * W_in : nullptr;
    ks.C = C; ks.c_shift = c_shift;
    const uint32_t N = ks.N, K = (uint32_t)W_out;
    UserState* st = state + u;
    uint32_t* upub = pub + (size_t)u * kMaxGroups;
    unsigned long long* ulist = list + (size_t)u * S * kEmitMax;   // the user's survivor list (S * kEmitMax entries)
    RelSlot* urel = rel + (size_t)u * S;                       // release slot of CTA s at urel[s]
    const int n_chunks = (int)((N + kChunk - 1) / kChunk);
    const int my_chunks = s < n_chunks ? (n_chunks - s + S - 1) / S : 0;
    const float ninf = __int_as_float(0xff800000);

    if (tid == 0) { sh.sv_count = 0; sh.sv_count2 = 0; sh.flag = 0; }
    PROF(0);

    // key vector of local chunk k (global chunk s + k*S): 4 consecutive candidates of one parent beam
    auto idx_of = [&](int k) -> uint32_t { return (uint32_t)(s + k * S) * kChunk + (uint32_t)tid * 4u; };

    float4 lv[kUnroll];
    uint32_t ib[kUnroll];
    auto load_batch = [&](int k0) {                          // all loads of a batch in flight at once
#pragma unroll
        for (int x = 0; x < kUnroll; ++x) {
            ib[x] = k0 + x < my_chunks ? idx_of(k0 + x) : N;
            lv[x] = __ldg(reinterpret_cast<const float4*>(ks.lp + min(ib[x], N - 4)));
        }
    };

    // ---- 1. first batch: parked in shared memory, per-thread maximum ---------------------------------
    float tmax = ninf;
    bool any = false;
    load_batch(0);
#pragma unroll
    for (int x = 0; x < kUnroll; ++x) {
        float4 kx = make_float4(ninf, ninf, ninf, ninf);
        if (ib[x] < N) {
            const float sx = ks.score_of(ks.row_of(ib[x]));
            kx.x = __fadd_rn(sx, lv[x].x); kx.y = __fadd_rn(sx, lv[x].y);
            kx.z = __fadd_rn(sx, lv[x].z); kx.w = __fadd_rn(sx, lv[x].w);
            tmax = fmaxf(tmax, fmaxf(fmaxf(kx.x, kx.y), fmaxf(kx.z, kx.w)));
            any = true;
        }
        *reinterpret_cast<float4*>(cache + x * kChunk + tid * 4) = kx;
    }
    PROF(1);
    // ---- 2. publish the G group maxima; the user's last CTA to arrive computes the bound ---------------
    {
        uint32_t gmax = any ? ord_of(tmax) : 0u;          // 0 = no key (ord of a real key is never 0)
        const int gsz = kThreads / G;                     // threads per group: 1..32, a power of two
        for (int o = 1; o < gsz; o <<= 1) gmax = max(gmax, __shfl_xor_sync(0xffffffffu, gmax, o));
        if ((tid & (gsz - 1)) == 0) __stcg(upub + (size_t)s * G + tid / gsz, gmax);
    }
    if (kUnroll < my_chunks) load_batch(kUnroll);         // the next batch is in flight across the barrier
    // barrier pattern: the CTA barrier orders every thread's writes before thread 0's fence + atomic
    __syncthreads();
    if (tid == 0) sh.flag = atom_add_acq_rel(&st->arrived_a, 1u) == (uint32_t)(S - 1) ? 1u : 0u;
    __syncthreads();
    uint32_t bound;
    PROF(2);
    if (sh.flag) {                                        // everyone's maxima are published
        const int M = S * G;                              // <= kMaxGroups = kPubPerThread * kThreads
        uint32_t pv[kPubPerThread];
#pragma unroll
        for (int x = 0; x < kPubPerThread; ++x) {         // all loads in flight at once
            const int i = tid + x * kThreads;
            pv[x] = i < M ? __ldcg(upub + i) : 0u;
        }
        PROF(11);
        bound = kth_largest<kPubPerThread>(sh, pv, K);
        PROF(12);
        __syncthreads();
        if (tid < S) st_release(&urel[tid].a, (1ull << 32) | bound);
    } else {
        if (tid == 0) {
            unsigned long long r;
            while ((r = ld_acquire(&urel[s].a)) == 0ull) __nanosleep(20);
            sh.bound = (uint32_t)r;
        }
        __syncthreads();
        bound = sh.bound;
    }
    float thr = bound <= 0x007fffffu ? ninf : ord_inv(bound);     // (ord(-inf) = 0x007fffff; 0 = no bound)
    PROF(3);

    // ---- 3. the rest of the slice, once, against the bound ---------------------------------------------------
    bool lost = false;                                   // survivors were dropped: the user takes the slow path
    // 3a. the parked batch first: that frees the key cache, of which a thread only ever touches its OWN 16-byte
    // slots (8 of them), so no barrier is needed before it is reused as the ring of 3c
#pragma unroll 2
    for (int x = 0; x < kUnroll; ++x) {
        const uint32_t i0 = x < my_chunks ? idx_of(x) : N;
        if (i0 < N) {
            const float4 k4 = *reinterpret_cast<const float4*>(cache + x * kChunk + tid * 4);
            if (fmaxf(fmaxf(k4.x, k4.y), fmaxf(k4.z, k4.w)) >= thr) append4(sh, sv, thr, k4, i0);
        }
    }
    // 3b. chunks kRing0 .. go through a ring of kUnroll slots per thread filled by cp.async: 7-8 loads of the thread
    // are in flight ALL the time (batches held in registers went 8 -> 0 -> 8: one HBM round trip per batch, and
    // the 64-register budget has no room for a second batch).  Primed here, under the batch that is already in
    // registers (loaded across the barrier).
    constexpr int kRing0 = 2 * kUnroll;
    const uint32_t ring_base = (uint32_t)__cvta_generic_to_shared(cache) + (uint32_t)tid * 16u;
    auto ring_issue = [&](int k) {                       // chunk k into slot k % kUnroll (always commits a group)
        if (k < my_chunks) {
            const uint32_t i0 = min(idx_of(k), N - 4);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(ring_base + (uint32_t)(k & (kUnroll - 1)) * (kChunk * 4u)),
                         "l"(ks.lp + i0) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
#pragma unroll
    for (int j = 0; j < kUnroll; ++j) ring_issue(kRing0 + j);
    if (kUnroll < my_chunks) {
#pragma unroll
        for (int x = 0; x < kUnroll; ++x) {
            if (ib[x] < N) {
                const float sx = ks.score_of(ks.row_of(ib[x]));
                const float4 k4 = make_float4(__fadd_rn(sx, lv[x].x), __fadd_rn(sx, lv[x].y), __fadd_rn(sx, lv[x].z),
                                              __fadd_rn(sx, lv[x].w));
                if (fmaxf(fmaxf(k4.x, k4.y), fmaxf(k4.z, k4.w)) >= thr) append4(sh, sv, thr, k4, ib[x]);   // rare
            }
        }
    }
    // 3c. the ring
    int since_check = 0;
#pragma unroll 1
    for (int k = kRing0; k < my_chunks; ++k) {
        asm volatile("cp.async.wait_group %0;" ::"n"(kUnroll - 1) : "memory");   // chunk k has landed
        const float4 v = *reinterpret_cast<const float4*>(cache + (k & (kUnroll - 1)) * kChunk + tid * 4);
        ring_issue(k + kUnroll);                         // (its slot is free again)
        const uint32_t i0 = idx_of(k);
        if (i0 < N) {
            const float sx = ks.score_of(ks.row_of(i0));
            const float4 k4 = make_float4(__fadd_rn(sx, v.x), __fadd_rn(sx, v.y), __fadd_rn(sx, v.z), __fadd_rn(sx, v.w));
            if (fmaxf(fmaxf(k4.x, k4.y), fmaxf(k4.z, k4.w)) >= thr) append4(sh, sv, thr, k4, i0);   // rare
        }
        // the list is inspected every 32 chunks only (a block barrier per batch would stop the warps from
        // overlapping each other's load latency)
        if (++since_check < 4 * kUnroll && k + 1 < my_chunks) continue;
        since_check = 0;
        __syncthreads();
        const uint32_t c1 = sh.sv_count;                 // (block-uniform)
        __syncthreads();
        if (c1 > (uint32_t)kSvCap) { lost = true; break; }
        if (c1 > (uint32_t)(kSvCap / 2)) {
            if (retighten(sh, sv, c1, bound, K) > (uint32_t)(kSvCap / 2)) { lost = true; break; }
            thr = bound <= 0x007fffffu ? ninf : ord_inv(bound);
        }
    }
    asm volatile("cp.async.wait_all;" ::: "memory");     // (nothing of the ring is in flight when the cache is reused)
    PROF(4);
    uint32_t cnt = 0;
    if (!lost) {
        __syncthreads();
        cnt = sh.sv_count;
        __syncthreads();
        if (cnt > (uint32_t)kSvCap) lost = true;
        else if (cnt > (uint32_t)kEmitMax) { cnt = retighten(sh, sv, cnt, bound, K); if (cnt > (uint32_t)kEmitMax) lost = true; }
    }
    // ---- 4. append to the user's list (one reservation per CTA); second barrier ------------------------------
    if (tid == 0) sh.cursor = atomicAdd(&st->count, lost ? kOverflow : cnt);
    __syncthreads();
    {
        const uint32_t at = sh.cursor;
        if (!lost && at + cnt <= (uint32_t)(S * kEmitMax))
            for (uint32_t e = tid; e < cnt; e += kThreads)
                __stcg(ulist + at + e, ((unsigned long long)(~sv[e].x) << 32) | sv[e].y);
    }
    PROF(5);
    __syncthreads();
    if (tid == 0) sh.flag = atom_add_acq_rel(&st->arrived_b, 1u) == (uint32_t)(S - 1) ? 1u : 0u;
    __syncthreads();
    const bool last_b = sh.flag != 0u;
    // the last CTA to arrive sees the final count and decides how the user is finished:
    // mode 0: every CTA ranks a slice of the list; 1: the last CTA alone (too many survivors, or some were lost)
    uint32_t n_list, mode;
    if (last_b) {
        if (tid == 0) sh.sel_rem = __ldcg(&st->count);
        __syncthreads();
        n_list = sh.sel_rem;
        mode = (n_list > (uint32_t)kRankCap || n_list < K) ? 1u : 0u;      // (kOverflow > kRankCap)
        if (tid < S) st_release(&urel[tid].b, (1ull << 63) | ((unsigned long long)mode << 32) | n_list);
    } else {
        if (tid == 0) {
            unsigned long long r;
            while ((r = ld_acquire(&urel[s].b)) == 0ull) __nanosleep(20);
            sh.sel_bin = (uint32_t)(r >> 32) & 1u;
            sh.sel_rem = (uint32_t)r;
        }
        __syncthreads();
        mode = sh.sel_bin;
        n_list = sh.sel_rem;
    }
    PROF(6);
    Out out;
    out.score = out_score; out.parent = out_parent; out.code = out_code; out.row0 = (size_t)u * W_out;
    if (mode == 1u) {                                    // exceptional: the last CTA finishes the user alone
        if (!last_b) {
            if (tid == 0) atomicAdd(&st->done, 1u);      // (this CTA has read its release word)
            return;
        }
        if (tid == 0)
            while (ld_acquire32(&st->done) < (uint32_t)(S - 1)) __nanosleep(100);   // nobody polls the workspace any more
        __syncthreads();
        const bool some_lost = n_list >= kOverflow;
        finish_user(sh, reinterpret_cast<unsigned long long*>(cache), reinterpret_cast<uint32_t*>(sv), ks, out, K,
                    n_list, some_lost || n_list > (uint32_t)(S * kEmitMax), S, G, st, upub, ulist, urel);
        return;
    }
    // ---- every CTA: the user's whole list into shared memory, rank a slice of it --------------------------------
    unsigned long long* ent = reinterpret_cast<unsigned long long*>(cache);   // n_list <= kRankCap composites
#pragma unroll 4
    for (uint32_t i = tid; i < n_list; i += kThreads) ent[i] = __ldcg(ulist + i);
    __syncthreads();
    PROF(7);
    PROF_VAL(9, n_list);
    {   // CTA s ranks the s-th slice of the list (balanced, whatever CTA the survivors came from): a warp per
        // entry; the composites are distinct, so rank = number of smaller composites
        const int lane = tid & 31, warp = tid >> 5;
        const uint32_t per = (n_list + S - 1) / S, e1 = min(n_list, (uint32_t)(s + 1) * per);
#pragma unroll 1
        for (uint32_t e = (uint32_t)s * per + warp; e < e1; e += kWarps) {
            const unsigned long long c = ent[e];
            uint32_t rk = 0;
#pragma unroll 4
            for (uint32_t i = lane; i < n_list; i += 32) rk += ent[i] < c ? 1u : 0u;
            rk = __reduce_add_sync(0xffffffffu, rk);
            if (lane == 0 && rk < K) out.put(ks, rk, c);
        }
    }
    PROF(14);
    // ---- 5. the last CTA to finish leaves the workspace zeroed -----------------------------------------------
    __syncthreads();
    if (tid == 0) sh.flag = atomicAdd(&st->done, 1u) == (uint32_t)(S - 1) ? 1u : 0u;
    __syncthreads();
    if (!sh.flag) return;
    for (int i = tid; i < S * G; i += kThreads) upub[i] = 0u;
    if (tid < S) { urel[tid].a = 0ull; urel[tid].b = 0ull; }
    if (tid < (int)(sizeof(UserState) / 4)) reinterpret_cast<uint32_t*>(st)[tid] = 0u;
    PROF(8);
}

// ---- wide selections over SMALL candidate sets (decode step 0 with a wide beam) ---------------------------------
// N <= 8192 candidates per user, W_out up to 1024 (512 of the 8192 first-level codes; config 4: 512
// of 1024).  The cluster kernel of topk.cu spends 14.5 us there, nearly all of it latency: cluster launch, radix
// passes with cluster barriers, a one-CTA sort.  Here R CTAs per user work WITHOUT talking to each other: each of
// them reads all N keys (32 KB, the second reader finds them in L2), finds by bisection on the order-preserving
// uint32 image of the key -- warp votes, a block barrier per step -- a bound with at most K + K/32 keys at or
// above it (exact ties at the K-th key: a second bisection on the index inside the tie), gathers those survivors
// as composites (~ord . index) in shared memory, and ranks ITS share of them (by a hash of the index) by counting.
// All CTAs of a user hold the same survivor set (the counts are exact), so the ranks agree without any exchange;
// rank r writes row r.
constexpr int kWideNV = 16;                       // keys per thread
constexpr int kWideMaxN = kThreads * kWideNV;     // 8192
constexpr int kWideCap = 2048;                    // survivors (>= kWideMaxK + kWideMaxK / 32)
constexpr int kWideMaxK = 1024;

__global__ void __launch_bounds__(kThreads, 2)
topk_wide_kernel(const float* __restrict__ logp, const float* __restrict__ score, int W_in, int C, int c_shift,
                 int W_out, float* __restrict__ out_score, int32_t* __restrict__ out_parent,
                 int32_t* __restrict__ out_code, int R) {
    __shared__ Shared sh;
    __shared__ unsigned long long ent[kWideCap];
    const int s = blockIdx.x, u = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    Keys ks;
    ks.N = (uint32_t)((long long)W_in * C);
    ks.lp = logp + (size_t)u * ks.N;
    ks.sc = score ? score + (size_t)u * W_in : nullptr;
    ks.C = C; ks.c_shift = c_shift;
    const uint32_t N = ks.N, K = (uint32_t)W_out;
    if (tid == 0) sh.cursor = 0;

    // ---- all keys of the user, as ord (0 = no key), in registers: key x of this thread has index x * 512 + tid ----
    uint32_t v[kWideNV];
    {
        float lv[kWideNV];
#pragma unroll
        for (int x = 0; x < kWideNV; ++x) {
            const uint32_t idx = (uint32_t)(x * kThreads + tid);
            lv[x] = __ldg(ks.lp + min(idx, N - 1));
        }
#pragma unroll
        for (int x = 0; x < kWideNV; ++x) {
            const uint32_t idx = (uint32_t)(x * kThreads + tid);
            v[x] = idx < N ? ord_of(__fadd_rn(ks.score_of(ks.row_of(idx)), lv[x])) : 0u;
        }
    }
    // block-wide number of keys for which `pred(x)` holds (block-uniform; two barriers)
    auto block_count = [&](auto pred) -> uint32_t {
        uint32_t c = 0;
#pragma unroll
        for (int x = 0; x < kWideNV; ++x) c += __popc(__ballot_sync(0xffffffffu, pred(x)));
        if (lane == 0) sh.wcnt[warp] = c;
        __syncthreads();
        c = __reduce_add_sync(0xffffffffu, lane < kWarps ? sh.wcnt[lane] : 0u);
        __syncthreads();
        return c;
    };
    // ---- range of the keys -----------------------------------------------------------------------------------------
    uint32_t vmax = 0u, vmin = 0xffffffffu;
#pragma unroll
    for (int x = 0; x < kWideNV; ++x)
        if (v[x]) { vmax = max(vmax, v[x]); vmin = min(vmin, v[x]); }
    vmax = __reduce_max_sync(0xffffffffu, vmax);
    vmin = __reduce_min_sync(0xffffffffu, vmin);
    if (lane == 0) { sh.wmax[warp] = vmax; sh.wmin[warp] = vmin; }
    __syncthreads();
    vmax = __reduce_max_sync(0xffffffffu, lane < kWarps ? sh.wmax[lane] : 0u);
    vmin = __reduce_min_sync(0xffffffffu, lane < kWarps ? sh.wmin[lane] : 0xffffffffu);
    __syncthreads();
    // ---- bisection: count(v >= lo) >= K > count(v >= hi), until few enough keys are at or above lo ------------------
    const uint32_t slack = max(K >> 5, 8u);
    uint32_t lo = vmin, n_lo = N;
    unsigned long long hi = (unsigned long long)vmax + 1ull;      // (exclusive: no key is >= vmax + 1)
#pragma unroll 1
    while (hi - lo > 1ull && n_lo > K + slack) {
        const uint32_t mid = (uint32_t)(lo + ((hi - lo) >> 1));
        const uint32_t c = block_count([&](int x) { return v[x] >= mid; });      // (mid > 0: absent keys never count)
        if (c >= K) { lo = mid; n_lo = c; } else hi = mid;
    }
    // more keys at or above lo than the list holds: they are exact ties at ord == lo (hi == lo + 1).  Take the keys
    // above it and, of the tie, the K - count(v > lo) entries of lowest index (found by bisection on the index).
    uint32_t tie_last = 0xffffffffu;                              // ties with index <= tie_last are kept
    if (n_lo > (uint32_t)kWideCap) {
        const uint32_t n_gt = block_count([&](int x) { return v[x] > lo; });
        const uint32_t need = K - n_gt;                           // >= 1: count(v >= hi) < K
        long long jl = -1, jh = (long long)N - 1;                 // count(idx <= jl) < need <= count(idx <= jh)
#pragma unroll 1
        while (jh - jl > 1) {
            const long long jm = (jl + jh) >> 1;
            const uint32_t c = block_count([&](int x) { return v[x] == lo && (long long)(x * kThreads + tid) <= jm; });
            if (c >= need) jh = jm; else jl = jm;
        }
        tie_last = (uint32_t)jh;
    }
    // ---- gather the survivors (warp-aggregated reservation; the order in the list does not matter) -----------------
#pragma unroll
    for (int x = 0; x < kWideNV; ++x) {
        const uint32_t idx = (uint32_t)(x * kThreads + tid);
        const bool keep = v[x] != 0u && (v[x] > lo || (v[x] == lo && idx <= tie_last));
        const uint32_t bal = __ballot_sync(0xffffffffu, keep);
        if (bal) {
            uint32_t base = 0;
            if (lane == 0) base = atomicAdd(&sh.cursor, (uint32_t)__popc(bal));
            base = __shfl_sync(0xffffffffu, base, 0);
            const uint32_t pos = base + (uint32_t)__popc(bal & ((1u << lane) - 1u));
            if (keep && pos < (uint32_t)kWideCap) ent[pos] = ((unsigned long long)(~v[x]) << 32) | idx;
        }
    }
    __syncthreads();
    const uint32_t n_s = min(sh.cursor, (uint32_t)kWideCap);      // K <= n_s (the min: memory safety on NaN-poisoned counts)
    // ---- CTA s ranks its share of the survivors: a warp per entry, rank = number of smaller composites (all
    // distinct).  The share is defined by the entry's INDEX (hashed, so that strided survivors still spread), not
    // by its position: the lists of a user's CTAs hold the same set in different orders.
    Out out;
    out.score = out_score; out.parent = out_parent; out.code = out_code; out.row0 = (size_t)u * W_out;
    // (R is a power of two; a warp looks at 32 entries at a time, one per lane, and then ranks the ones that are its
    // CTA's, one after the other)
#pragma unroll 1
    for (uint32_t e0 = (uint32_t)warp * 32u; e0 < n_s; e0 += kWarps * 32u) {
        const uint32_t e = e0 + lane;
        const unsigned long long cand = e < n_s ? ent[e] : 0ull;
        uint32_t todo = __ballot_sync(0xffffffffu, e < n_s && (int)((((uint32_t)cand * 2654435761u) >> 16) & (uint32_t)(R - 1)) == s);
#pragma unroll 1
        while (todo) {
            const int src = __ffs(todo) - 1;
            todo &= todo - 1u;
            const unsigned long long c = __shfl_sync(0xffffffffu, cand, src);
            uint32_t rk = 0;
#pragma unroll 4
            for (uint32_t i = lane; i < n_s; i += 32) rk += ent[i] < c ? 1u : 0u;
            rk = __reduce_add_sync(0xffffffffu, rk);
            if (lane == 0 && rk < K) out.put(ks, rk, c);
        }
    }
}

// per device: CTAs of topk_grid_kernel that can be co-resident (a cooperative launch must fit)
int grid_capacity() {
    static PerDevice<int> cap;
    int& c = cap.here();
    if (c == 0) {
        if (cudaFuncSetAttribute(topk_grid_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes) != cudaSuccess) {
            (void)cudaGetLastError();
            return 0;
        }
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, topk_grid_kernel, kThreads, kSmemBytes) != cudaSuccess) {
            (void)cudaGetLastError();
            return 0;
        }
        c = per_sm * num_sms();
        if (c <= 0) c = -1;
    }
    return c > 0 ? c : 0;
}

bool grid_shape_ok(long long N, int C) { return N >= kGridMinN && (C & 3) == 0; }

// workspace: [B] UserState | [B][kMaxGroups] published maxima | [kGridMaxCtas][kEmitMax] survivor lists |
//            [kGridMaxCtas] release slots  (the B * S <= kGridMaxCtas CTAs of a launch share the last two)
constexpr size_t kWsTail = (size_t)kGridMaxCtas * kEmitMax * 8 + (size_t)kGridMaxCtas * sizeof(RelSlot);

}  // namespace

size_t topk_grid_workspace_bytes(int B, int W_in, int C) {
    const long long N = (long long)W_in * C;
    if (!grid_shape_ok(N, C)) return 0;
    return (size_t)B * (sizeof(UserState) + (size_t)kMaxGroups * 4) + kWsTail;
}

// Returns STARK_ERR_UNSUPPORTED when this path does not serve the problem (the caller falls back to topk.cu).
int launch_topk_grid(const float* logp, const float* score, int B, int W_in, int C, int W_out, float* out_score,
                     int32_t* out_parent, int32_t* out_code, void* ws, size_t ws_bytes, cudaStream_t st) {
    const long long N = (long long)W_in * C;
    if (!grid_shape_ok(N, C) || W_out > kMaxK || !ws || (reinterpret_cast<uintptr_t>(logp) & 15u) != 0)
        return STARK_ERR_UNSUPPORTED;
    if (ws_bytes < topk_grid_workspace_bytes(B, W_in, C)) return STARK_ERR_UNSUPPORTED;
    int cap = grid_capacity();
    if (cap > kGridMaxCtas) cap = kGridMaxCtas;
    if (cap < B) return STARK_ERR_UNSUPPORTED;           // more users than co-resident CTAs: one cluster per user
    const int n_chunks = (int)((N + kChunk - 1) / kChunk);
    int S = cap / B;
    if (S > n_chunks / 2) S = n_chunks / 2 > 0 ? n_chunks / 2 : 1;     // at least two chunks per CTA
    // G groups per CTA: M = S * G published maxima, 4 K .. 8 K (a tight bound), at most kMaxGroups
    int G = 16;
    while (G < kThreads && (long long)S * G < 4096) G <<= 1;
    if ((long long)S * G < 2LL * W_out || (long long)S * G > kMaxGroups) return STARK_ERR_UNSUPPORTED;
    char* p = static_cast<char*>(ws);
    UserState* state = reinterpret_cast<UserState*>(p);
    uint32_t* pub = reinterpret_cast<uint32_t*>(p + (size_t)B * sizeof(UserState));
    unsigned long long* list = reinterpret_cast<unsigned long long*>(p + (size_t)B * (sizeof(UserState) + (size_t)kMaxGroups * 4));
    RelSlot* rel = reinterpret_cast<RelSlot*>(list + (size_t)kGridMaxCtas * kEmitMax);
    int c_shift = -1;
    if ((C & (C - 1)) == 0) { c_shift = 0; while ((1 << c_shift) < C) ++c_shift; }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)S, (unsigned)B);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = kSmemBytes;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeCooperative;           // all CTAs co-resident: the per-user barrier is legal
    at[0].val.cooperative = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    STARK_CUDA_TRY(cudaLaunchKernelEx(&cfg, topk_grid_kernel, logp, score, W_in, C, c_shift, W_out, out_score,
                                      out_parent, out_code, S, G, state, pub, list, rel));
    return STARK_OK;
}

// Wide selections over small candidate sets (topk_wide_kernel).  UNSUPPORTED = not served here.
bool topk_wide_serves(long long N, int W_out) { return N <= kWideMaxN && W_out <= kWideMaxK; }

int launch_topk_wide(const float* logp, const float* score, int B, int W_in, int C, int W_out, float* out_score,
                     int32_t* out_parent, int32_t* out_code, cudaStream_t st) {
    const long long N = (long long)W_in * C;
    // measured (us per launch, here vs the cluster kernel): B = 8: 9.1-12.6 vs 13.9-14.4; B = 16: 11.3-12.6 vs 14.4;
    // B = 32: 14.8 vs 13.6; B = 64: 19.2 vs 14.4 -- with few CTAs per user the ranking is no longer spread thin
    if (!topk_wide_serves(N, W_out) || B > 16) return STARK_ERR_UNSUPPORTED;
    int c_shift = -1;
    if ((C & (C - 1)) == 0) { c_shift = 0; while ((1 << c_shift) < C) ++c_shift; }
    // CTAs per user: enough that the ranking (n_s^2 compares per user) is spread thin, no more than two per SM in all
    const int sms = num_sms() > 0 ? num_sms() : 148;
    int R = 16;                                       // a power of two (the kernel masks a hash with R - 1)
    while (R > 1 && R * B > sms) R >>= 1;             // (every CTA repeats the bisection: one CTA per SM at most)
    topk_wide_kernel<<<dim3((unsigned)R, (unsigned)B), kThreads, 0, st>>>(logp, score, W_in, C, c_shift, W_out, out_score,
                                                                         out_parent, out_code, R);
    STARK_LAUNCH_CHECK();
    return STARK_OK;
}

}  // namespace stark

#ifdef STARK_TOPK_PROF
extern "C" int stark_debug_topk_prof(unsigned long long* host_out) {
    return (int)cudaMemcpyFromSymbol(host_out, stark::g_topk_prof, sizeof(stark::g_topk_prof));
}
extern "C" int stark_debug_topk_prof_reset(void) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, stark::g_topk_prof) != cudaSuccess) return -1;
    return (int)cudaMemset(p, 0, sizeof(stark::g_topk_prof));
}
#endif
