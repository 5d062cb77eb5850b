// A3: stark_beam_topk -- per-level beam selection, bit-exact and deterministic.
//
// Beam score = sum of per-level log-probabilities (Eq. 1);
// each level keeps the top-W candidate paths.  Per user:
//   key[i*C + c] = fl32(score[i] + logp[i, c])          (one fp32 add, reading R4)
//   keep the W_out entries first in (key descending, flat index ascending)
//   (reading R6), output sorted in that order.
//
// Three kernels by problem size (launch_topk): N <= 512 candidates per user: one
// 256-thread CTA ranking by counting (topk_small_kernel); N <= 16384 and
// W_out <= 256: one 1024-thread CTA per user, bound from per-thread maxima +
// ranking by counting (topk_mid_kernel); N <= 8192, W_out <= 1024 and B <= 16
// (decode step 0 with a wide beam): R independent CTAs per user, bound by
// bisection, every CTA ranks a share (topk_wide_kernel in topk_grid.cu); from
// 131 072 candidates per user the whole-GPU kernel of topk_grid.cu; otherwise
// the cluster kernel described here (topk_kernel).  All produce the same order.
// stark_beam_topk_logits (reading R22) feeds the same kernels (raw logits, per-beam offset from
// logits_offset.cu); for a single-row user the small kernel computes that offset itself (kFold).
//
// The work is tiny next to its latency (1 MB per level at config 2), so the
// design minimises dependent phases and cross-CTA traffic (measured on B200: a
// DSMEM pull of whole 8 KB histograms from every rank costs 2-15k cycles, a
// block barrier ~130, a cluster barrier ~650):
//   load     one thread-block CLUSTER per user.  The user's candidates are dealt
//            to the CTAs in interleaved chunks of kChunk keys -- parent beams
//            arrive sorted by score, so contiguous slices would put nearly all
//            winners into rank 0.  Every CTA streams its chunks ONCE from HBM,
//            maps each key to an order-preserving uint32 `ord`, parks it in
//            shared memory and tracks (max, min) ord in registers.
//   range    the cluster-wide (max, min), exchanged through distributed shared
//            memory, gives the number `nb` of low ord bits in which keys can
//            differ at all.  Selection then runs on the virtual 64-bit key
//                 V = (ord's low nb bits) . (bitwise-not of the flat index)
//            -- all V are distinct, so "key descending, index ascending" is the
//            plain descending order of V and ties need no special path.
//   select   radix passes of 11 bits from the top of V: shared-memory histogram
//            (2048 bins) + a 64-entry coarse histogram (32 bins each); cluster
//            barrier; ONE warp per CTA pulls the coarse histograms of all ranks
//            (256 B each), finds the coarse bin holding the W_out-th key, pulls
//            only that bin's 32 fine counters from all ranks and finishes the
//            scan with shuffles.  Every CTA computes the same answer: no
//            broadcast.  The loop stops as soon as "keys above the boundary bin
//            + keys inside it" fits the sort buffer -- normally after one or two
//            passes; heavy ties simply run on into the index bits.
//   gather   every CTA appends its qualifying keys as composites (~ord, idx) to
//            its own list; CTA 0 pulls the lists after a cluster barrier.
//   prune    (large slices) shared-memory atomics cost ~1 cycle per key, so
//            every CTA first derives a bound L such that at least W_out of its
//            own keys are >= L (the W_out-th largest of its per-thread bucket
//            maxima): no key below L can be selected.  The first pass touches
//            the histogram only for keys >= L and parks them in a survivor list
//            that all later steps walk instead of the whole slice.  Keys beyond
//            the shared-memory cache are never parked: they are streamed ONCE
//            against L, and whenever the survivor list fills up L is
//            re-tightened from the list itself and the list compacted (a
//            streaming top-K).  Bursts or heavy ties that overflow the list fall
//            back to re-reading those keys through L2.
//   sort     CTA 0 sorts the composites (a strict total order: the result does
//            not depend on arrival order): rank sort up to 256; up to 1024 every
//            warp bitonic-sorts a run of 64 in registers and the runs are merged
//            by ranking (binary searches); writes the first W_out as (score,
//            parent, code), recomputing score with the same fp32 add.
// Algorithmic HBM bytes: 4 per candidate (read once) + 4 per input beam + 12
// per selected beam; keys beyond the shared-memory
// cache (paper-scale codebooks) are read once (see `prune`).
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace stark {

namespace {

constexpr int kThreads = 512;
constexpr int kWarps = kThreads / 32;
constexpr int kUnroll = 8;
constexpr int kChunk = 1024;          // keys dealt to one rank at a time
constexpr int kBins = 2048;           // 11-bit digits
constexpr int kCoarse = 64;           // coarse bins, 32 fine bins each
constexpr int kMaxCluster = 16;       // non-portable size, used only when the device can co-schedule it
constexpr int kSliceMin = 2048;       // do not split a user into slices smaller than this
constexpr int kRankSortMax = 256;    // up to here a counting rank sort beats the bitonic network
constexpr int kRegSortMax = 1024;     // sorted runs of 64 per warp + merge by ranking
constexpr int kSmemBudget = 227 * 1024;
constexpr int kMinCacheKeys = 8192;   // smallest key cache worth launching with (launch_topk)

struct Shared {
    uint32_t hist[2][kBins];       // ping-pong by pass parity
    uint32_t coarse[2][kCoarse];
    uint32_t warp_max[kWarps], warp_min[kWarps];
    uint32_t list_len[kMaxCluster];
    uint32_t sel_bin, sel_rem, sel_cnt;
    uint32_t cta_max, cta_min;     // this CTA's keys (read remotely)
    uint32_t cursor;               // length of this CTA's list (read remotely)
    uint32_t warp_cnt[kWarps];
    uint32_t prune_lb;             // lower bound (ord value) below which no key of this CTA can be selected
    uint32_t sv_count2;            // second counter for compacting the survivor list
    uint32_t sv_count;             // survivors of the pruning pass (may exceed the list capacity: overflow)
};

__device__ __forceinline__ uint32_t ord_of(float key) {
    uint32_t b = __float_as_uint(key);
    if (b == 0x80000000u) b = 0u;  // -0.0 == +0.0 (IEEE comparison, reading R6)
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

// One warp: descending-bin suffix scan over 32 per-lane counts c (lane l = bin base+l).  Finds the highest
// bin with  sum_{b' >= b} c(b') >= rem.  Returns (bin offset 0..31, rem minus the counts above it, count
// inside it) to every lane.  Requires the warp total >= rem.
__device__ __forceinline__ void warp_select32(uint32_t c, uint32_t rem, int& bin, uint32_t& rem_out, uint32_t& cnt) {
    const int lane = threadIdx.x & 31;
    uint32_t inc = c;  // inclusive suffix sum: lanes >= l
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_down_sync(0xffffffffu, inc, o);
        if (lane + o < 32) inc += t;
    }
    const uint32_t above = inc - c;
    const bool hit = above < rem && rem <= inc;  // exactly one lane
    const uint32_t bal = __ballot_sync(0xffffffffu, hit);
    const int src = bal ? __ffs(bal) - 1 : 0;    // bal == 0 only on inconsistent (NaN-poisoned) counts
    bin = src;
    rem_out = __shfl_sync(0xffffffffu, rem - above, src);
    cnt = __shfl_sync(0xffffffffu, c, src);
}

__global__ void __launch_bounds__(kThreads, 1)
topk_kernel(const float* __restrict__ logp, const float* __restrict__ score, int W_in, int C, int c_shift,
            int W_out, float* __restrict__ out_score, int32_t* __restrict__ out_parent,
            int32_t* __restrict__ out_code, int cache_cap, int cap, int prune) {
    cg::cluster_group cluster = cg::this_cluster();
    const int nc = (int)cluster.num_blocks();
    const int rank = (int)cluster.block_rank();
    const int u = blockIdx.x / nc;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    Shared& sh = *reinterpret_cast<Shared*>(smem_raw);
    unsigned long long* sel = reinterpret_cast<unsigned long long*>(smem_raw + ((sizeof(Shared) + 15) / 16) * 16);
    const int svcap = 4 * cap;                                // entries of each survivor buffer (iff prune)
    uint2* sv = reinterpret_cast<uint2*>(sel + cap);          // survivors (ord, idx)
    uint2* sv_alt = sv + (prune ? svcap : 0);                 // compaction target; the two swap roles
    uint32_t* cache = reinterpret_cast<uint32_t*>(sv + (prune ? 2 * svcap : 0));

    // ---- this rank's keys: chunks rank, rank + nc, ... of kChunk consecutive flat indices -------------
    const uint32_t N = (uint32_t)((long long)W_in * C);  // < 2^31 (validated by the API)
    const int n_chunks = (int)((N + kChunk - 1) / kChunk);
    const int my_chunks = rank < n_chunks ? (n_chunks - rank + nc - 1) / nc : 0;
    const int span = my_chunks * kChunk;  // local positions j in [0, span); the last chunk may be ragged
    const float* __restrict__ lp = logp + (size_t)u * N;
    const float* __restrict__ sc = score ? score + (size_t)u * W_in : nullptr;

    auto idx_of = [&](int j) -> uint32_t {
        return ((uint32_t)(j / kChunk) * (uint32_t)nc + (uint32_t)rank) * kChunk + (uint32_t)(j % kChunk);
    };

    for (int b = tid; b < 2 * kBins + 2 * kCoarse; b += kThreads) (&sh.hist[0][0])[b] = 0;  // hist + coarse
    if (tid == 0) { sh.cursor = 0; sh.prune_lb = 0; sh.sv_count = 0; sh.sv_count2 = 0; }

    // ---- load: the one pass over HBM ---------------------------------------------------
    // All loads of an iteration are issued before any is consumed: indices are clamped instead of branched
    // around (a branch per key made ptxas wait for each load pair in turn: 8 round trips instead of 1).
    // bm[]: running maxima of 4 disjoint key subsets per thread ("buckets"), used to prune the histograms.
    uint32_t mx = 0u, mn = 0xffffffffu;
    uint32_t bm[4] = {0u, 0u, 0u, 0u};
    // With pruning, only the keys that fit the cache are loaded here; the rest is streamed ONCE further down,
    // after a selection bound is known, and only its few survivors are kept.
    const bool pruning = prune && N > (uint32_t)cap;
    const int span_c = (pruning && span > cache_cap) ? cache_cap : span;   // keys handled by this first loop
    const bool vec = (N & 3u) == 0 && (!sc || (C & 3) == 0) && ((reinterpret_cast<uintptr_t>(lp) & 15u) == 0) &&
                     (cache_cap & 3) == 0;
    if (vec) {
        // 16-byte loads: 4 consecutive candidates of one parent beam per load, 64 KB in flight per CTA
        const int span4 = span_c >> 2;
        for (int base4 = 0; base4 < span4; base4 += kThreads * kUnroll) {
            float4 lv[kUnroll];
            float sv[kUnroll];
#pragma unroll
            for (int x = 0; x < kUnroll; ++x) {
                const uint32_t idx = min(idx_of(4 * (base4 + x * kThreads + tid)), N - 4);
                const int row = c_shift >= 0 ? (int)(idx >> c_shift) : (int)(idx / (uint32_t)C);
                lv[x] = __ldg(reinterpret_cast<const float4*>(lp + idx));
                sv[x] = sc ? __ldg(sc + row) : 0.f;
            }
#pragma unroll
            for (int x = 0; x < kUnroll; ++x) {
                const int j = 4 * (base4 + x * kThreads + tid);
                if (j < span_c && idx_of(j) < N) {
                    uint4 o;
                    o.x = ord_of(__fadd_rn(sv[x], lv[x].x)); o.y = ord_of(__fadd_rn(sv[x], lv[x].y));
                    o.z = ord_of(__fadd_rn(sv[x], lv[x].z)); o.w = ord_of(__fadd_rn(sv[x], lv[x].w));
                    if (j < cache_cap) *reinterpret_cast<uint4*>(cache + j) = o;
                    const uint32_t hi = max(max(o.x, o.y), max(o.z, o.w)), lo4 = min(min(o.x, o.y), min(o.z, o.w));
                    mx = max(mx, hi); mn = min(mn, lo4);
                    bm[x & 3] = max(bm[x & 3], hi);
                }
            }
        }
    } else {
        for (int base = 0; base < span_c; base += kThreads * kUnroll) {
            float lv[kUnroll], sv[kUnroll];
#pragma unroll
            for (int x = 0; x < kUnroll; ++x) {
                const uint32_t idx = min(idx_of(base + x * kThreads + tid), N - 1);
                const int row = c_shift >= 0 ? (int)(idx >> c_shift) : (int)(idx / (uint32_t)C);
                lv[x] = __ldg(lp + idx);
                sv[x] = sc ? __ldg(sc + row) : 0.f;
            }
#pragma unroll
            for (int x = 0; x < kUnroll; ++x) {
                const int j = base + x * kThreads + tid;
                if (j < span_c && idx_of(j) < N) {
                    const uint32_t o = ord_of(__fadd_rn(sv[x], lv[x]));
                    if (j < cache_cap) cache[j] = o;
                    mx = max(mx, o); mn = min(mn, o);
                    bm[x & 3] = max(bm[x & 3], o);
                }
            }
        }
    }
    // ---- pruning bound (large slices) -----------------------------------------------------------
    // Shared-memory atomics cost ~1 cycle per key, so a histogram over all keys would dominate.  Any value L such
    // that at least K of this CTA's keys are >= L is a lower bound of the user's W_out-th key, so this CTA may
    // drop every key below L (the histograms then miss only keys below the user's threshold: the boundary bin is
    // still found).  L = lower edge of the 11-bit bin holding the K-th largest of a set of
    // real keys: first the per-thread bucket maxima of the parked keys, later the survivor list itself.
    auto block_minmax = [&](uint32_t& vmax, uint32_t& vmin, uint32_t& cnt) {   // block-wide (max, min, sum)
        vmax = __reduce_max_sync(0xffffffffu, vmax);
        vmin = __reduce_min_sync(0xffffffffu, vmin);
        cnt = __reduce_add_sync(0xffffffffu, cnt);
        if (lane == 0) { sh.warp_max[warp] = vmax; sh.warp_min[warp] = vmin; sh.warp_cnt[warp] = cnt; }
        __syncthreads();
        vmax = __reduce_max_sync(0xffffffffu, lane < kWarps ? sh.warp_max[lane] : 0u);
        vmin = __reduce_min_sync(0xffffffffu, lane < kWarps ? sh.warp_min[lane] : 0xffffffffu);
        cnt = __reduce_add_sync(0xffffffffu, lane < kWarps ? sh.warp_cnt[lane] : 0u);
        __syncthreads();                             // (the per-warp slots are reused)
    };
    // K-th largest of the values `each` enumerates (>= K of them, all inside [vmin, vmax]), as a bin edge
    auto kth_bound = [&](auto&& each, uint32_t vmax, uint32_t vmin) -> uint32_t {
        const int nbl = vmax == vmin ? 0 : 32 - __clz((int)(vmax ^ vmin));
        const int shl = max(nbl - 11, 0);
        const uint32_t mkl = nbl >= 32 ? 0xffffffffu : ((1u << nbl) - 1u);
        for (int b = tid; b < kBins + kCoarse; b += kThreads) (b < kBins ? sh.hist[1][b] : sh.coarse[1][b - kBins]) = 0;
        __syncthreads();
        each([&](uint32_t v) { atomicAdd(&sh.hist[1][(v & mkl) >> shl], 1u); });
        __syncthreads();
        {
            const uint4 v = reinterpret_cast<const uint4*>(&sh.hist[1][0])[tid];
            uint32_t c4 = v.x + v.y + v.z + v.w;
            c4 += __shfl_xor_sync(0xffffffffu, c4, 1);
            c4 += __shfl_xor_sync(0xffffffffu, c4, 2);
            c4 += __shfl_xor_sync(0xffffffffu, c4, 4);
            if ((lane & 7) == 0) sh.coarse[1][tid >> 3] = c4;
        }
        __syncthreads();
        if (warp == 0) {
            const uint32_t chi = sh.coarse[1][32 + lane], clo = sh.coarse[1][lane];
            const uint32_t tot_hi = __reduce_add_sync(0xffffffffu, chi);
            const bool in_hi = (uint32_t)W_out <= tot_hi;
            int cbin, fbin; uint32_t rem2, rem3, cnt;
            warp_select32(in_hi ? chi : clo, in_hi ? (uint32_t)W_out : (uint32_t)W_out - tot_hi, cbin, rem2, cnt);
            const int coarse_bin = (in_hi ? 32 : 0) + cbin;
            warp_select32(sh.hist[1][coarse_bin * 32 + lane], rem2, fbin, rem3, cnt);
            if (lane == 0) sh.prune_lb = (vmax & ~mkl) | ((uint32_t)(coarse_bin * 32 + fbin) << shl);
        }
        __syncthreads();                             // (hist[1] / coarse[1] are re-zeroed during pass 0)
        return sh.prune_lb;
    };
    uint32_t ord_lb = 0u;
    if (pruning) {
        uint32_t bx = max(max(bm[0], bm[1]), max(bm[2], bm[3])), bn = 0xffffffffu, nv = 0;
#pragma unroll
        for (int b = 0; b < 4; ++b)
            if (bm[b]) { bn = min(bn, bm[b]); ++nv; }
        block_minmax(bx, bn, nv);
        if (nv >= (uint32_t)W_out)                   // (block-uniform)
            ord_lb = kth_bound([&](auto&& put) {
#pragma unroll
                for (int b = 0; b < 4; ++b)
                    if (bm[b]) put(bm[b]);
            }, bx, bn);
    }
    // ---- the keys beyond the cache: streamed ONCE; only those above the bound are kept, and the bound is
    // re-tightened from the survivor list itself whenever that fills up (a streaming top-K) -----------------
    const bool tail_streamed = pruning && span > cache_cap;
    bool tail_ok = true;                             // false: survivors were lost, fall back to re-reading
    if (tail_streamed) {
        const int batch = kThreads * kUnroll * (vec ? 4 : 1);
        int since_check = 0;
        for (int base = cache_cap; base < span; base += batch) {
            auto keep = [&](uint32_t o, uint32_t idx) {
                mx = max(mx, o); mn = min(mn, o);
                if (tail_ok && o >= ord_lb) {        // rare: K-ish keys per user
                    const uint32_t pos = atomicAdd(&sh.sv_count, 1u);
                    if (pos < (uint32_t)svcap) sv[pos] = make_uint2(o, idx);
                }
            };
            if (vec) {
                float4 lv[kUnroll];
                float sv1[kUnroll];
                uint32_t ib[kUnroll];
#pragma unroll
                for (int x = 0; x < kUnroll; ++x) {
                    const int j = base + 4 * (x * kThreads + tid);
                    ib[x] = j < span ? idx_of(j) : N;
                    const uint32_t idc = min(ib[x], N - 4);
                    const int row = c_shift >= 0 ? (int)(idc >> c_shift) : (int)(idc / (uint32_t)C);
                    lv[x] = __ldg(reinterpret_cast<const float4*>(lp + idc));
                    sv1[x] = sc ? __ldg(sc + row) : 0.f;
                }
#pragma unroll
                for (int x = 0; x < kUnroll; ++x) {
                    if (ib[x] < N) {
                        keep(ord_of(__fadd_rn(sv1[x], lv[x].x)), ib[x]);
                        keep(ord_of(__fadd_rn(sv1[x], lv[x].y)), ib[x] + 1);
                        keep(ord_of(__fadd_rn(sv1[x], lv[x].z)), ib[x] + 2);
                        keep(ord_of(__fadd_rn(sv1[x], lv[x].w)), ib[x] + 3);
                    }
                }
            } else {
                float lv[kUnroll], sv1[kUnroll];
                uint32_t ib[kUnroll];
#pragma unroll
                for (int x = 0; x < kUnroll; ++x) {
                    const int j = base + x * kThreads + tid;
                    ib[x] = j < span ? idx_of(j) : N;
                    const uint32_t idc = min(ib[x], N - 1);
                    const int row = c_shift >= 0 ? (int)(idc >> c_shift) : (int)(idc / (uint32_t)C);
                    lv[x] = __ldg(lp + idc);
                    sv1[x] = sc ? __ldg(sc + row) : 0.f;
                }
#pragma unroll
                for (int x = 0; x < kUnroll; ++x)
                    if (ib[x] < N) keep(ord_of(__fadd_rn(sv1[x], lv[x])), ib[x]);
            }
            // the list is inspected every 4th batch only: a block barrier per batch would stop the warps from
            // overlapping each other's load latency (measured 2x on the whole stream)
            if (++since_check < 4 && base + batch < span) continue;
            since_check = 0;
            __syncthreads();
            const uint32_t cnt = sh.sv_count;        // (block-uniform)
            __syncthreads();                         // everyone has read it before the next batch appends
            if (tail_ok && cnt > (uint32_t)(svcap / 2)) {
                if (cnt > (uint32_t)svcap) {
                    tail_ok = false;                 // entries were dropped
                } else {                             // re-tighten: K-th largest survivor, then compact the list
                    uint32_t bx = 0u, bn = 0xffffffffu, nv = 0;
                    for (uint32_t e = tid; e < cnt; e += kThreads) { bx = max(bx, sv[e].x); bn = min(bn, sv[e].x); ++nv; }
                    block_minmax(bx, bn, nv);
                    const uint32_t nl = kth_bound([&](auto&& put) {
                        for (uint32_t e = tid; e < cnt; e += kThreads) put(sv[e].x);
                    }, bx, bn);
                    ord_lb = max(ord_lb, nl);
                    for (uint32_t e = tid; e < cnt; e += kThreads)
                        if (sv[e].x >= ord_lb) sv_alt[atomicAdd(&sh.sv_count2, 1u)] = sv[e];
                    __syncthreads();
                    const uint32_t c2 = sh.sv_count2;
                    __syncthreads();
                    if (tid == 0) { sh.sv_count = c2; sh.sv_count2 = 0; }
                    uint2* t2 = sv; sv = sv_alt; sv_alt = t2;
                    if (c2 > (uint32_t)(svcap / 2)) tail_ok = false;       // ties: the list cannot shrink
                    __syncthreads();
                }
            }
        }
    }
    mx = __reduce_max_sync(0xffffffffu, mx);
    mn = __reduce_min_sync(0xffffffffu, mn);
    if (lane == 0) { sh.warp_max[warp] = mx; sh.warp_min[warp] = mn; }
    __syncthreads();
    if (warp == 0) {
        mx = __reduce_max_sync(0xffffffffu, lane < kWarps ? sh.warp_max[lane] : 0u);
        mn = __reduce_min_sync(0xffffffffu, lane < kWarps ? sh.warp_min[lane] : 0xffffffffu);
        if (lane == 0) { sh.cta_max = mx; sh.cta_min = mn; }
    }
    cluster.sync();

    // ---- range: low ord bits in which any two keys of this user can differ ----------------------
    {
        uint32_t a = 0u, b = 0xffffffffu;
        if (lane < nc) {
            a = *cluster.map_shared_rank(&sh.cta_max, lane);
            b = *cluster.map_shared_rank(&sh.cta_min, lane);
        }
        mx = __reduce_max_sync(0xffffffffu, a);
        mn = __reduce_min_sync(0xffffffffu, b);
    }
    const int nb = (mx == mn) ? 0 : 32 - __clz((int)(mx ^ mn));
    const int nbi = N > 1 ? 32 - __clz((int)(N - 1)) : 0;  // index bits
    const uint32_t lowmask = nb >= 32 ? 0xffffffffu : ((1u << nb) - 1u);
    const uint32_t idxmask = (uint32_t)((1ull << nbi) - 1ull);
    // virtual key: all distinct, descending V == (key descending, index ascending)
    auto vkey = [&](uint32_t o, uint32_t idx) -> unsigned long long {
        return ((unsigned long long)(o & lowmask) << nbi) | (unsigned long long)(~idx & idxmask);
    };

    // Walk ALL keys of this rank, warp-uniformly: fn(valid, ord, idx).  Parked keys come from shared memory,
    // 4 in flight per thread; keys beyond the cache are recomputed from global memory (L2) with the same
    // batched, branch-free loads as the first pass.
    auto scan_cached = [&](auto&& fn) {
        const int n_c = min(span, cache_cap);
        for (int base = 0; base < n_c; base += kThreads * 4) {
            uint32_t o4[4], i4[4];
#pragma unroll
            for (int x = 0; x < 4; ++x) {
                const int j = base + x * kThreads + tid;
                i4[x] = j < n_c ? idx_of(j) : N;
                o4[x] = i4[x] < N ? cache[j] : 0u;
            }
#pragma unroll
            for (int x = 0; x < 4; ++x) fn(i4[x] < N, o4[x], i4[x]);
        }
    };
    auto scan_all = [&](auto&& fn) {
        scan_cached(fn);
        if (span <= cache_cap) return;
        if (vec) {
            for (int base4 = cache_cap >> 2; base4 < (span >> 2); base4 += kThreads * 4) {
                float4 lv[4];
                float sv[4];
                uint32_t ib[4];
#pragma unroll
                for (int x = 0; x < 4; ++x) {
                    const int j = 4 * (base4 + x * kThreads + tid);
                    const uint32_t id = j < span ? idx_of(j) : N;
                    ib[x] = id;
                    const uint32_t idc = min(id, N - 4);
                    const int row = c_shift >= 0 ? (int)(idc >> c_shift) : (int)(idc / (uint32_t)C);
                    lv[x] = __ldg(reinterpret_cast<const float4*>(lp + idc));
                    sv[x] = sc ? __ldg(sc + row) : 0.f;
                }
#pragma unroll
                for (int x = 0; x < 4; ++x) {
                    const bool ok = ib[x] < N;
                    fn(ok, ord_of(__fadd_rn(sv[x], lv[x].x)), ib[x]);
                    fn(ok, ord_of(__fadd_rn(sv[x], lv[x].y)), ib[x] + 1);
                    fn(ok, ord_of(__fadd_rn(sv[x], lv[x].z)), ib[x] + 2);
                    fn(ok, ord_of(__fadd_rn(sv[x], lv[x].w)), ib[x] + 3);
                }
            }
        } else {
            for (int base = cache_cap; base < span; base += kThreads * 4) {
                float lv[4], sv[4];
                uint32_t ib[4];
#pragma unroll
                for (int x = 0; x < 4; ++x) {
                    const int j = base + x * kThreads + tid;
                    const uint32_t id = j < span ? idx_of(j) : N;
                    ib[x] = id;
                    const uint32_t idc = min(id, N - 1);
                    const int row = c_shift >= 0 ? (int)(idc >> c_shift) : (int)(idc / (uint32_t)C);
                    lv[x] = __ldg(lp + idc);
                    sv[x] = sc ? __ldg(sc + row) : 0.f;
                }
#pragma unroll
                for (int x = 0; x < 4; ++x) fn(ib[x] < N, ord_of(__fadd_rn(sv[x], lv[x])), ib[x]);
            }
        }
    };

    // ---- radix select on V over the parked keys ----------------------------------------------------
    const uint32_t K = (uint32_t)W_out;
    uint32_t rem = K;                 // keys still to take from the candidate set
    unsigned long long pref = 0ull;   // value of V >> r shared by every candidate
    int r = nb + nbi;                 // unresolved low bits of V (<= 63)
    uint32_t cb = N;                  // candidates (= keys with V >> r == pref)

    // Survivor list: the streamed tail's survivors are already in it; the first pass adds the parked keys above
    // the bound.  If it overflows (heavy ties), every loop falls back to walking all keys (tail re-read via L2).
    const uint32_t n_tail = tail_streamed ? sh.sv_count : 0u;    // (complete: written before the cluster barrier)
    if (tail_streamed) __syncthreads();                          // read by everyone before the first pass appends
    bool use_sv = false;                             // later loops walk the survivor list instead of all keys
    uint32_t n_sv = 0;
#pragma unroll 1
    for (int pass = 0; (K - rem) + cb > (uint32_t)cap; ++pass) {  // same decision in every CTA
        const int arr = pass & 1;
        const int w = min(11, r), shift = r - w;
        const uint32_t mask = (1u << w) - 1u;
        if (use_sv) {
            for (uint32_t e = tid; e < n_sv; e += kThreads) {
                const uint2 k = sv[e];
                const unsigned long long v = vkey(k.x, k.y);
                if (k.x >= ord_lb && (v >> r) == pref) atomicAdd(&sh.hist[arr][(uint32_t)(v >> shift) & mask], 1u);
            }
        } else {
            if (pruning && pass == 0 && tail_ok) {
                // first pass of a pruned run: nearly every parked key fails the bound (one compare); the few
                // that pass enter the histogram and join the tail's survivors in the list
                for (uint32_t e = tid; e < n_tail; e += kThreads) {
                    const uint2 k = sv[e];
                    if (k.x >= ord_lb) atomicAdd(&sh.hist[arr][(uint32_t)(vkey(k.x, k.y) >> shift) & mask], 1u);
                }
                scan_cached([&](bool ok, uint32_t o, uint32_t idx) {
                    if (ok && o >= ord_lb) {
                        atomicAdd(&sh.hist[arr][(uint32_t)(vkey(o, idx) >> shift) & mask], 1u);
                        const uint32_t pos = atomicAdd(&sh.sv_count, 1u);
                        if (pos < (uint32_t)svcap) sv[pos] = make_uint2(o, idx);
                    }
                });
            } else {
                scan_all([&](bool ok, uint32_t o, uint32_t idx) {
                    if (!ok || o < ord_lb) return;
                    const unsigned long long v = vkey(o, idx);
                    if ((v >> r) == pref) atomicAdd(&sh.hist[arr][(uint32_t)(v >> shift) & mask], 1u);
                });
            }
        }
        __syncthreads();
        if (pruning && pass == 0 && tail_ok) {           // list complete?  else fall back to scanning all keys
            n_sv = sh.sv_count;
            use_sv = n_sv <= (uint32_t)svcap;
        }
        {   // coarse histogram: 32 fine bins = 8 threads x 4 bins
            const uint4 v = reinterpret_cast<const uint4*>(&sh.hist[arr][0])[tid];
            uint32_t s = v.x + v.y + v.z + v.w;
            s += __shfl_xor_sync(0xffffffffu, s, 1);
            s += __shfl_xor_sync(0xffffffffu, s, 2);
            s += __shfl_xor_sync(0xffffffffu, s, 4);
            if ((lane & 7) == 0) sh.coarse[arr][tid >> 3] = s;
        }
        cluster.sync();
        if (warp == 0) {
            // coarse counts of all ranks, one bin of each half per lane; ranks >= nc re-read this rank (ignored)
            uint32_t chi = 0, clo = 0;
            {
                uint32_t vh[kMaxCluster], vl[kMaxCluster];
#pragma unroll
                for (int rr = 0; rr < kMaxCluster; ++rr) {
                    const uint32_t* rc = cluster.map_shared_rank(&sh.coarse[arr][0], rr < nc ? rr : rank);
                    vh[rr] = rc[32 + lane]; vl[rr] = rc[lane];
                }
#pragma unroll
                for (int rr = 0; rr < kMaxCluster; ++rr)
                    if (rr < nc) { chi += vh[rr]; clo += vl[rr]; }
            }
            const uint32_t tot_hi = __reduce_add_sync(0xffffffffu, chi);
            const bool in_hi = rem <= tot_hi;
            int cbin; uint32_t rem2, ccnt;
            warp_select32(in_hi ? chi : clo, in_hi ? rem : rem - tot_hi, cbin, rem2, ccnt);
            const int coarse_bin = (in_hi ? 32 : 0) + cbin;
            // the 32 fine counters of that coarse bin, all ranks
            uint32_t f = 0;
            {
                uint32_t vf[kMaxCluster];
#pragma unroll
                for (int rr = 0; rr < kMaxCluster; ++rr) {
                    const uint32_t* rh = cluster.map_shared_rank(&sh.hist[arr][0], rr < nc ? rr : rank);
                    vf[rr] = rh[coarse_bin * 32 + lane];
                }
#pragma unroll
                for (int rr = 0; rr < kMaxCluster; ++rr)
                    if (rr < nc) f += vf[rr];
            }
            int fbin; uint32_t rem3, fcnt;
            warp_select32(f, rem2, fbin, rem3, fcnt);
            if (lane == 0) { sh.sel_bin = (uint32_t)(coarse_bin * 32 + fbin); sh.sel_rem = rem3; sh.sel_cnt = fcnt; }
        } else {
            // the other array was last read (remotely) before the readers arrived at this pass's barrier
            for (int b = tid - 32; b < kBins; b += kThreads - 32) sh.hist[arr ^ 1][b] = 0;
            if (tid - 32 < kCoarse) sh.coarse[arr ^ 1][tid - 32] = 0;
        }
        __syncthreads();
        pref = (pref << w) | (unsigned long long)sh.sel_bin;
        rem = sh.sel_rem;
        cb = sh.sel_cnt;
        r = shift;
        if (r == 0) break;  // V fully resolved: cb == 1 (all V distinct)
    }
    // Now: keys with (V >> r) > pref are selected (K - rem of them); `rem` more come from the `cb` keys with
    // (V >> r) == pref, and (K - rem) + cb <= cap: gather them all, the sort decides inside the boundary bin.
    auto take = [&](bool ok, uint32_t o, uint32_t idx) {
        const bool f = ok && o >= ord_lb && (vkey(o, idx) >> r) >= pref;
        const uint32_t bal = __ballot_sync(0xffffffffu, f);
        if (bal) {  // one shared-memory atomic per warp-iteration reserves the slots
            const int leader = __ffs(bal) - 1;
            uint32_t pos = 0;
            if (lane == leader) pos = atomicAdd(&sh.cursor, (uint32_t)__popc(bal));
            pos = __shfl_sync(0xffffffffu, pos, leader) + __popc(bal & ((1u << lane) - 1u));
            if (f && pos < (uint32_t)cap) sel[pos] = ((unsigned long long)(~o) << 32) | idx;
        }
    };
    if (use_sv) {
        for (uint32_t base = 0; base < n_sv; base += kThreads) {
            const uint32_t e = base + tid;
            const uint2 k = e < n_sv ? sv[e] : make_uint2(0u, N);
            take(e < n_sv, k.x, k.y);
        }
    } else {
        scan_all(take);
    }
    cluster.sync();

    // ---- CTA 0 pulls the other ranks' lists behind its own; the others wait until it has them ----------
    const int n_g = (int)min((K - rem) + cb, (uint32_t)cap);
    if (nc > 1) {
        if (rank == 0) {
            if (tid < nc) sh.list_len[tid] = *cluster.map_shared_rank(&sh.cursor, tid);
            __syncthreads();
            for (int e = (int)sh.list_len[0] + tid; e < n_g; e += kThreads) {
                int rr = 0, off = 0;
                while (rr < nc - 1 && e >= off + (int)sh.list_len[rr]) { off += (int)sh.list_len[rr]; ++rr; }
                sel[e] = cluster.map_shared_rank(sel, rr)[e - off];
            }
        }
        cluster.sync();
        if (rank != 0) return;
    }

    // ---- CTA 0: bitonic sort of the n_g composites, ascending (= key descending, index ascending) -----
    int S = 64;
    while (S < n_g) S <<= 1;
    for (int i = n_g + tid; i < S; i += kThreads) sel[i] = ~0ull;
    __syncthreads();
    if (n_g <= kRankSortMax) {
        // rank sort: position of a key = number of smaller keys (all composites are distinct).  Every thread
        // reads every key once, as shared-memory broadcasts; no barrier until the scatter.
        unsigned long long mine = 0ull;
        int rank_of = 0;
        if (tid < n_g) {
            mine = sel[tid];
#pragma unroll 8
            for (int i = 0; i < n_g; ++i) rank_of += sel[i] < mine;
        }
        __syncthreads();
        if (tid < n_g) sel[rank_of] = mine;
        __syncthreads();
    } else if (S <= kRegSortMax && cache_cap >= 2 * S) {
        // (1) every warp bitonic-sorts a run of 64 composites in registers: lane holds e0 = 64w + lane and
        //     e1 = e0 + 32; stride 32 is thread-local, smaller strides exchange by shuffle; no barrier.
        // (2) merge by ranking: final position = position in the own run + lower bounds in the other runs
        //     (binary searches over shared memory); the result goes to the dead key cache.
        const int n_runs = S >> 6;
        const int e0 = warp * 64 + lane, e1 = e0 + 32;
        unsigned long long a = ~0ull, b = ~0ull;
        if (warp < n_runs) {
            a = sel[e0]; b = sel[e1];
            for (int k = 2; k <= 64; k <<= 1) {
                for (int j = k >> 1; j > 0; j >>= 1) {
                    if (j == 32) {
                        if (a > b) { const unsigned long long t = a; a = b; b = t; }  // k = 64: ascending
                    } else {
                        const unsigned long long pa = __shfl_xor_sync(0xffffffffu, a, j);
                        const unsigned long long pb = __shfl_xor_sync(0xffffffffu, b, j);
                        const bool lower = (lane & j) == 0;
                        // directions from the position INSIDE the run (lane, lane + 32): every run ascending
                        const bool min_a = lower == ((lane & k) == 0), min_b = lower == (((lane + 32) & k) == 0);
                        a = min_a ? min(a, pa) : max(a, pa);
                        b = min_b ? min(b, pb) : max(b, pb);
                    }
                }
            }
            sel[e0] = a; sel[e1] = b;
        }
        __syncthreads();
        unsigned long long* dst = reinterpret_cast<unsigned long long*>(cache);
        if (warp < n_runs) {
            int ra = 0, rb = 0;                          // (the own run contributes the position inside it)
#pragma unroll 4
            for (int w2 = 0; w2 < n_runs; ++w2) {        // independent binary searches: unrolled for overlap
                const unsigned long long* run = sel + w2 * 64;
                int ca = 0, cb2 = 0;
#pragma unroll
                for (int st = 32; st > 0; st >>= 1) {
                    if (run[ca + st - 1] < a) ca += st;
                    if (run[cb2 + st - 1] < b) cb2 += st;
                }
                if (ca == 63 && run[63] < a) ca = 64;
                if (cb2 == 63 && run[63] < b) cb2 = 64;
                ra += ca; rb += cb2;
            }
            dst[ra] = a; dst[rb] = b;                    // composites are distinct: a permutation
        }
        __syncthreads();
        for (int i2 = tid; i2 < S; i2 += kThreads) sel[i2] = dst[i2];
        __syncthreads();
    } else {
        for (int k = 2; k <= S; k <<= 1) {
            for (int j = k >> 1; j > 0; j >>= 1) {
                for (int t = tid; t < (S >> 1); t += kThreads) {
                    const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));  // insert a 0 at bit log2(j)
                    const int ixj = i | j;
                    const bool up = (i & k) == 0;
                    const unsigned long long a = sel[i], b = sel[ixj];
                    if ((a > b) == up) { sel[i] = b; sel[ixj] = a; }
                }
                __syncthreads();
            }
        }
    }
    for (int rr = tid; rr < (int)K; rr += kThreads) {
        const uint32_t idx = min((uint32_t)sel[rr], N - 1);  // (clamp: memory safety on NaN-poisoned input)
        const int row = c_shift >= 0 ? (int)(idx >> c_shift) : (int)(idx / (uint32_t)C);
        const int code = (int)idx - row * C;
        const float s = sc ? __ldg(sc + row) : 0.f;
        out_score[(size_t)u * W_out + rr] = __fadd_rn(s, __ldg(lp + idx));
        out_parent[(size_t)u * W_out + rr] = row;
        out_code[(size_t)u * W_out + rr] = code;
    }
}

// ---- small problems (N <= kSmallMax candidates per user: decode step 0 of a 256-code level) ---------------
// One CTA per user, no cluster, no radix pass: every candidate's composite (~ord, idx) goes to shared memory,
// each thread counts how many composites are smaller than its own (shared-memory broadcasts) and the
// candidates of rank < W_out write their result row directly.  Same order as the general kernel: key
// descending, flat index ascending (reading R6).
constexpr int kSmallMax = 512;       // beyond this the N^2 / 2 compares cost more than the radix passes
constexpr int kSmallThreads = 256;

// kFold (W_in == 1 only: decode step 0, the user's single row IS the candidate set): the input holds RAW logits
// and the log-softmax normaliser is folded into the score here (reading R22, as logits_offset.cu does for
// general shapes): offset = fl32(score - fl32(logsumexp(row))), fp64 sum -- no separate launch.
template <int PER, bool kFold>  // candidates per thread
__global__ void __launch_bounds__(kSmallThreads)
topk_small_kernel(const float* __restrict__ logp, const float* __restrict__ score, int W_in, int C, int W_out,
                  float* __restrict__ out_score, int32_t* __restrict__ out_parent, int32_t* __restrict__ out_code) {
    __shared__ __align__(16) unsigned long long comp[PER * kSmallThreads];
    const int u = blockIdx.x, tid = threadIdx.x;
    const int N = W_in * C;
    const float* __restrict__ lp = logp + (size_t)u * N;
    const float* __restrict__ sc = score ? score + (size_t)u * W_in : nullptr;
    float key[PER];
    unsigned long long mine[PER];
    int row[PER], rk[PER];
#pragma unroll
    for (int x = 0; x < PER; ++x) {
        const int idx = min(tid + x * kSmallThreads, N - 1);
        row[x] = idx / C;
        key[x] = __ldg(lp + idx);
    }
    float fold_off = 0.f;
    if constexpr (kFold) {
        __shared__ float fm[kSmallThreads / 32];
        __shared__ double fs[kSmallThreads / 32];
        const float ninf = __int_as_float(0xff800000);
        float m = ninf;
#pragma unroll
        for (int x = 0; x < PER; ++x) if (tid + x * kSmallThreads < N) m = fmaxf(m, key[x]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
        if ((tid & 31) == 0) fm[tid >> 5] = m;
        __syncthreads();
        m = fm[0];
#pragma unroll
        for (int w = 1; w < kSmallThreads / 32; ++w) m = fmaxf(m, fm[w]);
        double s = 0.0;
        if (m != ninf) {
#pragma unroll
            for (int x = 0; x < PER; ++x)
                if (tid + x * kSmallThreads < N) s += exp((double)key[x] - (double)m);   // exp(-inf) = 0
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if ((tid & 31) == 0) fs[tid >> 5] = s;
        __syncthreads();
        s = fs[0];
#pragma unroll
        for (int w = 1; w < kSmallThreads / 32; ++w) s += fs[w];
        fold_off = m == ninf ? ninf : __fsub_rn(sc ? __ldg(sc) : 0.f, __double2float_rn((double)m + log(s)));
    }
#pragma unroll
    for (int x = 0; x < PER; ++x) {
        const int idx = tid + x * kSmallThreads;
        key[x] = __fadd_rn(kFold ? fold_off : (sc ? __ldg(sc + row[x]) : 0.f), key[x]);
        mine[x] = idx < N ? (((unsigned long long)(~ord_of(key[x])) << 32) | (uint32_t)idx) : ~0ull;
        comp[idx] = mine[x];
        rk[x] = 0;
    }
    __syncthreads();
    const int N2 = (N + 1) & ~1;                         // (a ragged last pair reads a dead slot: ~0, never smaller)
#pragma unroll 4
    for (int i = 0; i < N2; i += 2) {
        const ulonglong2 c = *reinterpret_cast<const ulonglong2*>(comp + i);  // broadcast
#pragma unroll
        for (int x = 0; x < PER; ++x) rk[x] += (int)(c.x < mine[x]) + (int)(c.y < mine[x]);
    }
#pragma unroll
    for (int x = 0; x < PER; ++x) {
        const int idx = tid + x * kSmallThreads;
        if (idx < N && rk[x] < W_out) {
            const size_t o = (size_t)u * W_out + rk[x];
            out_score[o] = key[x];
            out_parent[o] = row[x];
            out_code[o] = idx - row[x] * C;
        }
    }
}

// ---- medium problems (kSmallMax < N <= kMidMaxN candidates per user, W_out <= kMidMaxK) ---------------------
// One 1024-thread CTA per user, 16 candidates per thread, no cluster: at these sizes (config 2: 16 K candidates,
// W_out = 64) the general kernel's time is its chain of cluster barriers and DSMEM pulls, not its data.
//   1. load once; the order-preserving keys are parked in shared memory (64 KB);
//   2. bound: if K of the 1024 per-thread maxima lie in 11-bit bins >= b, at least K keys do, so the W_out-th key
//      cannot lie below bin b (the pruning argument of the general kernel): one tiny histogram of 1024 values;
//   3. the candidates at or above the bound (normally W_out plus a few) go to a list; each list entry counts the
//      entries smaller than itself and the ranks < W_out write their result rows -- no sort;
//   4. more than 1024 survivors (massive ties): exact radix select of the W_out-th key over the parked keys
//      (up to three 11-bit passes), keys above it plus the lowest-index keys equal to it (index-order prefix
//      counts) form the list; then step 3's ranking.
constexpr int kMidThreads = 1024;
constexpr int kMidKeysPerThread = 16;
constexpr int kMidMaxN = kMidThreads * kMidKeysPerThread;
constexpr int kMidMaxK = 1024;       // capacity of the list (the kernel is exact up to here)
constexpr int kMidUseK = 256;        // ... but it is dispatched only where it was measured to win

struct __align__(16) MidShared {
    uint32_t hist[kBins];
    uint32_t coarse[kCoarse];          // (directly behind hist: zeroed together)
    uint32_t wred[2][32];
    uint32_t sel_bin, sel_rem, sel_cnt, cursor, cursor2, pad[3];
    unsigned long long list[kMidMaxK];
};

// warp 0: highest bin of sh.hist with suffix count >= rem (requires the total >= rem)
__device__ __forceinline__ void mid_select(MidShared& sh, uint32_t rem) {
    const int lane = threadIdx.x & 31;
    const uint32_t cu = sh.coarse[32 + lane], cl = sh.coarse[lane];
    uint32_t tot_u = cu;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tot_u += __shfl_xor_sync(0xffffffffu, tot_u, o);
    int g, b;
    uint32_t r2, c2, r3, c3;
    if (tot_u >= rem) { warp_select32(cu, rem, g, r2, c2); g += 32; }
    else warp_select32(cl, rem - tot_u, g, r2, c2);
    warp_select32(sh.hist[32 * g + lane], r2, b, r3, c3);
    if (lane == 0) { sh.sel_bin = (uint32_t)(32 * g + b); sh.sel_rem = r3; sh.sel_cnt = c3; }
}

template <int kMidKeys>  // candidates per thread
__global__ void __launch_bounds__(kMidThreads, 1)
topk_mid_kernel(const float* __restrict__ logp, const float* __restrict__ score, int W_in, int C, int c_shift,
                int W_out, float* __restrict__ out_score, int32_t* __restrict__ out_parent,
                int32_t* __restrict__ out_code) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t* ords = reinterpret_cast<uint32_t*>(smem_raw);        // [kMidThreads * kMidKeys]
    __shared__ MidShared sh;
    const int u = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t N = (uint32_t)(W_in * C), K = (uint32_t)W_out;
    const float* __restrict__ lp = logp + (size_t)u * N;
    const float* __restrict__ sc = score ? score + (size_t)u * W_in : nullptr;

    for (int b = tid; b < kBins + kCoarse; b += kMidThreads) sh.hist[b] = 0;   // hist + coarse
    if (tid == 0) { sh.cursor = 0; sh.cursor2 = 0; }

    // ---- 1. load: 16 log-prob loads of a thread in flight at once (one cold round trip per 16 K candidates);
    // the parent scores (a few cache lines per user) follow and hit L1 ----------------------------------------
    uint32_t tmax = 0u, tmin = 0xffffffffu;
#pragma unroll
    for (int h = 0; h < kMidKeys / 16; ++h) {
        float lv[16];
#pragma unroll
        for (int x = 0; x < 16; ++x) lv[x] = __ldg(lp + min((uint32_t)(tid + kMidThreads * (16 * h + x)), N - 1));
#pragma unroll
        for (int x = 0; x < 16; ++x) {
            const uint32_t idx = (uint32_t)(tid + kMidThreads * (16 * h + x)), idc = min(idx, N - 1);
            const int row = c_shift >= 0 ? (int)(idc >> c_shift) : (int)(idc / (uint32_t)C);
            const uint32_t o = ord_of(__fadd_rn(sc ? __ldg(sc + row) : 0.f, lv[x]));
            ords[idx] = o;
            if (idx < N) { tmax = max(tmax, o); tmin = min(tmin, o); }
        }
    }
    uint32_t mx = tmax, mn = tmin;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o));
    }
    if (lane == 0) { sh.wred[0][warp] = mx; sh.wred[1][warp] = mn; }
    __syncthreads();
    mx = sh.wred[0][lane]; mn = sh.wred[1][lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o));
    }
    const uint32_t span_v = mx - mn;
    const int nbits = span_v ? 32 - __clz(span_v) : 0;
    const int sh1 = max(nbits - 11, 0);                            // shift of the top 11-bit digit of (ord - mn)

    // ---- 2. bound from the per-thread maxima ------------------------------------------------------------
    if ((uint32_t)tid < N) {
        const uint32_t b = (tmax - mn) >> sh1;
        atomicAdd(&sh.hist[b], 1u);
        atomicAdd(&sh.coarse[b >> 5], 1u);
    }
    __syncthreads();
    const uint32_t n_thr = min((uint32_t)kMidThreads, N);          // threads that hold at least one candidate
    if (warp == 0) {
        if (K <= n_thr) mid_select(sh, K);
        else if (lane == 0) sh.sel_bin = 0;
    }
    __syncthreads();
    const uint32_t lb = mn + (sh.sel_bin << sh1);

    auto append = [&](uint32_t* cursor, bool f, uint32_t o, uint32_t idx) {
        const uint32_t bal = __ballot_sync(0xffffffffu, f);
        if (bal) {
            const int leader = __ffs(bal) - 1;
            uint32_t pos = 0;
            if (lane == leader) pos = atomicAdd(cursor, (uint32_t)__popc(bal));
            pos = __shfl_sync(0xffffffffu, pos, leader) + __popc(bal & ((1u << lane) - 1u));
            if (f && pos < (uint32_t)kMidMaxK) sh.list[pos] = ((unsigned long long)(~o) << 32) | idx;
        }
    };

    // ---- 3. survivors ------------------------------------------------------------------------------------
#pragma unroll 4
    for (int j = 0; j < kMidKeys; ++j) {
        const uint32_t idx = (uint32_t)(tid + kMidThreads * j);
        const uint32_t o = ords[idx];
        append(&sh.cursor, idx < N && o >= lb, o, idx);
    }
    __syncthreads();
    uint32_t n_list = sh.cursor;

    if (n_list > (uint32_t)kMidMaxK) {
        // ---- 4. exact selection: value T of the K-th largest (ord - mn), then ties by index ---------------
        uint32_t pref = 0, rem = K;
        int shift_prev = 32, width = min(11, nbits), shift = nbits - width;   // first digit: the top `width` bits
        bool first = true;
        while (true) {
            for (int b = tid; b < kBins + kCoarse; b += kMidThreads) sh.hist[b] = 0;
            __syncthreads();
#pragma unroll 4
            for (int j = 0; j < kMidKeys; ++j) {
                const uint32_t idx = (uint32_t)(tid + kMidThreads * j);
                const uint32_t v = ords[idx] - mn;
                if (idx < N && (first || (v >> shift_prev) == pref)) {
                    const uint32_t dgt = (v >> shift) & ((1u << width) - 1u);
                    atomicAdd(&sh.hist[dgt], 1u);
                    atomicAdd(&sh.coarse[dgt >> 5], 1u);
                }
            }
            __syncthreads();
            if (warp == 0) mid_select(sh, rem);
            __syncthreads();
            pref = (pref << width) | sh.sel_bin;
            rem = sh.sel_rem;
            first = false;
            shift_prev = shift;
            if (shift == 0) break;
            width = min(11, shift);
            shift -= width;
        }
        const uint32_t T = pref, need = rem;                       // keys > T: K - need; `need` of the keys == T
        uint32_t tie_base = 0;                                     // (the list is rebuilt from entry 0: cursor2)
        for (int j = 0; j < kMidKeys; ++j) {                       // index order: j major, thread minor
            const uint32_t idx = (uint32_t)(tid + kMidThreads * j);
            const uint32_t o = ords[idx];
            const uint32_t v = o - mn;
            const bool live = idx < N;
            const bool eq = live && v == T;
            const uint32_t bal = __ballot_sync(0xffffffffu, eq);
            if (lane == 0) sh.wred[j & 1][warp] = (uint32_t)__popc(bal);
            __syncthreads();
            uint32_t inc = sh.wred[j & 1][lane];                   // inclusive prefix over the warps
#pragma unroll
            for (int o2 = 1; o2 < 32; o2 <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o2);
                if (lane >= o2) inc += t;
            }
            const uint32_t before_warp = __shfl_sync(0xffffffffu, inc, warp) - __shfl_sync(0xffffffffu, sh.wred[j & 1][lane], warp);
            const uint32_t total = __shfl_sync(0xffffffffu, inc, 31);
            const uint32_t pos = tie_base + before_warp + (uint32_t)__popc(bal & ((1u << lane) - 1u));
            append(&sh.cursor2, (live && v > T) || (eq && pos < need), o, idx);
            tie_base += total;
        }
        __syncthreads();
        n_list = sh.cursor2;                                       // == K
    }

    // ---- ranking by counting: composites are distinct; ranks < K are the result, in order ---------------
    n_list = min(n_list, (uint32_t)kMidMaxK);
    if ((uint32_t)tid < n_list) {
        const unsigned long long mine = sh.list[tid];
        uint32_t rk = 0;
        const uint32_t n2 = n_list & ~1u;
#pragma unroll 4
        for (uint32_t i = 0; i < n2; i += 2) {
            const ulonglong2 c = *reinterpret_cast<const ulonglong2*>(&sh.list[i]);   // broadcast
            rk += (uint32_t)(c.x < mine) + (uint32_t)(c.y < mine);
        }
        if (n_list & 1u) rk += (uint32_t)(sh.list[n_list - 1] < mine);
        if (rk < K) {
            const uint32_t idx = min((uint32_t)mine, N - 1);
            const int row = c_shift >= 0 ? (int)(idx >> c_shift) : (int)(idx / (uint32_t)C);
            const size_t o = (size_t)u * W_out + rk;
            out_score[o] = __fadd_rn(sc ? __ldg(sc + row) : 0.f, __ldg(lp + idx));
            out_parent[o] = row;
            out_code[o] = (int)idx - row * C;
        }
    }
}

int next_pow2(int x) { int p = 1; while (p < x) p <<= 1; return p; }

}  // namespace

size_t topk_workspace_bytes(int B, int W_in, int C) { return topk_grid_workspace_bytes(B, W_in, C); }

bool topk_can_fold_lse(int W_in, int C) { return W_in == 1 && C <= kSmallMax; }

int launch_topk(const float* logp, const float* score, int B, int W_in, int C, int W_out,
                float* out_score, int32_t* out_parent, int32_t* out_code, void* ws, size_t ws_bytes,
                cudaStream_t st, bool fold_lse) {
    const long long N = (long long)W_in * C;
    if (fold_lse && !topk_can_fold_lse(W_in, C)) return STARK_ERR_INVALID_ARG;
    if (N <= kSmallMax) {
        if (fold_lse) {
            if (N <= kSmallThreads)
                topk_small_kernel<1, true><<<B, kSmallThreads, 0, st>>>(logp, score, W_in, C, W_out, out_score, out_parent, out_code);
            else
                topk_small_kernel<2, true><<<B, kSmallThreads, 0, st>>>(logp, score, W_in, C, W_out, out_score, out_parent, out_code);
        } else if (N <= kSmallThreads)
            topk_small_kernel<1, false><<<B, kSmallThreads, 0, st>>>(logp, score, W_in, C, W_out, out_score, out_parent, out_code);
        else
            topk_small_kernel<2, false><<<B, kSmallThreads, 0, st>>>(logp, score, W_in, C, W_out, out_score, out_parent, out_code);
        STARK_LAUNCH_CHECK();
        return STARK_OK;
    }
    // (measured: W_out = 512 of 8192 candidates, 20 us against 15 us for the cluster kernel; 32 K candidates with
    // 32 per thread, 13.1 against 12.8 us: two cold load rounds)
    if (N <= kMidMaxN && W_out <= kMidUseK) {
        static PerDevice<bool> mid_attr;
        bool& mid_attr_done = mid_attr.here();
        if (!mid_attr_done) {
            STARK_CUDA_TRY(cudaFuncSetAttribute(topk_mid_kernel<kMidKeysPerThread>,
                                                cudaFuncAttributeMaxDynamicSharedMemorySize, kMidMaxN * 4));
            mid_attr_done = true;
        }
        int c_sh = -1;
        if ((C & (C - 1)) == 0) { c_sh = 0; while ((1 << c_sh) < C) ++c_sh; }
        topk_mid_kernel<kMidKeysPerThread><<<B, kMidThreads, kMidMaxN * 4, st>>>(logp, score, W_in, C, c_sh, W_out,
                                                                                 out_score, out_parent, out_code);
        STARK_LAUNCH_CHECK();
        return STARK_OK;
    }
    // wide selections over small candidate sets (decode step 0 with a wide beam): independent CTAs, no cluster
    if (topk_wide_serves(N, W_out)) {
        const int rc = launch_topk_wide(logp, score, B, W_in, C, W_out, out_score, out_parent, out_code, st);
        if (rc != STARK_ERR_UNSUPPORTED) return rc;
    }
    // large candidate sets: the whole GPU on every user (topk_grid.cu); UNSUPPORTED = shape not served there
    if (ws) {
        const int rc = launch_topk_grid(logp, score, B, W_in, C, W_out, out_score, out_parent, out_code, ws, ws_bytes, st);
        if (rc != STARK_ERR_UNSUPPORTED) return rc;
    }
    const int cap = next_pow2(W_out) * 2 < 128 ? 128 : next_pow2(W_out) * 2;  // sort buffer entries
    // pruning pays once a thread holds many keys (>= 16: slices of 8192) and needs K <= the 2048 buckets of a CTA
    int prune = (N / kMaxCluster >= 8192 || N >= 32768) && W_out <= 2048 ? 1 : 0;
    auto fixed_bytes = [&](int pr) {  // Shared + sel (+ the two survivor lists of 4 * cap entries when pruning)
        return ((sizeof(Shared) + 15) / 16) * 16 + (size_t)cap * 8 * (pr ? 9 : 1);
    };
    // the survivor lists of a wide selection (1024 < W_out <= 2048: cap = 4096, 288 KB) do not fit next to a
    // useful key cache: select without pruning then (the slice beyond the cache is re-read through L2)
    if (prune && (long long)kSmemBudget - (long long)fixed_bytes(1) < (long long)kMinCacheKeys * 4) prune = 0;
    const size_t fixed = fixed_bytes(prune);
    const long long cache_max = ((long long)kSmemBudget - (long long)fixed) / 4;
    if (cache_max < kMinCacheKeys) return STARK_ERR_UNSUPPORTED;  // (unreachable for W_out <= 4096)
    static PerDevice<bool> attr;  // idempotent; a benign race at worst repeats the calls
    bool& attr_done = attr.here();
    if (!attr_done) {
        STARK_CUDA_TRY(cudaFuncSetAttribute(topk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBudget));
        STARK_CUDA_TRY(cudaFuncSetAttribute(topk_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        attr_done = true;
    }
    // cluster size: split a user over more CTAs while slices stay >= kSliceMin -- but never more clusters
    // than the device can keep resident at once (a second wave would double the latency): B200 co-schedules
    // only 15 clusters of 8 CTAs, so the occupancy API decides, not SMs / cluster size.
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(kThreads);
    cfg.stream = st;
    cfg.attrs = at; cfg.numAttrs = 1;
    int nc = 1, cache_cap = 0;
    auto configure = [&](int n) {
        const long long slice = ((N + kChunk - 1) / kChunk + n - 1) / n * kChunk;  // whole chunks
        cache_cap = (int)(slice < cache_max ? slice : cache_max) & ~3;  // whole 16-byte groups
        cfg.gridDim = dim3((unsigned)(B * n));
        cfg.dynamicSmemBytes = fixed + (size_t)cache_cap * 4;
        at[0].val.clusterDim.x = n;
    };
    auto max_clusters = [&](int n) -> int {  // resident clusters of size n with the current smem; cached
        struct Memo { int smem[5], val[5]; };
        static PerDevice<Memo> memo;  // (zero-initialised: no launch has 0 bytes of dynamic shared memory)
        int* memo_smem = memo.here().smem;
        int* memo_val = memo.here().val;
        int slot = 0;
        while ((1 << slot) < n) ++slot;
        if (memo_smem[slot] != (int)cfg.dynamicSmemBytes) {
            int v = 0;
            if (cudaOccupancyMaxActiveClusters(&v, topk_kernel, &cfg) != cudaSuccess) { (void)cudaGetLastError(); v = 0; }
            memo_smem[slot] = (int)cfg.dynamicSmemBytes; memo_val[slot] = v;
        }
        return memo_val[slot];
    };
    configure(1);
    while (nc < kMaxCluster && (N + nc - 1) / nc > kSliceMin) {
        configure(nc * 2);
        if (max_clusters(nc * 2) < B) break;
        nc *= 2;
    }
    configure(nc);
    int c_shift = -1;
    if ((C & (C - 1)) == 0) { c_shift = 0; while ((1 << c_shift) < C) ++c_shift; }
    STARK_CUDA_TRY(cudaLaunchKernelEx(&cfg, topk_kernel, logp, score, W_in, C, c_shift, W_out, out_score,
                                      out_parent, out_code, cache_cap, cap, prune));
    return STARK_OK;
}

}  // namespace stark
