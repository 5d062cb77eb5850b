// A3: stark_beam_topk -- per-level beam selection, bit-exact and deterministic.
//
// Beam score = sum of per-level log-probabilities (Eq. 1);
// each level keeps the top-W candidate paths.  Per user:
//   key[i*C + c] = fl32(score[i] + logp[i, c])          (one fp32 add, reading R4)
//   keep the W_out entries first in (key descending, flat index ascending)
//   (reading R6), output sorted in that order.
//
// The work is tiny next to its latency (1 MB per level at config 2), so the
// design minimises the number of dependent phases rather than instructions:
//   load     one thread-block CLUSTER per user; every CTA streams its
//            contiguous slice of the user's candidates ONCE from HBM, maps each
//            key to an order-preserving uint32 `ord`, parks it in shared memory
//            and tracks the slice's (max, min) ord in registers.
//   range    the cluster-wide (max, min) -- exchanged through distributed shared
//            memory -- gives the highest bit `hb` in which any two keys differ.
//            Radix digits are taken from bit hb downwards, so the first
//            histogram already separates the keys (raw float bits would put
//            nearly every log-probability into a handful of exponent bins).
//   select   <= 3 radix passes of 11 bits over the parked keys: shared-memory
//            histogram, cluster barrier, every CTA pulls all ranks' histograms
//            (one 16-byte DSMEM load per rank per thread) and runs the same
//            suffix scan, so no broadcast is needed.  The loop stops as soon as
//            "keys above the boundary bin + keys inside it" fits the sort
//            buffer -- typically after the first or second pass.
//   gather   those keys are appended as 64-bit composites (~ord, idx) to CTA 0's
//            shared memory (warp-aggregated DSMEM atomics reserve the slots).
//   sort     CTA 0 bitonic-sorts them -- a strict total order, so the result
//            does not depend on arrival order and ties at the boundary resolve
//            by index for free -- and writes the first W_out as (score, parent,
//            code), recomputing score with the same fp32 add.
//   ties     only if the boundary VALUE itself occurs more often than the sort
//            buffer can hold (e.g. thousands of -inf or quantised keys) are the
//            equal keys counted per CTA and taken in index order explicitly.
// Algorithmic HBM bytes: 4 per candidate (read once) + 4 per input beam + 12
// per selected beam.  Slice tails beyond the
// shared-memory cache (paper-scale codebooks) are re-read through L2.
#include <cooperative_groups.h>
#include <cstdlib>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace stark {

namespace {

constexpr int kThreads = 512;
constexpr int kWarps = kThreads / 32;
constexpr int kUnroll = 8;
constexpr int kBins = 2048;           // 11-bit digits
constexpr int kBpt = kBins / kThreads;  // bins per thread in the scan (4 = one uint4)
constexpr int kMaxOut = 4096;         // W_out limit
constexpr int kMaxCluster = 16;       // non-portable size, used only when the device can co-schedule it
constexpr int kSliceMin = 2048;       // do not split a user into slices smaller than this
constexpr int kSmemBudget = 227 * 1024;

struct Shared {
    uint32_t hist[3][kBins];
    uint32_t warp_tot[kWarps];
    uint32_t warp_max[kWarps], warp_min[kWarps];
    uint32_t sel_bin, sel_rem, sel_cnt;
    uint32_t cta_max, cta_min;     // this CTA's slice (read remotely)
    uint32_t all_max, all_min;     // cluster-wide
    uint32_t n_gt, n_eq;           // tie path: this CTA's counts (read remotely)
    uint32_t cursor;               // CTA 0: next free slot of the sort buffer (remote atomics)
    uint32_t eq_cursor, scan_base;
};

__device__ __forceinline__ uint32_t ord_of(float key) {
    uint32_t b = __float_as_uint(key);
    if (b == 0x80000000u) b = 0u;  // -0.0 == +0.0 (IEEE comparison, reading R6)
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

// Block-wide: find the largest bin b with  sum_{b' >= b} g(b') >= rem.
// Thread t passes the counts of bins (kThreads-1-t)*kBpt .. +kBpt-1 (thread 0 owns the highest bins).
// Result in sh.sel_bin / sh.sel_rem (= rem minus the count in bins above sel_bin) / sh.sel_cnt (= count
// inside sel_bin).  Requires total >= rem (guaranteed by the callers); contains two block barriers.
__device__ __forceinline__ void block_select(Shared& sh, const uint32_t (&cnt)[kBpt], uint32_t rem) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t mine = 0;
#pragma unroll
    for (int j = 0; j < kBpt; ++j) mine += cnt[j];
    uint32_t inc = mine;  // inclusive scan over threads (thread 0 = highest bins)
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) sh.warp_tot[warp] = inc;
    __syncthreads();
    uint32_t wbase = 0;
    {
        const uint32_t w = lane < kWarps ? sh.warp_tot[lane] : 0;
        uint32_t winc = w;
#pragma unroll
        for (int o = 1; o < kWarps; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += t;
        }
        wbase = __shfl_sync(0xffffffffu, winc - w, warp);
    }
    uint32_t before = wbase + inc - mine;  // keys in bins above this thread's bins
    if (before < rem && rem <= before + mine) {
        // the crossing is inside my bins: walk them from the highest down
        const int top = (kThreads - 1 - tid) * kBpt + (kBpt - 1);
#pragma unroll
        for (int j = 0; j < kBpt; ++j) {
            const uint32_t c = cnt[kBpt - 1 - j];
            if (before < rem && rem <= before + c) { sh.sel_bin = top - j; sh.sel_rem = rem - before; sh.sel_cnt = c; }
            before += c;
        }
    }
    __syncthreads();
}

__device__ __forceinline__ uint32_t shr32(uint32_t v, int s) { return s >= 32 ? 0u : v >> s; }

__global__ void __launch_bounds__(kThreads, 1)
topk_kernel(const float* __restrict__ logp, const float* __restrict__ score, int W_in, int C, int c_shift,
            int W_out, float* __restrict__ out_score, int32_t* __restrict__ out_parent,
            int32_t* __restrict__ out_code, int cache_cap, int cap) {
    cg::cluster_group cluster = cg::this_cluster();
    const int nc = (int)cluster.num_blocks();
    const int rank = (int)cluster.block_rank();
    const int u = blockIdx.x / nc;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    Shared& sh = *reinterpret_cast<Shared*>(smem_raw);
    unsigned long long* sel = reinterpret_cast<unsigned long long*>(smem_raw + ((sizeof(Shared) + 15) / 16) * 16);
    uint32_t* cache = reinterpret_cast<uint32_t*>(sel + cap);

    const long long N = (long long)W_in * C;
    const long long slice = (N + nc - 1) / nc;
    const long long lo = min(N, (long long)rank * slice);
    const long long hi = min(N, lo + slice);
    const int n_local = (int)(hi - lo);
    const float* __restrict__ lp = logp + (size_t)u * N;
    const float* __restrict__ sc = score ? score + (size_t)u * W_in : nullptr;

    auto key_ord = [&](int j) -> uint32_t {  // j: index inside the slice
        const uint32_t idx = (uint32_t)(lo + j);  // N < 2^31 (validated by the API)
        const int row = c_shift >= 0 ? (int)(idx >> c_shift) : (int)(idx / (uint32_t)C);
        const float s = sc ? __ldg(sc + row) : 0.f;
        return ord_of(__fadd_rn(s, __ldg(lp + idx)));
    };
    auto ord_at = [&](int j) -> uint32_t { return j < cache_cap ? cache[j] : key_ord(j); };

    for (int b = tid; b < 3 * kBins; b += kThreads) (&sh.hist[0][0])[b] = 0;
    if (tid == 0) { sh.n_gt = 0; sh.n_eq = 0; sh.cursor = 0; sh.eq_cursor = 0; sh.scan_base = 0; }

    // ---- load: the one pass over HBM ---------------------------------------------------
    uint32_t mx = 0u, mn = 0xffffffffu;
    for (int base = 0; base < n_local; base += kThreads * kUnroll) {
        uint32_t o[kUnroll];
#pragma unroll
        for (int x = 0; x < kUnroll; ++x) {
            const int j = base + x * kThreads + tid;
            o[x] = j < n_local ? key_ord(j) : 0u;
        }
#pragma unroll
        for (int x = 0; x < kUnroll; ++x) {
            const int j = base + x * kThreads + tid;
            if (j < n_local) {
                if (j < cache_cap) cache[j] = o[x];
                mx = max(mx, o[x]); mn = min(mn, o[x]);
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

    // ---- range: highest bit in which any two keys of this user differ ------------------------
    {
        uint32_t a = 0u, b = 0xffffffffu;
        if (lane < nc) {
            a = *cluster.map_shared_rank(&sh.cta_max, lane);
            b = *cluster.map_shared_rank(&sh.cta_min, lane);
        }
        mx = __reduce_max_sync(0xffffffffu, a);
        mn = __reduce_min_sync(0xffffffffu, b);
    }
    const int nb = (mx == mn) ? 0 : 32 - __clz((int)(mx ^ mn));  // low bits that can differ
    const int npass = (nb + 10) / 11;

    // ---- radix select over the parked keys ----------------------------------------------------
    const uint32_t K = (uint32_t)W_out;
    uint32_t rem = K;                    // keys still to take from the candidate set
    uint32_t pref = shr32(mx, nb);       // value of ord >> r shared by every candidate
    int r = nb;                          // unresolved low bits
    uint32_t cb = (uint32_t)N;           // candidates (= keys whose ord >> r == pref)
#pragma unroll 1
    for (int pass = 0; pass < npass; ++pass) {
        const int w = min(11, r), shift = r - w;
        const uint32_t mask = (1u << w) - 1u;
        for (int j = tid; j < n_local; j += kThreads) {
            const uint32_t o = ord_at(j);
            if (shr32(o, r) == pref) atomicAdd(&sh.hist[pass][(o >> shift) & mask], 1u);
        }
        cluster.sync();
        uint32_t cnt[kBpt] = {0u, 0u, 0u, 0u};
        {
            // all ranks' loads in flight together (a DSMEM load takes ~200 cycles); ranks >= nc re-read rank 0
            uint4 v[kMaxCluster];
#pragma unroll
            for (int rr = 0; rr < kMaxCluster; ++rr) {
                const uint4* rh = reinterpret_cast<const uint4*>(cluster.map_shared_rank(&sh.hist[pass][0], rr < nc ? rr : 0));
                v[rr] = rh[kThreads - 1 - tid];
            }
#pragma unroll
            for (int rr = 0; rr < kMaxCluster; ++rr)
                if (rr < nc) { cnt[0] += v[rr].x; cnt[1] += v[rr].y; cnt[2] += v[rr].z; cnt[3] += v[rr].w; }
        }
        block_select(sh, cnt, rem);
        pref = (pref << w) | sh.sel_bin;
        rem = sh.sel_rem;
        cb = sh.sel_cnt;
        r = shift;
        if ((K - rem) + cb <= (uint32_t)cap) break;  // same decision in every CTA: they scanned the same counts
    }
    // Now: keys with (ord >> r) > pref are selected (K - rem of them); `rem` more come from the `cb` keys
    // with (ord >> r) == pref.
    const uint32_t n_above = K - rem;
    unsigned long long* sel0 = cluster.map_shared_rank(sel, 0);
    const bool simple = n_above + cb <= (uint32_t)cap;

    // append f-flagged keys of this thread to THIS CTA's list (sel[0 .. sh.cursor)); one shared-memory
    // atomic per warp-iteration.  CTA 0 pulls every rank's list after the cluster barrier: remote atomics
    // and scattered remote stores from every CTA were measured ~8x slower than one bulk pull.
    auto append = [&](bool f, uint32_t o, int j) {
        const uint32_t bal = __ballot_sync(0xffffffffu, f);
        if (bal) {
            const int leader = __ffs(bal) - 1;
            uint32_t pos = 0;
            if (lane == leader) pos = atomicAdd(&sh.cursor, (uint32_t)__popc(bal));
            pos = __shfl_sync(0xffffffffu, pos, leader);
            if (f) sel[pos + __popc(bal & ((1u << lane) - 1u))] = ((unsigned long long)(~o) << 32) | (uint32_t)(lo + j);
        }
    };

    if (simple) {
        // gather "above" and the whole boundary bin; the sort decides inside the bin (ties by index)
        for (int base = 0; base < n_local; base += kThreads) {
            const int j = base + tid;
            const uint32_t o = j < n_local ? ord_at(j) : 0u;
            append(j < n_local && shr32(o, r) >= pref, o, j);
        }
    } else {
        // ---- ties: the boundary VALUE T (r == 0 here) occurs more often than the buffer holds ----
        const uint32_t T = pref, need_eq = rem;
        uint32_t cg_ = 0, ce_ = 0;
        for (int j = tid; j < n_local; j += kThreads) {
            const uint32_t o = ord_at(j);
            cg_ += o > T; ce_ += o == T;
        }
        cg_ = __reduce_add_sync(0xffffffffu, cg_);
        ce_ = __reduce_add_sync(0xffffffffu, ce_);
        if (lane == 0) { atomicAdd(&sh.n_gt, cg_); atomicAdd(&sh.n_eq, ce_); }
        cluster.sync();
        uint32_t eq_before = 0;
        for (int rr = 0; rr < rank; ++rr) eq_before += *cluster.map_shared_rank(&sh.n_eq, rr);
        const uint32_t my_eq = sh.n_eq;
        // 0: take none of my equals, 1: take all (any order), 2: boundary CTA (index order)
        const int eq_mode = eq_before >= need_eq ? 0 : (eq_before + my_eq <= need_eq ? 1 : 2);
        for (int base = 0; base < n_local; base += kThreads) {
            const int j = base + tid;
            const uint32_t o = j < n_local ? ord_at(j) : 0u;
            append(j < n_local && o > T, o, j);  // slots [0, n_above)
            if (j < n_local && o == T && eq_mode == 1)
                sel0[n_above + eq_before + atomicAdd(&sh.eq_cursor, 1u)] = ((unsigned long long)(~o) << 32) | (uint32_t)(lo + j);
        }
        if (eq_mode == 2) {
            // ordered: the first (need_eq - eq_before) equals of this slice, by index
            const uint32_t want = need_eq - eq_before;
            for (int base = 0; base < n_local; base += kThreads) {
                const uint32_t taken = sh.scan_base;
                if (taken >= want) break;  // uniform: read after a barrier
                const int j = base + tid;
                const uint32_t o = j < n_local ? ord_at(j) : 0u;
                const bool f = j < n_local && o == T;
                const uint32_t bal = __ballot_sync(0xffffffffu, f);
                if (lane == 0) sh.warp_tot[warp] = __popc(bal);
                __syncthreads();
                uint32_t wb = 0, tot = 0;
                for (int w2 = 0; w2 < kWarps; ++w2) {
                    const uint32_t c = sh.warp_tot[w2];
                    wb += w2 < warp ? c : 0;
                    tot += c;
                }
                const uint32_t rnk = taken + wb + __popc(bal & ((1u << lane) - 1u));
                if (f && rnk < want)
                    sel0[n_above + eq_before + rnk] = ((unsigned long long)(~o) << 32) | (uint32_t)(lo + j);
                __syncthreads();
                if (tid == 0) sh.scan_base = taken + tot;
                __syncthreads();
            }
        }
    }
    cluster.sync();
    // ---- CTA 0 pulls the other ranks' lists behind its own; the others wait until it has them ----------
    const int n_g = simple ? (int)(n_above + cb) : (int)K;
    if (rank == 0 && nc > 1) {
        if (tid < nc) sh.warp_tot[tid] = *cluster.map_shared_rank(&sh.cursor, tid);  // list lengths (nc <= 16)
        __syncthreads();
        const int n_lists = simple ? n_g : (int)n_above;  // tie path: equals were written in place
        for (int e = (int)sh.warp_tot[0] + tid; e < n_lists; e += kThreads) {
            int rr = 0, off = 0;
            while (rr < nc - 1 && e >= off + (int)sh.warp_tot[rr]) { off += (int)sh.warp_tot[rr]; ++rr; }
            sel[e] = cluster.map_shared_rank(sel, rr)[e - off];
        }
    }
    if (nc > 1) cluster.sync();
    if (rank != 0) return;

    // ---- CTA 0: bitonic sort of the gathered composites, ascending ------------------------------
    int sort_n = 2;
    while (sort_n < n_g) sort_n <<= 1;
    for (int i = n_g + tid; i < sort_n; i += kThreads) sel[i] = ~0ull;
    __syncthreads();
    if (sort_n <= 64) {
        if (warp == 0) {  // one warp, warp-level barriers only
            for (int k = 2; k <= sort_n; k <<= 1)
                for (int j = k >> 1; j > 0; j >>= 1) {
                    if (lane < (sort_n >> 1)) {
                        const int i = ((lane & ~(j - 1)) << 1) | (lane & (j - 1));
                        const int ixj = i | j;
                        const bool up = (i & k) == 0;
                        const unsigned long long a = sel[i], b = sel[ixj];
                        if ((a > b) == up) { sel[i] = b; sel[ixj] = a; }
                    }
                    __syncwarp();
                }
        }
        __syncthreads();
    } else {
        for (int k = 2; k <= sort_n; k <<= 1) {
            for (int j = k >> 1; j > 0; j >>= 1) {
                for (int t = tid; t < (sort_n >> 1); t += kThreads) {
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
        const uint32_t idx = (uint32_t)sel[rr];
        const int row = c_shift >= 0 ? (int)(idx >> c_shift) : (int)(idx / (uint32_t)C);
        const int code = (int)idx - row * C;
        const float s = sc ? __ldg(sc + row) : 0.f;
        out_score[(size_t)u * W_out + rr] = __fadd_rn(s, __ldg(lp + idx));
        out_parent[(size_t)u * W_out + rr] = row;
        out_code[(size_t)u * W_out + rr] = code;
    }
}

int next_pow2(int x) { int p = 1; while (p < x) p <<= 1; return p; }

}  // namespace

size_t topk_workspace_bytes(int, int, int) { return 0; }

int launch_topk(const float* logp, const float* score, int B, int W_in, int C, int W_out,
                float* out_score, int32_t* out_parent, int32_t* out_code, void*, size_t,
                cudaStream_t st) {
    const long long N = (long long)W_in * C;
    const int cap = next_pow2(W_out) * 2 < 128 ? 128 : next_pow2(W_out) * 2;  // sort buffer entries
    const size_t fixed = ((sizeof(Shared) + 15) / 16) * 16 + (size_t)cap * 8;
    const long long cache_max = ((long long)kSmemBudget - (long long)fixed) / 4;
    static bool attr_done = false;  // idempotent; a benign race at worst repeats the calls
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
        const long long slice = (N + n - 1) / n;
        cache_cap = (int)(slice < cache_max ? slice : cache_max);
        cfg.gridDim = dim3((unsigned)(B * n));
        cfg.dynamicSmemBytes = fixed + (size_t)cache_cap * 4;
        at[0].val.clusterDim.x = n;
    };
    auto max_clusters = [&](int n) -> int {  // resident clusters of size n with the current smem; cached
        static int memo_smem[5] = {-1, -1, -1, -1, -1}, memo_val[5] = {0, 0, 0, 0, 0};
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
    if (const char* e = getenv("STARK_TOPK_NC")) nc = atoi(e);  // TEMP experiment
    configure(nc);
    int c_shift = -1;
    if ((C & (C - 1)) == 0) { c_shift = 0; while ((1 << c_shift) < C) ++c_shift; }
    STARK_CUDA_TRY(cudaLaunchKernelEx(&cfg, topk_kernel, logp, score, W_in, C, c_shift, W_out, out_score,
                                      out_parent, out_code, cache_cap, cap));
    return STARK_OK;
}

}  // namespace stark
