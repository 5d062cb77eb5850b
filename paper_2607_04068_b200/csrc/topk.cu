// A3: stark_beam_topk -- per-level beam selection, bit-exact and deterministic.
//
// Beam score = sum of per-level log-probabilities (Eq. 1);
// each level keeps the top-W candidate paths.  Per user:
//   key[i*C + c] = fl32(score[i] + logp[i, c])          (one fp32 add, reading R4)
//   keep the W_out entries first in (key descending, flat index ascending)
//   (reading R6), output sorted in that order.
//
// Design (one thread-block CLUSTER per user, a single pass over HBM):
//   phase 0  every CTA of the cluster streams its contiguous slice of the
//            user's candidates once, maps each key to an order-preserving
//            uint32 `ord`, parks it in shared memory and histograms its top
//            11 bits.  A running lower bound `dmin` (the CTA has already seen
//            >= W_out keys in bins >= dmin) prunes the shared-memory atomics to
//            the tail of the distribution.
//   select   3 radix passes (11 + 11 + 10 bits) find the exact 32-bit threshold
//            T = ord of the W_out-th largest key.  Per-CTA histograms are
//            combined through distributed shared memory (DSMEM); every CTA
//            redundantly runs the same suffix scan, so no broadcast is needed.
//   gather   keys with ord > T, plus the lowest-index (W_out - #greater) keys
//            with ord == T (index order = cluster-rank order x in-slice order),
//            are written as 64-bit composites (~ord, idx) into CTA 0's shared
//            memory through DSMEM.
//   sort     CTA 0 bitonic-sorts the W_out composites -- a strict total order,
//            so the result does not depend on arrival order -- and writes
//            (score, parent, code), recomputing score with the same fp32 add.
// Algorithmic HBM bytes: 4 per candidate (read once) + 4 per input beam + 12
// per selected beam.  Slices beyond the shared-memory
// cache are re-read through L2 in the later passes.
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace stark {

namespace {

constexpr int kThreads = 1024;
constexpr int kWarps = kThreads / 32;
constexpr int kUnroll = 8;
constexpr int kBins = 2048;
constexpr int kCacheMax = 40960;   // ord keys parked in shared memory per CTA
constexpr int kMaxOut = 4096;      // W_out limit (sort buffer)
constexpr int kMaxCluster = 8;     // portable cluster size
constexpr int kSliceTarget = 8192; // candidates per CTA the host aims for

struct Shared {
    uint32_t hist[3][kBins];
    uint32_t warp_tot[kWarps];
    uint32_t sel_bin, sel_rem, dmin;
    uint32_t n_gt, n_eq;           // this CTA's counts (read remotely)
    uint32_t gt_cursor, eq_cursor; // local output cursors
    uint32_t scan_base;
};

__device__ __forceinline__ uint32_t ord_of(float key) {
    uint32_t b = __float_as_uint(key);
    if (b == 0x80000000u) b = 0u;  // -0.0 == +0.0 (IEEE comparison, reading R6)
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

// Block-wide: find the largest bin b with  sum_{b' >= b} g(b') >= rem.
// Every thread passes the counts of ITS bins (BPT consecutive bins starting at
// (kThreads-1-tid)*BPT ... i.e. thread 0 owns the highest bins).  Result in
// sh.sel_bin / sh.sel_rem (= rem minus the count in bins above sel_bin).
// If the total is < rem, sel_bin = 0 and sel_rem = 0xffffffff.
template <int BPT>
__device__ __forceinline__ void block_select(Shared& sh, const uint32_t (&cnt)[BPT], uint32_t rem) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t mine = 0;
#pragma unroll
    for (int j = 0; j < BPT; ++j) mine += cnt[j];
    uint32_t inc = mine;  // inclusive scan over threads (thread 0 = highest bins)
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (tid == 0) { sh.sel_bin = 0; sh.sel_rem = 0xffffffffu; }
    if (lane == 31) sh.warp_tot[warp] = inc;
    __syncthreads();
    uint32_t wbase = 0;
    {
        uint32_t w = lane < kWarps ? sh.warp_tot[lane] : 0;
        uint32_t winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += t;
        }
        wbase = __shfl_sync(0xffffffffu, winc - w, warp);
    }
    uint32_t before = wbase + inc - mine;  // elements in bins above this thread's bins
    if (before < rem && rem <= before + mine) {
        // the crossing is inside my bins: walk them from the highest down
        const int top = (kThreads - 1 - tid) * BPT + (BPT - 1);
#pragma unroll
        for (int j = 0; j < BPT; ++j) {
            const uint32_t c = cnt[BPT - 1 - j];
            if (before < rem && rem <= before + c) { sh.sel_bin = top - j; sh.sel_rem = rem - before; }
            before += c;
        }
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kThreads, 1)
topk_kernel(const float* __restrict__ logp, const float* __restrict__ score, int W_in, int C, int c_shift,
            int W_out, float* __restrict__ out_score, int32_t* __restrict__ out_parent,
            int32_t* __restrict__ out_code, int cache_cap, int sort_n) {
    cg::cluster_group cluster = cg::this_cluster();
    const int nc = (int)cluster.num_blocks();
    const int rank = (int)cluster.block_rank();
    const int u = blockIdx.x / nc;
    const int tid = threadIdx.x;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    Shared& sh = *reinterpret_cast<Shared*>(smem_raw);
    unsigned long long* sel = reinterpret_cast<unsigned long long*>(smem_raw + ((sizeof(Shared) + 15) / 16) * 16);
    uint32_t* cache = reinterpret_cast<uint32_t*>(sel + sort_n);

    const long long N = (long long)W_in * C;
    long long slice = (N + nc - 1) / nc;
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
    if (tid == 0) { sh.dmin = 0; sh.n_gt = 0; sh.n_eq = 0; sh.gt_cursor = 0; sh.eq_cursor = 0; }
    __syncthreads();

    // ---- phase 0: one pass over HBM ------------------------------------------
    const uint32_t K = (uint32_t)W_out;
    {
        const int per_iter = kThreads * kUnroll;
        const int n_iter = (n_local + per_iter - 1) / per_iter;
        const bool prune = n_iter >= 2;
        for (int it = 0; it < n_iter; ++it) {
            uint32_t o[kUnroll];
#pragma unroll
            for (int x = 0; x < kUnroll; ++x) {
                const int j = it * per_iter + x * kThreads + tid;
                o[x] = j < n_local ? key_ord(j) : 0u;
            }
            const uint32_t dm = sh.dmin;
#pragma unroll
            for (int x = 0; x < kUnroll; ++x) {
                const int j = it * per_iter + x * kThreads + tid;
                if (j < n_local) {
                    if (j < cache_cap) cache[j] = o[x];
                    const uint32_t dg = o[x] >> 21;
                    if (dg >= dm) atomicAdd(&sh.hist[0][dg], 1u);
                }
            }
            // refresh the pruning bound after iterations 0, 1, 3, 7, ... (not the last)
            if (prune && it + 1 < n_iter && ((it + 1) & it) == 0) {
                __syncthreads();
                uint32_t cnt[2];
                const int b0 = (kThreads - 1 - tid) * 2;
                cnt[0] = sh.hist[0][b0]; cnt[1] = sh.hist[0][b0 + 1];
                block_select<2>(sh, cnt, K);
                if (tid == 0 && sh.sel_rem != 0xffffffffu) sh.dmin = sh.sel_bin;
                __syncthreads();
            }
        }
    }
    cluster.sync();

    // ---- 3 radix passes: exact threshold ---------------------------------------
    uint32_t prefix = 0, rem = K;
#pragma unroll 1
    for (int pass = 0; pass < 3; ++pass) {
        const int bits = pass < 2 ? 11 : 10;
        if (pass > 0) {
            const int sh_hi = pass == 1 ? 21 : 10;     // bits above this digit
            const uint32_t mask = (1u << bits) - 1u;
            const int sh_lo = pass == 1 ? 10 : 0;
            for (int j = tid; j < n_local; j += kThreads) {
                const uint32_t o = ord_at(j);
                if ((o >> sh_hi) == prefix) atomicAdd(&sh.hist[pass][(o >> sh_lo) & mask], 1u);
            }
            cluster.sync();
        }
        uint32_t cnt[2] = {0u, 0u};
        const int b0 = (kThreads - 1 - tid) * 2;
        if (bits == 11 || b0 < 1024) {
            for (int r = 0; r < nc; ++r) {
                const uint32_t* rh = cluster.map_shared_rank(&sh.hist[pass][0], r);
                cnt[0] += rh[b0]; cnt[1] += rh[b0 + 1];
            }
        }
        block_select<2>(sh, cnt, rem);
        prefix = (prefix << bits) | sh.sel_bin;
        rem = sh.sel_rem;
        __syncthreads();
    }
    const uint32_t T = prefix;      // ord of the W_out-th largest key
    const uint32_t need_eq = rem;   // how many keys == T are selected (lowest indices)
    const uint32_t n_gt_total = K - need_eq;

    // ---- count, exchange, gather ------------------------------------------------
    {
        uint32_t cg_ = 0, ce_ = 0;
        for (int j = tid; j < n_local; j += kThreads) {
            const uint32_t o = ord_at(j);
            cg_ += o > T; ce_ += o == T;
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            cg_ += __shfl_xor_sync(0xffffffffu, cg_, off);
            ce_ += __shfl_xor_sync(0xffffffffu, ce_, off);
        }
        if ((tid & 31) == 0) { atomicAdd(&sh.n_gt, cg_); atomicAdd(&sh.n_eq, ce_); }
    }
    cluster.sync();
    uint32_t gt_off = 0, eq_before = 0;
    for (int r = 0; r < rank; ++r) {
        gt_off += *cluster.map_shared_rank(&sh.n_gt, r);
        eq_before += *cluster.map_shared_rank(&sh.n_eq, r);
    }
    const uint32_t my_eq = sh.n_eq;
    unsigned long long* sel0 = cluster.map_shared_rank(sel, 0);
    // 0: take none of my equals, 1: take all (any order), 2: boundary CTA (index order)
    const int eq_mode = eq_before >= need_eq ? 0 : (eq_before + my_eq <= need_eq ? 1 : 2);
    for (int j = tid; j < n_local; j += kThreads) {
        const uint32_t o = ord_at(j);
        const unsigned long long comp = ((unsigned long long)(~o) << 32) | (uint32_t)(lo + j);
        if (o > T) {
            sel0[gt_off + atomicAdd(&sh.gt_cursor, 1u)] = comp;
        } else if (o == T && eq_mode == 1) {
            sel0[n_gt_total + eq_before + atomicAdd(&sh.eq_cursor, 1u)] = comp;
        }
    }
    if (eq_mode == 2) {
        // ordered: the first (need_eq - eq_before) equals of this slice, by index
        const uint32_t want = need_eq - eq_before;
        if (tid == 0) sh.scan_base = 0;
        __syncthreads();
        for (int base = 0; base < n_local; base += kThreads) {
            const uint32_t taken = sh.scan_base;
            if (taken >= want) break;  // uniform: read after a barrier
            const int j = base + tid;
            const uint32_t o = j < n_local ? ord_at(j) : 0u;
            const bool f = j < n_local && o == T;
            const uint32_t bal = __ballot_sync(0xffffffffu, f);
            const int lane = tid & 31, warp = tid >> 5;
            if (lane == 0) sh.warp_tot[warp] = __popc(bal);
            __syncthreads();
            uint32_t wb = 0, tot = 0;
            for (int w = 0; w < kWarps; ++w) {
                const uint32_t c = sh.warp_tot[w];
                wb += w < warp ? c : 0;
                tot += c;
            }
            const uint32_t rnk = taken + wb + __popc(bal & ((1u << lane) - 1u));
            if (f && rnk < want)
                sel0[n_gt_total + eq_before + rnk] = ((unsigned long long)(~o) << 32) | (uint32_t)(lo + j);
            __syncthreads();
            if (tid == 0) sh.scan_base = taken + tot;
            __syncthreads();
        }
    }
    cluster.sync();
    if (rank != 0) return;

    // ---- CTA 0: bitonic sort of the W_out composites, ascending ------------------
    for (int i = K + tid; i < sort_n; i += kThreads) sel[i] = ~0ull;
    __syncthreads();
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
    for (int r = tid; r < (int)K; r += kThreads) {
        const uint32_t idx = (uint32_t)sel[r];
        const int row = c_shift >= 0 ? (int)(idx >> c_shift) : (int)(idx / (uint32_t)C);
        const int code = (int)idx - row * C;
        const float s = sc ? __ldg(sc + row) : 0.f;
        out_score[(size_t)u * W_out + r] = __fadd_rn(s, __ldg(lp + idx));
        out_parent[(size_t)u * W_out + r] = row;
        out_code[(size_t)u * W_out + r] = code;
    }
}

int next_pow2(int x) { int p = 1; while (p < x) p <<= 1; return p; }

}  // namespace

size_t topk_workspace_bytes(int, int, int) { return 0; }

int launch_topk(const float* logp, const float* score, int B, int W_in, int C, int W_out,
                float* out_score, int32_t* out_parent, int32_t* out_code, void*, size_t,
                cudaStream_t st) {
    const long long N = (long long)W_in * C;
    int nc = 1;
    while (nc < kMaxCluster && (N + nc - 1) / nc > kSliceTarget) nc <<= 1;
    const long long slice = (N + nc - 1) / nc;
    const int cache_cap = (int)(slice < kCacheMax ? slice : kCacheMax);
    const int sort_n = next_pow2(W_out < 2 ? 2 : W_out);
    int c_shift = -1;
    if ((C & (C - 1)) == 0) { c_shift = 0; while ((1 << c_shift) < C) ++c_shift; }
    const size_t smem = ((sizeof(Shared) + 15) / 16) * 16 + (size_t)sort_n * 8 + (size_t)cache_cap * 4;
    static bool attr_done = false;  // idempotent; a benign race at worst repeats the call
    if (!attr_done) {
        STARK_CUDA_TRY(cudaFuncSetAttribute(topk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        attr_done = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(B * nc));
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = nc; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    STARK_CUDA_TRY(cudaLaunchKernelEx(&cfg, topk_kernel, logp, score, W_in, C, c_shift, W_out, out_score,
                                      out_parent, out_code, cache_cap, sort_n));
    return STARK_OK;
}

}  // namespace stark
