// A3: stark_beam_topk -- per-level beam selection, bit-exact and deterministic.
//
// Beam score = sum of per-level log-probabilities (Eq. 1);
// each level keeps the top-W candidate paths.  Per user:
//   key[i*C + c] = fl32(score[i] + logp[i, c])          (one fp32 add, reading R4)
//   keep the W_out entries first in (key descending, flat index ascending)
//   (reading R6), output sorted in that order.
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
//   sort     CTA 0 sorts the composites (a strict total order: the result does
//            not depend on arrival order): bitonic, 64 keys per warp in
//            registers with shuffles, shared memory only for the strides that
//            cross warps; writes the first W_out as (score, parent, code),
//            recomputing score with the same fp32 add.
// Algorithmic HBM bytes: 4 per candidate (read once) + 4 per input beam + 12
// per selected beam.  Keys beyond the shared-memory
// cache (paper-scale codebooks) are re-read through L2 in each pass.
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
constexpr int kRegSortMax = 1024;     // register bitonic handles up to 2 keys per thread
constexpr int kSmemBudget = 227 * 1024;

struct Shared {
    uint32_t hist[2][kBins];       // ping-pong by pass parity
    uint32_t coarse[2][kCoarse];
    uint32_t warp_max[kWarps], warp_min[kWarps];
    uint32_t list_len[kMaxCluster];
    uint32_t sel_bin, sel_rem, sel_cnt;
    uint32_t cta_max, cta_min;     // this CTA's keys (read remotely)
    uint32_t cursor;               // length of this CTA's list (read remotely)
};

__device__ __forceinline__ uint32_t ord_of(float key) {
    uint32_t b = __float_as_uint(key);
    if (b == 0x80000000u) b = 0u;  // -0.0 == +0.0 (IEEE comparison, reading R6)
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

__device__ __forceinline__ void named_barrier(int id, int n_threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n_threads) : "memory");
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
    auto key_ord = [&](uint32_t idx) -> uint32_t {
        const int row = c_shift >= 0 ? (int)(idx >> c_shift) : (int)(idx / (uint32_t)C);
        const float s = sc ? __ldg(sc + row) : 0.f;
        return ord_of(__fadd_rn(s, __ldg(lp + idx)));
    };
    auto ord_at = [&](int j, uint32_t idx) -> uint32_t { return j < cache_cap ? cache[j] : key_ord(idx); };

    for (int b = tid; b < 2 * kBins + 2 * kCoarse; b += kThreads) (&sh.hist[0][0])[b] = 0;  // hist + coarse
    if (tid == 0) sh.cursor = 0;

    // ---- load: the one pass over HBM ---------------------------------------------------
    uint32_t mx = 0u, mn = 0xffffffffu;
    for (int base = 0; base < span; base += kThreads * kUnroll) {
        // all 2 * kUnroll loads are issued before any is consumed: indices are clamped instead of branched
        // around (a branch per key made ptxas wait for each load pair in turn: 8 round trips instead of 1)
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
            if (j < span && idx_of(j) < N) {
                const uint32_t o = ord_of(__fadd_rn(sv[x], lv[x]));
                if (j < cache_cap) cache[j] = o;
                mx = max(mx, o); mn = min(mn, o);
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

    // ---- radix select on V over the parked keys ----------------------------------------------------
    const uint32_t K = (uint32_t)W_out;
    uint32_t rem = K;                 // keys still to take from the candidate set
    unsigned long long pref = 0ull;   // value of V >> r shared by every candidate
    int r = nb + nbi;                 // unresolved low bits of V (<= 63)
    uint32_t cb = N;                  // candidates (= keys with V >> r == pref)
#pragma unroll 1
    for (int pass = 0; (K - rem) + cb > (uint32_t)cap; ++pass) {  // same decision in every CTA
        const int arr = pass & 1;
        const int w = min(11, r), shift = r - w;
        const uint32_t mask = (1u << w) - 1u;
        for (int base = 0; base < span; base += kThreads * 4) {  // 4 parked keys in flight per thread
            uint32_t o4[4], i4[4];
#pragma unroll
            for (int x = 0; x < 4; ++x) {
                const int j = base + x * kThreads + tid;
                i4[x] = j < span ? idx_of(j) : N;
                o4[x] = i4[x] < N ? ord_at(j, i4[x]) : 0u;
            }
#pragma unroll
            for (int x = 0; x < 4; ++x) {
                if (i4[x] < N) {
                    const unsigned long long v = vkey(o4[x], i4[x]);
                    if ((v >> r) == pref) atomicAdd(&sh.hist[arr][(uint32_t)(v >> shift) & mask], 1u);
                }
            }
        }
        __syncthreads();
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
    for (int base = 0; base < span; base += kThreads * 4) {
        uint32_t o4[4], i4[4];
#pragma unroll
        for (int x = 0; x < 4; ++x) {
            const int j = base + x * kThreads + tid;
            i4[x] = j < span ? idx_of(j) : N;
            o4[x] = i4[x] < N ? ord_at(j, i4[x]) : 0u;
        }
#pragma unroll
        for (int x = 0; x < 4; ++x) {
            const bool f = i4[x] < N && (vkey(o4[x], i4[x]) >> r) >= pref;
            const uint32_t bal = __ballot_sync(0xffffffffu, f);
            if (bal) {  // one shared-memory atomic per warp-iteration reserves the slots
                const int leader = __ffs(bal) - 1;
                uint32_t pos = 0;
                if (lane == leader) pos = atomicAdd(&sh.cursor, (uint32_t)__popc(bal));
                pos = __shfl_sync(0xffffffffu, pos, leader);
                pos += __popc(bal & ((1u << lane) - 1u));
                if (f && pos < (uint32_t)cap) sel[pos] = ((unsigned long long)(~o4[x]) << 32) | i4[x];
            }
        }
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
    } else if (S <= kRegSortMax) {
        // registers: warp w owns elements [64w, 64w+64): lane holds e0 = 64w + lane and e1 = e0 + 32.
        // Strides < 32 exchange by shuffle, stride 32 is thread-local, strides >= 64 go through shared memory.
        const int n_warps = S >> 6, n_thr = n_warps * 32;
        if (warp < n_warps) {
            const int e0 = warp * 64 + lane, e1 = e0 + 32;
            unsigned long long a = sel[e0], b = sel[e1];
            for (int k = 2; k <= S; k <<= 1) {
                for (int j = k >> 1; j > 0; j >>= 1) {
                    if (j >= 64) {
                        sel[e0] = a; sel[e1] = b;
                        named_barrier(1, n_thr);
                        const unsigned long long pa = sel[e0 ^ j], pb = sel[e1 ^ j];
                        const bool keep_min = ((e0 & j) == 0) == ((e0 & k) == 0);  // same for e1: j, k >= 64
                        a = keep_min ? min(a, pa) : max(a, pa);
                        b = keep_min ? min(b, pb) : max(b, pb);
                        named_barrier(1, n_thr);
                    } else if (j == 32) {
                        const bool up = (e0 & k) == 0;
                        if ((a > b) == up) { const unsigned long long t = a; a = b; b = t; }
                    } else {
                        const unsigned long long pa = __shfl_xor_sync(0xffffffffu, a, j);
                        const unsigned long long pb = __shfl_xor_sync(0xffffffffu, b, j);
                        const bool lower = (lane & j) == 0;
                        const bool min_a = lower == ((e0 & k) == 0), min_b = lower == ((e1 & k) == 0);
                        a = min_a ? min(a, pa) : max(a, pa);
                        b = min_b ? min(b, pb) : max(b, pb);
                    }
                }
            }
            sel[e0] = a; sel[e1] = b;
        }
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
        const uint32_t idx = (uint32_t)sel[rr];
        const int row = c_shift >= 0 ? (int)(idx >> c_shift) : (int)(idx / (uint32_t)C);
        const int code = (int)idx - row * C;
        const float s = sc ? __ldg(sc + row) : 0.f;
        out_score[(size_t)u * W_out + rr] = __fadd_rn(s, __ldg(lp + min(idx, N - 1)));
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
        const long long slice = ((N + kChunk - 1) / kChunk + n - 1) / n * kChunk;  // whole chunks
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
    configure(nc);
    int c_shift = -1;
    if ((C & (C - 1)) == 0) { c_shift = 0; while ((1 << c_shift) < C) ++c_shift; }
    STARK_CUDA_TRY(cudaLaunchKernelEx(&cfg, topk_kernel, logp, score, W_in, C, c_shift, W_out, out_score,
                                      out_parent, out_code, cache_cap, cap));
    return STARK_OK;
}

}  // namespace stark
