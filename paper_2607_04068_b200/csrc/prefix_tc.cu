// A1 and A1+A2 (tensor-core form): stark_prefix_attn and the fused stark_decode_attn for bf16, any number
// of query rows.
//
// the conventional path recomputes attention over the shared
// user-history prefix once per beam; STARK computes it once.  Here all
// (beam, group-head) query rows of one (user, KV head) are packed into the M
// dimension of a dense contraction against that user's prefix K/V tiles, so
// each prefix byte is fetched once per step per CTA instead of once per beam.
// This is a real GEMM-shaped op (AI ~ M flop per KV byte), so it runs on the
// 5th-generation tensor cores, organised like a two-accumulator flash-attention
// forward:
//
//   * 384 threads = 3 warpgroups: warpgroup 0 holds the TMA producer warp and
//     the MMA issuer warp (one elected lane each; two idle warps), warpgroups 1
//     and 2 are the softmax warpgroups of accumulator sets 0 and 1, one TMEM
//     lane (= query row) per thread.  setmaxnreg moves registers from
//     warpgroup 0 to the softmax warpgroups, whose threads keep a whole S row
//     (128 fp32) in registers between its maximum and its exponentials;
//   * Q tiles and K/V tiles arrive by TMA (cp.async.bulk.tensor, 128-byte
//     swizzle); K and V alternate through one NS-slot mbarrier ring; the first
//     loads are issued before TMEM is allocated;
//   * S_t = Q K^T by tcgen05.mma (SS, both operands K-major) into TMEM, one
//     128-column accumulator per set; P_t (bf16) overwrites S_t in place;
//     O_t += P_t V by tcgen05.mma with A = P_t from TMEM and B = V from shared
//     memory (MN-major descriptor: V is [kv][D] with D contiguous);
//     TMEM columns: S0/P0 [0,128) S1/P1 [128,256) O0 [256,256+D) O1 [384,384+D);
//   * the MMA warp issues  PV_0, QK_0(next), PV_1, QK_1(next), ...  so the tensor
//     pipe works for one set while the other set's warpgroup runs its softmax
//     (exp2 on the MUFU pipe).  The pipe executes in issue order, so when
//     S_t(j) is ready PV_t(j-1) has completed and O_t may be rescaled (lazily:
//     only when a row maximum grows by > 2^8) without another barrier;
//   * pair mode: the CTA owns two 128-row Q tiles, set t = Q tile t, every K/V
//     tile serves 256 rows.  Parity mode (when its doubled CTA count still
//     fits one wave): the CTA owns one Q tile, set t = the KV tiles of parity
//     t; the two partial softmaxes are folded inside the CTA at the end;
//   * FUSED = false: the epilogue stages the O rows in the idle K/V ring and
//     writes coalesced split-softmax partials (m, l, o) for
//     stark_tree_attn_step.  FUSED = true: the prefix splits of one (Q tiles,
//     KV head, user) are a thread-block cluster; partial rows are exchanged
//     through distributed shared memory and the owner of each 32-row block
//     merges them, adds the suffix chain (scores computed while the first
//     tiles are in flight), normalises and writes bf16 rows -- no partial ever
//     reaches HBM.
//
// Decode step 0 (a single query per user, M = G rows) runs through the same
// kernel: the contraction is then a pure HBM stream of the prefix, and warps
// without live rows skip their softmax.
// Every mbarrier wait is bounded (trap after ~1 s) so that a protocol bug
// surfaces as a launch failure instead of a hung GPU.
#include <cuda.h>

#include "common.cuh"

namespace stark {

namespace {

constexpr int BM = 128;          // query rows per Q tile = MMA M (two Q tiles per CTA)
constexpr int BN = 128;          // KV rows per tile      = MMA N of S, K-extent of P V
constexpr int kThreadsTC = 384;  // warpgroup 0: TMA warp, MMA warp (2 idle); warpgroups 1, 2: softmax
constexpr int kFirstSoftmaxWarp = 4;
constexpr int kSoftmaxThreads = 128;
constexpr float kRescaleThreshold = 8.0f;  // log2 units

// ---- PTX wrappers -------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    if (mbar_try(bar, parity)) return;
    const long long t0 = clock64();
    while (!mbar_try(bar, parity)) {
        if (clock64() - t0 > (1ll << 31)) __trap();  // protocol bug: fail loudly, never hang
    }
}
__device__ __forceinline__ void fence_barrier_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(dst), "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

// Store one box of a 4-d tensor map from shared memory (bulk async group of the issuing thread); elements outside
// the tensor are not written.
__device__ __forceinline__ void tma_store_4d(const CUtensorMap* tm, uint32_t src, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
                 ::"l"(tm), "r"(src), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

// The 32 finished bf16 rows of one warp, staged at `stage` (1024-byte aligned) in the layout of a 128-byte-swizzled
// TMA box per 64 columns ([D / 64][32 rows][128 B], 16-byte chunk c of row r at c ^ (r & 7)), go to
// out[u, beam, head, :] with one TMA store per box.  Row r of the warp is (beam, head) = (beam0 + r / hb, head0 +
// r % hb) with hb = min(G, 32) heads per beam in the box; beams >= n_q lie outside the tensor map and are clipped.
// (The copy loop this replaces took 2.2-2.7 k cycles per warp: 16 rounds of shared-memory load, shuffle, store.)
template <int D>
__device__ __forceinline__ void store_rows_tma(const CUtensorMap* tm_o, const unsigned char* stage, int lane, int u,
                                            int head0, int beam0) {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // this thread's staged row -> async proxy
    __syncwarp();
    if (lane == 0) {
#pragma unroll
        for (int bx = 0; bx < D / 64; ++bx)
            tma_store_4d(tm_o, smem_u32(stage) + bx * (32 * 128), bx * 64, head0, beam0, u);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the staging memory may go (CTA exit)
    }
}

__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t addr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]
__device__ __forceinline__ void umma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(acc) : "memory");
}

// 32 consecutive fp32 columns of this thread's TMEM lane.
__device__ __forceinline__ void tmem_ld32(uint32_t addr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(addr) : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t addr, const uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%32], "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31};"
        ::"r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
          "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]),
          "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]),
          "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31]),
          "r"(addr) : "memory");
}
// 16 consecutive 32-bit columns of this thread's TMEM lane.
__device__ __forceinline__ void tmem_st16(uint32_t addr, const uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%16], "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15};"
        ::"r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
          "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]),
          "r"(addr) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ float fast_exp2(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---- descriptors ----------------------------------------------------------------
// Shared-memory matrix descriptor, 128-byte swizzle, descriptor version 1 (sm_100):
//   [0,14) start>>4 | [16,30) leading byte offset>>4 | [32,46) stride byte offset>>4 |
//   [46,48) version=1 | [61,64) layout=2 (SWIZZLE_128B)
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((addr & 0x3ffffu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) |
           ((uint64_t)(sbo_bytes >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// Instruction descriptor, kind::f16: D=f32 [4,6)=1, A=bf16 [7,10)=1, B=bf16 [10,13)=1,
// a_major bit 15, b_major bit 16 (0 = K-major, 1 = MN-major), N>>3 at [17,23), M>>4 at [24,29).
__host__ __device__ constexpr uint32_t instr_desc(int M, int N, int b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(N >> 3) << 17) |
           ((uint32_t)(M >> 4) << 24);
}


// ---- fused decode attention (A1 + A2 in one launch) ---------------------------------
// Arguments of the suffix / merge / normalise tail that replaces the partial epilogue.
struct FusedArgs {
    const __nv_bfloat16* q;    // [B, n_q, Hq, D]
    const __nv_bfloat16* ks;   // suffix K [d, B, Wmax, Hkv, D]
    const __nv_bfloat16* vs;
    const int32_t* anc;        // this level's half of the ancestor index, [B, Wmax, d]
    __nv_bfloat16* out;        // [B, n_q, Hq, D]
    int level, Wmax, d;
    float scale;               // softmax scale (natural units)
    // stark_decode_step (A4 folded into the same launch), kn != nullptr: this level's own K/V rows are read from
    // kn / vn [B, n_q, Hkv, D], `anc` is the PREVIOUS level's half and each row's chain is its parent's chain plus
    // itself; the otherwise idle warps of warpgroup 0 copy kn / vn into the suffix level and write anc_new.
    const __nv_bfloat16* kn;
    const __nv_bfloat16* vn;
    const int32_t* parent;     // [B, n_q] (unused at level 1)
    int32_t* anc_new;          // this level's half of the ancestor index, or nullptr (layers > 0)
};

__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_rank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t map_to_rank(uint32_t smem_addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster_f4(uint32_t addr, float a, float b, float c, float d) {
    asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ void st_cluster_f2(uint32_t addr, float a, float b) {
    asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(a), "f"(b) : "memory");
}

#ifdef STARK_TC_PROF   // per-iteration timeline of ONE CTA (scratch builds only; never defined in the product build)
__device__ long long g_tc_prof[64 * 16];
#define TCPROF(j, slot) do { if ((j) < 64 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == STARK_TC_PROF) g_tc_prof[(j) * 16 + (slot)] = clock64(); } while (0)
#else
#define TCPROF(j, slot) do {} while (0)
#endif

template <int D> struct TcCfg {
    static constexpr int BOXES = D / 64;                 // 64-element (128-byte) column boxes per row
    static constexpr int TILE_BYTES = BOXES * BM * 128;  // one 128-row tile of Q, K or V
    static constexpr int NS = D == 128 ? 5 : 8;          // K/V ring slots (K_j, V_j, K_j+1, ... in turn)
    static constexpr int SMEM_BYTES = TILE_BYTES * (2 + NS) + 1024 /*align*/ + 256 /*barriers*/;
    static constexpr int TMEM_COLS = 512;
    static constexpr int COL_S = 0;                      // S_t / P_t at COL_S + t * 128
    static constexpr int COL_O = 256;                    // O_t at COL_O + t * 128
};

// Suffix-chain scores of one query row (Eq. 14: ancestors and itself), in log2 units of the
// scaled score, and the element offsets of the chain's rows in the suffix buffers.  Independent of the prefix:
// the fused kernel runs it right after its last softmax iteration, inside the wait for the last MMAs.  (Run
// ahead of the loop it held the first softmax iteration back: under the kernel's own K/V stream a dependent
// global load takes 2-3 k cycles, and there are three in a row here.  Measured A/B: 1-2.5 % per launch.)
template <int D>
__device__ __forceinline__ void chain_scores(const FusedArgs& fa, float scale_log2, int u, int i, int kv, int n_q,
                                          int Hkv, int B, const unsigned char* q_tile, int r, float* y,
                                          uint32_t* off_out) {
    const size_t level_stride = (size_t)B * fa.Wmax * Hkv * D;
    // the query row comes from the Q tile TMA left in shared memory (128-byte swizzle: 16-byte chunk c of row r of a
    // 64-column box sits at chunk c ^ (r & 7)); conflict-free, and a quarter of this function's global traffic less
    uint4 qv[D / 8];
#pragma unroll
    for (int c = 0; c < D / 8; ++c)
        qv[c] = *reinterpret_cast<const uint4*>(q_tile + (c / 8) * (BM * 128) + r * 128 + (((c % 8) ^ (r & 7)) << 4));
    const bool inl = fa.kn != nullptr;
    int chain_of = i;                                   // whose row of `anc` holds this query's ancestors
    if (inl && fa.level >= 2) chain_of = min(max(__ldg(fa.parent + (size_t)u * n_q + i), 0), fa.Wmax - 1);
#pragma unroll 1
    for (int t = 0; t < fa.level; ++t) {
        size_t off;
        const uint4* kp;
        if (inl && t == fa.level - 1) {                 // itself: not yet in the suffix buffers
            off = (((size_t)u * n_q + i) * Hkv + kv) * D;
            kp = reinterpret_cast<const uint4*>(fa.kn + off);
        } else {
            int a = __ldg(fa.anc + ((size_t)u * fa.Wmax + chain_of) * fa.d + t);
            a = min(max(a, 0), fa.Wmax - 1);            // memory safety on garbage input
            off = (size_t)t * level_stride + (((size_t)u * fa.Wmax + a) * Hkv + kv) * D;
            kp = reinterpret_cast<const uint4*>(fa.ks + off);
        }
        float dot = 0.f;
#pragma unroll
        for (int c = 0; c < D / 8; ++c) {
            const uint4 kk = __ldg(kp + c);
            const uint32_t qa[4] = {qv[c].x, qv[c].y, qv[c].z, qv[c].w}, ka[4] = {kk.x, kk.y, kk.z, kk.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                dot = fmaf(__uint_as_float(qa[e] << 16), __uint_as_float(ka[e] << 16), dot);
                dot = fmaf(__uint_as_float(qa[e] & 0xffff0000u), __uint_as_float(ka[e] & 0xffff0000u), dot);
            }
        }
        y[t] = dot * scale_log2;
        off_out[t] = (uint32_t)off;                     // suffix buffers are far below 2^32 elements
    }
}

// Tail of the fused kernel, run by the warp that owns one 32-row block (lane = row): merge the block's
// prefix partials of all splits (own rows in TMEM, the others' delivered into the K/V ring), add the suffix
// chain of each row (Eq. 14: ancestors and itself), normalise, write bf16 rows coalesced.
// Runs once per CTA, so it is written for SMALL CODE (rolled loops, per-lane scratch in shared memory): a
// fully unrolled version was instruction-fetch bound (~100 KB of straight-line code: 16 us).  The same holds
// for every once-per-CTA loop over 32-column chunks in this kernel (rescale, in-CTA merge, DSMEM send): rolled,
// they are worth 1.3 us per config-2 pass, where the kernel's code is re-fetched after every top-k launch.
template <int D>
__device__ __forceinline__ void fused_finish(const FusedArgs& fa, unsigned char* smem_raw, uint32_t ring_off, int ob, int me,
                                          int ns, int lane, uint32_t aO, bool has, float m_own, float l_own,
                                          int u, int n_q, int Hq, int G, int kv, int beam_base, int quarter,
                                          float* ch_y, const uint32_t* ch_off, const unsigned char* vstage,
                                          const CUtensorMap* tm_o) {
    constexpr uint32_t SLOT = 32 * D * 4;
    constexpr int CPR = D / 4;                          // 16-byte chunks per fp32 row
    unsigned char* ring = smem_raw + ring_off;
    // this block's own slot is never written remotely: bf16 output staging [32][D] + per-lane scratch
    unsigned char* stage = ring + (size_t)(ob * ns + me) * SLOT;
    float* wgt = reinterpret_cast<float*>(stage + 32 * D * 2);          // [8][32]: weights of the other splits
    const int r = quarter * 32 + lane;
    const int i = beam_base + r / G;
    const bool live = i < n_q;
    const int level = fa.level;
    tc_fence_after();
    float m_all = has ? m_own : -INFINITY;
    if (live)
        for (int t = 0; t < level; ++t) m_all = fmaxf(m_all, ch_y[t]);  // chain scores (log2 units), from the prologue
    // ---- log-sum-exp weights over {own split, delivered splits, chain} ------------------------------------
#pragma unroll 1
    for (int sidx = 0; sidx < ns; ++sidx)
        if (sidx != me) m_all = fmaxf(m_all, *reinterpret_cast<const float*>(ring + 8 * SLOT + (size_t)(ob * ns + sidx) * 256 + lane * 8));
    const bool any = m_all > -INFINITY;                 // false only for an empty prefix at level 0
    const float w_own = (has && any && m_own > -INFINITY) ? fast_exp2(m_own - m_all) : 0.f;
    float denom = w_own * l_own;
#pragma unroll 1
    for (int sidx = 0; sidx < ns; ++sidx) {
        if (sidx == me) continue;
        const float2 v = *reinterpret_cast<const float2*>(ring + 8 * SLOT + (size_t)(ob * ns + sidx) * 256 + lane * 8);
        const float w = (any && v.x > -INFINITY) ? fast_exp2(v.x - m_all) : 0.f;
        wgt[sidx * 32 + lane] = w;
        denom = fmaf(w, v.y, denom);
    }
#pragma unroll 1
    for (int t = 0; t < level; ++t) {
        const float e = (any && live) ? fast_exp2(ch_y[t] - m_all) : 0.f;
        ch_y[t] = e;                                    // score -> weight, in place
        denom += e;
    }
    const float inv = denom > 0.f ? 1.0f / denom : 0.f;

    // ---- output row, 32 columns at a time ---------------------------------------------------------------------
#pragma unroll 1
    for (int c = 0; c < D / 32; ++c) {
        float acc[32];
        {
            uint32_t o[32];
            tmem_ld32(aO + c * 32, o);
            tmem_wait_ld();
#pragma unroll
            for (int x = 0; x < 32; ++x) acc[x] = has ? w_own * __uint_as_float(o[x]) : 0.f;
        }
#pragma unroll 1
        for (int sidx = 0; sidx < ns; ++sidx) {
            if (sidx == me) continue;
            const float w = wgt[sidx * 32 + lane];
            const float* src = reinterpret_cast<const float*>(ring + (size_t)(ob * ns + sidx) * SLOT) + lane * D;
#pragma unroll
            for (int x = 0; x < 32; x += 4) {
                const float4 v = *reinterpret_cast<const float4*>(src + (((c * 8 + (x >> 2)) ^ (lane & (CPR - 1))) * 4));
                acc[x] = fmaf(w, v.x, acc[x]); acc[x + 1] = fmaf(w, v.y, acc[x + 1]);
                acc[x + 2] = fmaf(w, v.z, acc[x + 2]); acc[x + 3] = fmaf(w, v.w, acc[x + 3]);
            }
        }
        // chain V rows, two levels' loads in flight at a time (each is a dependent L2 / HBM round trip)
#pragma unroll 1
        for (int t0 = 0; t0 < (live ? level : 0); t0 += 2) {
            const bool two_lv = t0 + 1 < level;
            const float e[2] = {ch_y[t0], two_lv ? ch_y[t0 + 1] : 0.f};
            const int t1 = two_lv ? t0 + 1 : t0;
            const uint4* vp0 = reinterpret_cast<const uint4*>(((fa.vn && t0 == level - 1) ? fa.vn : fa.vs) + ch_off[t0]) + c * 4;
            const uint4* vp1 = reinterpret_cast<const uint4*>(((fa.vn && t1 == level - 1) ? fa.vn : fa.vs) + ch_off[t1]) + c * 4;
            uint4 vv[2][4];
            if (vstage != nullptr && t0 == 0) {         // staged by cp.async right after the last MMA (parity mode)
#pragma unroll
                for (int k4 = 0; k4 < 4; ++k4) {   // rows of D*2 bytes, 16-byte chunks XOR-swizzled by row
                    const int ch = ((c * 4 + k4) ^ (lane & 7)) * 16;
                    vv[0][k4] = *reinterpret_cast<const uint4*>(vstage + (size_t)lane * (D * 2) + ch);
                    vv[1][k4] = *reinterpret_cast<const uint4*>(vstage + (size_t)((two_lv ? 32 : 0) + lane) * (D * 2) + ch);
                }
            } else {
#pragma unroll
                for (int k4 = 0; k4 < 4; ++k4) { vv[0][k4] = __ldg(vp0 + k4); vv[1][k4] = __ldg(vp1 + k4); }
            }
#pragma unroll
            for (int lv = 0; lv < 2; ++lv)
#pragma unroll
                for (int k4 = 0; k4 < 4; ++k4) {
                    const uint32_t va[4] = {vv[lv][k4].x, vv[lv][k4].y, vv[lv][k4].z, vv[lv][k4].w};
#pragma unroll
                    for (int e2 = 0; e2 < 4; ++e2) {
                        acc[k4 * 8 + 2 * e2] = fmaf(e[lv], __uint_as_float(va[e2] << 16), acc[k4 * 8 + 2 * e2]);
                        acc[k4 * 8 + 2 * e2 + 1] = fmaf(e[lv], __uint_as_float(va[e2] & 0xffff0000u), acc[k4 * 8 + 2 * e2 + 1]);
                    }
                }
        }
#pragma unroll
        for (int k4 = 0; k4 < 4; ++k4) {                // 4 chunks of 8 bf16
            uint32_t pk[4];
#pragma unroll
            for (int e2 = 0; e2 < 4; ++e2) {
                const __nv_bfloat162 h = __floats2bfloat162_rn(acc[k4 * 8 + 2 * e2] * inv, acc[k4 * 8 + 2 * e2 + 1] * inv);
                pk[e2] = *reinterpret_cast<const uint32_t*>(&h);
            }
            const int ch = c * 4 + k4;                  // 16-byte chunk of the row: box ch / 8, swizzled inside it
            *reinterpret_cast<uint4*>(stage + (ch >> 3) * (32 * 128) + lane * 128 + (((ch & 7) ^ (lane & 7)) << 4)) =
                make_uint4(pk[0], pk[1], pk[2], pk[3]);
        }
    }
    store_rows_tma<D>(tm_o, stage, lane, u, kv * G + (quarter * 32) % G, beam_base + (quarter * 32) / G);
}

// Tail of the fused kernel for a CTA without splits in pair mode (the large-batch case).  The chain's part of the
// row -- weights relative to the chain's own maximum m_c, their sum l_c, and vs = sum_t e_t V_t -- is already in
// registers (chain_partial, run inside the wait for the last MMAs: one global round trip per LEVEL instead of one
// per level pair and 32-column chunk after it); here it is merged with the prefix part like a second split.
template <int D>
__device__ __forceinline__ void fused_finish_single(const FusedArgs& fa, unsigned char* smem_raw, uint32_t ring_off,
                                                 int blk, int lane, uint32_t aO, bool has, float m_own, float l_own,
                                                 int u, int n_q, int Hq, int G, int kv, int beam_base, int quarter,
                                                 float m_c, float l_c, const float (&vs)[D], const CUtensorMap* tm_o) {
    constexpr uint32_t SLOT = 32 * D * 4;
    unsigned char* stage = smem_raw + ring_off + (size_t)blk * SLOT;   // bf16 output staging (store_rows_tma)
    tc_fence_after();
    const float m_p = has ? m_own : -INFINITY;
    const float m_all = fmaxf(m_p, m_c);
    const bool any = m_all > -INFINITY;                 // false only for an empty prefix at level 0
    const float w_p = (any && m_p > -INFINITY) ? fast_exp2(m_p - m_all) : 0.f;
    const float w_c = (any && m_c > -INFINITY) ? fast_exp2(m_c - m_all) : 0.f;
    const float denom = fmaf(w_p, l_own, w_c * l_c);
    const float inv = denom > 0.f ? 1.0f / denom : 0.f;
    const float wp = w_p * inv, wc = w_c * inv;
#pragma unroll
    for (int c = 0; c < D / 32; ++c) {
        uint32_t o[32];
        if (has) {
            tmem_ld32(aO + c * 32, o);
            tmem_wait_ld();
        }
#pragma unroll
        for (int k4 = 0; k4 < 4; ++k4) {                // 4 chunks of 8 bf16
            uint32_t pk[4];
#pragma unroll
            for (int e2 = 0; e2 < 4; ++e2) {
                const int x = k4 * 8 + 2 * e2;
                const float a0 = fmaf(wc, vs[c * 32 + x], has ? wp * __uint_as_float(o[x]) : 0.f);
                const float a1 = fmaf(wc, vs[c * 32 + x + 1], has ? wp * __uint_as_float(o[x + 1]) : 0.f);
                const __nv_bfloat162 h = __floats2bfloat162_rn(a0, a1);
                pk[e2] = *reinterpret_cast<const uint32_t*>(&h);
            }
            const int ch = c * 4 + k4;                  // 16-byte chunk of the row: box ch / 8, swizzled inside it
            *reinterpret_cast<uint4*>(stage + (ch >> 3) * (32 * 128) + lane * 128 + (((ch & 7) ^ (lane & 7)) << 4)) =
                make_uint4(pk[0], pk[1], pk[2], pk[3]);
        }
    }
    store_rows_tma<D>(tm_o, stage, lane, u, kv * G + (quarter * 32) % G, beam_base + (quarter * 32) / G);
}

// FUSED = false: emit the split-softmax partials (stark_prefix_attn).
// FUSED = true : the n_splits CTAs of one (Q-tile pair, KV head, user) form a thread-block cluster; they
//                exchange their partial rows through distributed shared memory, and the owner of each
//                32-row block merges them, adds the suffix chain and writes the normalised bf16 output
//                (stark_decode_attn): no partial ever goes to HBM.
// SINGLE (fused only): pair mode, no splits, level >= 1 -- the instantiation with the register-resident chain part
//                and fused_finish_single as its tail (its own instantiation: carrying both tails in one kernel cost
//                the parity-mode and split launches 5-8 %).
template <int D, bool FUSED, bool SINGLE = false>
__global__ void __launch_bounds__(kThreadsTC, 1)
prefix_tc_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
                 const __grid_constant__ CUtensorMap tm_v, const __grid_constant__ CUtensorMap tm_o,
                 const int32_t* __restrict__ cu,
                 float* __restrict__ pm, float* __restrict__ pl, float* __restrict__ po, int B, int n_q,
                 int Hq, int Hkv, int G, int n_splits, float scale_log2, int parity, int lpt, const FusedArgs fa) {
    // Two TMEM accumulator sets (S_t/P_t, O_t), t = 0, 1, each served by its own softmax warpgroup:
    //   pair mode   (parity = 0): the CTA owns Q tiles 2x and 2x+1; set t = Q tile t; both see every KV tile.
    //   parity mode (parity = 1): the CTA owns ONE Q tile; set t = the KV tiles of parity t (two independent
    //                             partial softmaxes over the same rows, merged inside the CTA at the end).
    // Parity mode doubles the CTA count for the same work -- it is used when pair mode would leave SMs idle.
    using C = TcCfg<D>;
    constexpr int NS = C::NS;
    const int tile0 = parity ? blockIdx.x : 2 * blockIdx.x;  // first (or only) Q tile of this CTA
    // FUSED: the splits of one KV head are adjacent in y (cluster dims (1, n_splits, 1))
    const int kv = FUSED ? blockIdx.y / n_splits : blockIdx.y % Hkv;
    const int split = FUSED ? blockIdx.y % n_splits : blockIdx.y / Hkv;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int u = blockIdx.z;
    if (lpt) {
        // Ragged batch (B <= 64): CTAs are handed out in grid order, so the users are taken LONGEST PREFIX FIRST
        // (blockIdx.z = rank by length, ties by index): a long user started last would run alone at the end
        // (measured at config 5, lengths 1.2-8.2 K: SMs idle 8 % of the kernel).
        __shared__ int s_user;
        if (warp == 0) {
            const int l0 = lane < B ? cu[lane + 1] - cu[lane] : -1;
            const int l1 = lane + 32 < B ? cu[lane + 33] - cu[lane + 32] : -1;
            int rk0 = 0, rk1 = 0;
            for (int k = 0; k < B; ++k) {
                const int lk = __shfl_sync(0xffffffffu, k < 32 ? l0 : l1, k & 31);
                rk0 += (lk > l0 || (lk == l0 && k < lane)) ? 1 : 0;
                rk1 += (lk > l1 || (lk == l1 && k < lane + 32)) ? 1 : 0;
            }
            if (lane < B && rk0 == (int)blockIdx.z) s_user = lane;
            if (lane + 32 < B && rk1 == (int)blockIdx.z) s_user = lane + 32;
        }
        __syncthreads();
        u = s_user;
    }

    const int row_begin = cu[u];
    const int L = cu[u + 1] - row_begin;
    int chunk = (L + n_splits - 1) / n_splits;
    chunk = ((chunk + 127) / 128) * 128;
    const int r0 = split * chunk;
    const int r1 = min(L, r0 + chunk);
    const int n_tiles = r1 > r0 ? (r1 - r0 + BN - 1) / BN : 0;
    const int beams_per_tile = BM / G;
    const int M = n_q * G;
    const bool two = !parity && M > (tile0 + 1) * BM;    // pair mode: does the second Q tile hold any live row?
    const bool both = parity || two;                     // are both accumulator sets in use?
    const size_t split_stride = (size_t)B * n_q * Hq;

    if (!FUSED && n_tiles == 0) {  // empty split: (m, l, o) = (-inf, 0, 0), reading R18
        if (warp >= kFirstSoftmaxWarp) {
            const int t = (warp - kFirstSoftmaxWarp) >> 2;
            const int r = threadIdx.x & 127;
            const int i = (tile0 + (parity ? 0 : t)) * beams_per_tile + r / G, g = r % G;
            if (i < n_q && !(parity && t == 1)) {
                const size_t row = split * split_stride + ((size_t)u * n_q + i) * Hq + kv * G + g;
                pm[row] = -INFINITY; pl[row] = 0.f;
                float4* o4 = reinterpret_cast<float4*>(po + row * D);
                for (int c = 0; c < D / 4; ++c) o4[c] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
        return;
    }

    extern __shared__ unsigned char smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t sQ = smem_base;                       // Q0, Q1
    const uint32_t sKV = sQ + 2 * C::TILE_BYTES;         // NS slots
    const uint32_t sBar = sKV + NS * C::TILE_BYTES;
    // barrier slots (8 bytes each)
    const uint32_t bar_q = sBar;
    const uint32_t bar_full = sBar + 8;                  // [NS] slot filled by TMA
    const uint32_t bar_empty = bar_full + 8 * NS;        // [NS] slot consumed by the tensor pipe
    const uint32_t bar_sfull = bar_empty + 8 * NS;       // [2]  S_t ready (and every earlier MMA done)
    const uint32_t bar_pfull = bar_sfull + 16;           // [2]  P_t written by its warpgroup
    const uint32_t bar_done = bar_pfull + 16;            // all MMAs of this CTA done
    const uint32_t tmem_slot = bar_done + 8;             // uint32
    volatile uint32_t* tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    // Warp 0 lane 0 initialises the barriers and immediately starts the first TMA loads: they only need
    // the barriers, not TMEM, so the HBM latency of Q / K_0 / V_0 ... overlaps the TMEM allocation.
    // The n-th tile through the ring, in the order the tensor pipe consumes them.
    //   pair:   K_0 V_0 K_1 V_1 ...                      n_k(j) = 2j,  n_v(j) = 2j + 1
    //   parity: K_0 K_1 V_0 K_2 V_1 K_3 ... V_{nt-2} V_{nt-1}   n_k(x) = x < 2 ? x : 2x - 1,
    //                                                    n_v(x) = x == nt - 1 ? 2x + 1 : 2x + 2
    int n_issued = 0;
    auto seq_k = [&](int x) { return parity ? (x < 2 ? x : 2 * x - 1) : 2 * x; };
    auto seq_v = [&](int x) { return parity ? (x == n_tiles - 1 ? 2 * x + 1 : 2 * x + 2) : 2 * x + 1; };
    auto issue_kv = [&](int n) {
        bool is_v; int x;
        if (!parity) { is_v = n & 1; x = n >> 1; }
        else if (n_tiles == 1) { is_v = n == 1; x = 0; }
        else if (n < 2) { is_v = false; x = n; }
        else if (n >= 2 * n_tiles - 2) { is_v = true; x = n - n_tiles; }
        else { is_v = !(n & 1); x = is_v ? (n - 2) >> 1 : ((n - 3) >> 1) + 2; }
        const int s = n % NS;
        const int row = row_begin + r0 + x * BN;
        mbar_expect_tx(bar_full + 8 * s, C::TILE_BYTES);
#pragma unroll
        for (int bx = 0; bx < C::BOXES; ++bx)
            tma_load_3d(sKV + s * C::TILE_BYTES + bx * (BN * 128), is_v ? &tm_v : &tm_k, bar_full + 8 * s,
                        bx * 64, kv, row);
    };
    if (threadIdx.x == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_q) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_k) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_v) : "memory");
        if (FUSED) asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_o) : "memory");
        mbar_init(bar_q, 1);
        for (int s = 0; s < NS; ++s) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, 1); }
        for (int t = 0; t < 2; ++t) { mbar_init(bar_sfull + 8 * t, 1); mbar_init(bar_pfull + 8 * t, kSoftmaxThreads / 32); }
        mbar_init(bar_done, 1);
        fence_barrier_init();
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        const int beam0 = u * n_q + tile0 * beams_per_tile;
        if (n_tiles > 0 || (FUSED && fa.level > 0)) {    // (an empty split still needs q for the chain scores)
            mbar_expect_tx(bar_q, (two ? 2 : 1) * C::TILE_BYTES);
            for (int t = 0; t < (two ? 2 : 1); ++t)
#pragma unroll
                for (int bx = 0; bx < C::BOXES; ++bx)
                    tma_load_3d(sQ + t * C::TILE_BYTES + bx * (BM * 128), &tm_q, bar_q, bx * 64, kv * G,
                                beam0 + t * beams_per_tile);
        }
        for (; n_issued < min(NS, 2 * n_tiles); ++n_issued) issue_kv(n_issued);  // the ring starts empty
    }
    if (warp == 1) tmem_alloc(tmem_slot, C::TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot_ptr;

    // identity of a softmax warp (warps 2..9; harmless values for warps 0 and 1)
    const int t = (warp - kFirstSoftmaxWarp) >> 2;      // accumulator set (= warpgroup) of this warp
    const int quarter = warp & 3;                       // TMEM lane quarter this warp may access
    const int r = quarter * 32 + lane;                  // query row inside the Q tile
    const int i = (tile0 + (parity ? 0 : t)) * beams_per_tile + r / G, g = r % G;
    const bool live = warp >= kFirstSoftmaxWarp && i < n_q;
    const bool warp_live = __any_sync(0xffffffffu, live);
    const uint32_t lane_addr = tmem + ((uint32_t)(quarter * 32) << 16);
    const uint32_t aO = lane_addr + C::COL_O + t * 128;
    float m_ref = -INFINITY, l_sum = 0.f;               // m_ref in log2 units of the scaled score
    // fused mode: who finishes this warp's 32-row block (see the tail below)
    const bool mine = FUSED && warp >= kFirstSoftmaxWarp && (t == 0 || two) && warp_live;  // the block has live rows
    const int blk = t * 4 + quarter;                    // 32-row block of the CTA's (up to) 256 rows
    const int owner = blk % n_splits, ob = blk / n_splits;                 // cluster rank that finishes it
    const uint32_t me = (FUSED && n_splits > 1) ? cluster_rank() : 0u;
    // parity mode without splits: only blocks 0..3 finish, ring slots 4..7 are free for the chain's V rows
    const bool vpre = FUSED && parity && n_splits == 1 && mine && fa.level > 0;
    float ch_y[8];                                      // chain scores, later weights (fused mode)
    uint32_t ch_off[8];                                 // chain row offsets in the suffix buffers

    // Register budget (setmaxnreg works on whole, aligned warpgroups): warpgroup 0 holds the two single-thread
    // roles and gives registers back; the softmax warpgroups take them -- a thread keeps its whole S row
    // (128 fp32) in registers between the row maximum and the exponentials.
    // (The limits are set at the top of each role's branch, and the fused tail lives inside the softmax
    // branch: code after a join of the branches would have to fit the smallest budget.)
    if (warp < kFirstSoftmaxWarp) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        if (warp == 0) {
        // ===================== TMA producer (rest of the stream) =====================
        if (lane == 0) {
            for (int n = n_issued; n < 2 * n_tiles; ++n) {
                mbar_wait(bar_empty + 8 * (n % NS), (uint32_t)(((n / NS) & 1) ^ 1));
                issue_kv(n);
            }
        }
        } else if (warp == 1) {
        // ===================== MMA issuer =====================
        if (lane == 0 && n_tiles > 0) {
            constexpr uint32_t idesc_s = instr_desc(BM, BN, 0);
            constexpr uint32_t idesc_o = instr_desc(BM, D, 1);
            // S_t = Q_t K_j^T; K_j sits in ring slot s
            auto issue_qk = [&](int t, int s) {
                const uint32_t d_tmem = tmem + C::COL_S + t * BN;
#pragma unroll
                for (int k = 0; k < D / 16; ++k) {
                    const uint32_t off = (k / 4) * (BM * 128) + (k % 4) * 32;  // box, then 32 B per K=16 step
                    umma_ss(d_tmem, smem_desc(sQ + (parity ? 0 : t) * C::TILE_BYTES + off, 16, 1024),
                            smem_desc(sKV + s * C::TILE_BYTES + off, 16, 1024), idesc_s, k > 0 ? 1u : 0u);
                }
                umma_commit(bar_sfull + 8 * t);
            };
            // O_t (+)= P_t V_j; V tile: [kv row][64 d] boxes, MN-major B operand; 16 kv rows = 2048 B per K step
            auto issue_pv = [&](int t, int s, bool acc) {
#pragma unroll
                for (int k = 0; k < BN / 16; ++k)
                    umma_ts(tmem + C::COL_O + t * 128, tmem + C::COL_S + t * BN + k * 8,
                            smem_desc(sKV + s * C::TILE_BYTES + k * 2048, BN * 128, 1024), idesc_o,
                            (acc || k > 0) ? 1u : 0u);
            };
            auto slot_of = [&](int n) { return n % NS; };
            auto wait_full = [&](int n) { mbar_wait(bar_full + 8 * slot_of(n), (uint32_t)((n / NS) & 1)); tc_fence_after(); };
            mbar_wait(bar_q, 0);
            if (!parity) {
                // PV0_j, QK0_{j+1}, PV1_j, QK1_{j+1}: one Q tile's MMAs run while the other's softmax does
                const int nt = two ? 2 : 1;
                wait_full(0);
                for (int t = 0; t < nt; ++t) issue_qk(t, slot_of(0));
                umma_commit(bar_empty + 8 * slot_of(0));
                for (int j = 0; j < n_tiles; ++j) {
                    const bool more = j + 1 < n_tiles;
                    TCPROF(j, 13);
                    wait_full(2 * j + 1);                    // V_j
                    if (more) wait_full(2 * j + 2);          // K_{j+1}
                    TCPROF(j, 12);
                    for (int t = 0; t < nt; ++t) {
                        mbar_wait(bar_pfull + 8 * t, (uint32_t)(j & 1));
                        tc_fence_after();
                        TCPROF(j, 8 + 2 * t);
                        issue_pv(t, slot_of(2 * j + 1), j > 0);
                        if (more) issue_qk(t, slot_of(2 * j + 2));
                        TCPROF(j, 9 + 2 * t);
                    }
                    umma_commit(bar_empty + 8 * slot_of(2 * j + 1));
                    if (more) umma_commit(bar_empty + 8 * slot_of(2 * j + 2));
                }
            } else {
                // KV tile x belongs to accumulator set x & 1: PV_t(x), QK_t(x + 2), alternating t
                for (int x = 0; x < min(2, n_tiles); ++x) {
                    wait_full(seq_k(x));
                    issue_qk(x, slot_of(seq_k(x)));
                    umma_commit(bar_empty + 8 * slot_of(seq_k(x)));
                }
                for (int x = 0; x < n_tiles; ++x) {
                    const int t = x & 1;
                    wait_full(seq_v(x));
                    mbar_wait(bar_pfull + 8 * t, (uint32_t)((x >> 1) & 1));
                    tc_fence_after();
                    issue_pv(t, slot_of(seq_v(x)), x >= 2);
                    umma_commit(bar_empty + 8 * slot_of(seq_v(x)));
                    if (x + 2 < n_tiles) {
                        wait_full(seq_k(x + 2));
                        issue_qk(t, slot_of(seq_k(x + 2)));
                        umma_commit(bar_empty + 8 * slot_of(seq_k(x + 2)));
                    }
                }
            }
            umma_commit(bar_done);
        }
        }
        else if (FUSED && fa.kn != nullptr && split == 0 && fa.level > 0) {
        // ===================== inline KV append + index reorganisation (stark_decode_step) =====================
        // PAPER.md:284-286.  Warps 2 and 3 of the first split: the K/V rows of this CTA's beams and KV head go
        // into the suffix level; the CTAs of KV head 0 also extend the ancestor index.  Nothing in this launch
        // reads what is written here (a query's own row comes from kn / vn, its ancestors from lower levels).
        const int tid = threadIdx.x - 64;
        const int b0 = tile0 * beams_per_tile, nb = min(n_q, b0 + (parity ? 1 : 2) * beams_per_tile) - b0;
        constexpr int VPR = D / 8;                       // 16-byte vectors per row
        const size_t lvl_off = (size_t)(fa.level - 1) * B * fa.Wmax * Hkv * D;
        const int per = nb * VPR;
#pragma unroll 2
        for (int idx = tid; idx < 2 * per; idx += 64) {
            const int which = idx >= per, rem = idx - which * per, i2 = b0 + rem / VPR, c = rem % VPR;
            const __nv_bfloat16* src = (which ? fa.vn : fa.kn) + (((size_t)u * n_q + i2) * Hkv + kv) * D;
            __nv_bfloat16* dst = const_cast<__nv_bfloat16*>(which ? fa.vs : fa.ks) + lvl_off +
                                 (((size_t)u * fa.Wmax + i2) * Hkv + kv) * D;
            reinterpret_cast<uint4*>(dst)[c] = __ldg(reinterpret_cast<const uint4*>(src) + c);
        }
        if (fa.anc_new != nullptr && kv == 0)
            for (int bi = tid; bi < nb; bi += 64) {
                const int i2 = b0 + bi;
                int32_t* row = fa.anc_new + ((size_t)u * fa.Wmax + i2) * fa.d;
                if (fa.level >= 2) {
                    const int par = min(max(__ldg(fa.parent + (size_t)u * n_q + i2), 0), fa.Wmax - 1);
                    const int32_t* prow = fa.anc + ((size_t)u * fa.Wmax + par) * fa.d;
                    for (int t2 = 0; t2 < fa.level - 1; ++t2) row[t2] = __ldg(prow + t2);
                }
                row[fa.level - 1] = i2;
            }
        }
        if (FUSED && n_splits > 1) {                     // the two cluster barriers of the fused tail (B1, B2)
            __syncwarp();
            cluster_sync_all();
            cluster_sync_all();
        }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
        // ===================== softmax / correction / epilogue =====================
        // pair mode without splits: the chain's part of the row stays in registers until the tail (see below)
        const bool single = SINGLE && mine;
        float m_c = -INFINITY, l_c = 0.f;
        float vs[SINGLE ? D : 1];
        if (t == 0 || both) {
            const uint32_t aS = lane_addr + C::COL_S + t * BN;
            const int my_tiles = parity ? (n_tiles - t + 1) / 2 : n_tiles;  // KV tiles of this accumulator set
            for (int j = 0; j < my_tiles; ++j) {
                if (quarter == 0 && lane == 0) TCPROF(j, 4 * t + 0);
                mbar_wait(bar_sfull + 8 * t, (uint32_t)(j & 1));
                __syncwarp();
                if (quarter == 0 && lane == 0) TCPROF(j, 4 * t + 1);
                if (warp_live) {                        // warps without live rows only keep the barrier count
                    tc_fence_after();
                    const int x = parity ? 2 * j + t : j;            // KV tile of the split
                    const int valid = min(BN, r1 - (r0 + x * BN));   // columns of this tile inside the split
                    // the whole S row (128 fp32) into registers; the maximum of its first half is taken while
                    // the second half is still on its way from TMEM
                    uint32_t sr[4][32];
                    tmem_ld32(aS, sr[0]);
                    tmem_ld32(aS + 32, sr[1]);
                    tmem_wait_ld();
                    tmem_ld32(aS + 64, sr[2]);
                    tmem_ld32(aS + 96, sr[3]);
                    if (quarter == 0 && lane == 0) TCPROF(j, 4 * t + 2);
                    // 4 independent running maxima: with two warps per scheduler a single 128-long dependent
                    // chain (4 cycles per link) would cost as much as the exponentials themselves
                    float tm0 = -INFINITY, tm1 = -INFINITY, tm2 = -INFINITY, tm3 = -INFINITY;
                    auto max_half = [&](int c0) {
#pragma unroll
                        for (int c = c0; c < c0 + 2; ++c)
#pragma unroll
                            for (int x = 0; x < 32; x += 4) {
                                tm0 = fmaxf(tm0, __uint_as_float(sr[c][x]));
                                tm1 = fmaxf(tm1, __uint_as_float(sr[c][x + 1]));
                                tm2 = fmaxf(tm2, __uint_as_float(sr[c][x + 2]));
                                tm3 = fmaxf(tm3, __uint_as_float(sr[c][x + 3]));
                            }
                    };
                    auto mask_half = [&](int c0) {              // columns beyond the split: -inf (exp2 gives 0)
#pragma unroll
                        for (int c = c0; c < c0 + 2; ++c)
#pragma unroll
                            for (int x = 0; x < 32; ++x)
                                if (c * 32 + x >= valid) sr[c][x] = 0xff800000u;
                    };
                    if (valid < BN) mask_half(0);
                    max_half(0);
                    tmem_wait_ld();
                    if (valid < BN) mask_half(2);
                    max_half(2);
                    float tmax = fmaxf(fmaxf(tm0, tm1), fmaxf(tm2, tm3));
                    tmax *= scale_log2;
                    // lazy rescale: keep the reference maximum unless the row maximum grew by > 2^8
                    bool grow = false;
                    float m_new = m_ref;
                    if (j == 0) m_new = tmax;
                    else if (tmax > m_ref + kRescaleThreshold) { m_new = tmax; grow = true; }
                    if (__any_sync(0xffffffffu, grow)) {
                        // S_t(j) ready => PV_t(j-1) completed (in-order tensor pipe): O_t is quiescent
                        const float alpha = grow ? fast_exp2(m_ref - m_new) : 1.0f;
#pragma unroll 1
                        for (int c = 0; c < D / 32; ++c) {
                            uint32_t o[32];
                            tmem_ld32(aO + c * 32, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int x = 0; x < 32; ++x) o[x] = __float_as_uint(__uint_as_float(o[x]) * alpha);
                            tmem_st32(aO + c * 32, o);
                        }
                        l_sum *= alpha;
                    }
                    m_ref = m_new;
                    // P = exp2(s * scale - m_ref) as bf16, written over S in place (P chunk c covers columns
                    // [16c, 16c+16) of the S region, whose contents are already in registers)
                    const float neg_m = -m_ref;
                    float ps0 = 0.f, ps1 = 0.f;             // independent partial sums (same reason)
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        uint32_t pk[16];
#pragma unroll
                        for (int x = 0; x < 32; x += 2) {
                            const float p0 = fast_exp2(fmaf(__uint_as_float(sr[c][x]), scale_log2, neg_m));
                            const float p1 = fast_exp2(fmaf(__uint_as_float(sr[c][x + 1]), scale_log2, neg_m));
                            ps0 += p0; ps1 += p1;
                            const __nv_bfloat162 h = __floats2bfloat162_rn(p0, p1);  // element 2x in the low half
                            pk[x >> 1] = *reinterpret_cast<const uint32_t*>(&h);
                        }
                        tmem_st16(aS + c * 16, pk);
                    }
                    l_sum += ps0 + ps1;
                    tmem_wait_st();
                    tc_fence_before();
                    if (quarter == 0 && lane == 0) TCPROF(j, 4 * t + 3);
                }
                __syncwarp();                           // every lane's P is written and fenced: one arrival per warp
                if (lane == 0) mbar_arrive(bar_pfull + 8 * t);
            }
            // ---- epilogue: O row -> partials ----
            if (FUSED && fa.level > 0 && n_tiles == 0) mbar_wait(bar_q, 0);   // (otherwise S was ready: so was Q)
            if (FUSED && mine && owner == (int)me && live && fa.level > 0)  // inside the wait for the last MMAs
                chain_scores<D>(fa, scale_log2, u, i, kv, n_q, Hkv, B,
                                smem_raw + (sQ - smem_u32(smem_raw)) + (parity ? 0 : t) * C::TILE_BYTES, r, ch_y, ch_off);
            // pair mode without splits: the chain's weighted V sum, relative to the chain's own maximum, one level
            // (one global round trip) at a time, also inside that wait
            if constexpr (SINGLE) if (single) {
#pragma unroll
                for (int x = 0; x < D; ++x) vs[x] = 0.f;
                if (live && fa.level > 0) {
#pragma unroll 1
                    for (int t2 = 0; t2 < fa.level; ++t2) m_c = fmaxf(m_c, ch_y[t2]);
#pragma unroll 1
                    for (int t2 = 0; t2 < fa.level; ++t2) {
                        const float e = fast_exp2(ch_y[t2] - m_c);
                        l_c += e;
                        const uint4* vp = reinterpret_cast<const uint4*>(((fa.vn && t2 == fa.level - 1) ? fa.vn : fa.vs) + ch_off[t2]);
                        uint4 vv[D / 8];
#pragma unroll
                        for (int c = 0; c < D / 8; ++c) vv[c] = __ldg(vp + c);
#pragma unroll
                        for (int c = 0; c < D / 8; ++c) {
                            const uint32_t va[4] = {vv[c].x, vv[c].y, vv[c].z, vv[c].w};
#pragma unroll
                            for (int e2 = 0; e2 < 4; ++e2) {
                                vs[c * 8 + 2 * e2] = fmaf(e, __uint_as_float(va[e2] << 16), vs[c * 8 + 2 * e2]);
                                vs[c * 8 + 2 * e2 + 1] = fmaf(e, __uint_as_float(va[e2] & 0xffff0000u), vs[c * 8 + 2 * e2 + 1]);
                            }
                        }
                    }
                }
            }
            if (FUSED && vpre) {
                // The V rows of the first two chain levels of this warp's 32 rows go to ring bytes [4, 8) * 32*D*4
                // (K/V ring tiles 2 and 3; unused by the tail in parity mode without splits) asynchronously, as
                // soon as the tensor pipe has released those two tiles for the last time -- normally long before
                // the last MMA, so the copies are issued inside the wait for it and land during the in-CTA merge.
                // (A trace showed the tail paying one dependent round of V loads per 32-column chunk: 4 x ~1.2 k
                // cycles.)  The WARP copies row after row, D/8 lanes per row: whole lines per request (lane-per-row
                // copies cost 32 line slots of the load unit each: 4 k cycles).
                for (int sl = 2; sl <= 3; ++sl)
                    if (2 * n_tiles > sl) {
                        const int n_last = sl + ((2 * n_tiles - 1 - sl) / NS) * NS;   // last tile through this slot
                        mbar_wait(bar_empty + 8 * sl, (uint32_t)((n_last / NS) & 1));
                    }
                constexpr int LPR = D / 8, RPI = 32 / LPR;
                const int sub = lane % LPR, grp = lane / LPR;
                const uint32_t live_mask = __ballot_sync(0xffffffffu, live);
                const uint32_t dst0 = sKV + (uint32_t)(4 + quarter) * (32 * D * 4);
                const int nlv = min(fa.level, 2);
                for (int lv = 0; lv < nlv; ++lv) {
                    const __nv_bfloat16* vbase = (fa.vn && lv == fa.level - 1) ? fa.vn : fa.vs;
                    const uint32_t my_off = live ? ch_off[lv] : 0u;
#pragma unroll 4
                    for (int p = 0; p < 32 / RPI; ++p) {
                        const int row = p * RPI + grp;
                        const uint32_t off = __shfl_sync(0xffffffffu, my_off, row);
                        if ((live_mask >> row) & 1u)
                            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst0 + (uint32_t)((lv * 32 + row) * (D * 2) + ((sub ^ (row & 7)) * 16))),
                                         "l"(reinterpret_cast<const uint4*>(vbase + off) + sub) : "memory");
                    }
                }
                asm volatile("cp.async.commit_group;" ::: "memory");
            }
            if (n_tiles > 0) mbar_wait(bar_done, 0);
            __syncwarp();
            if (parity) {
                // ---- parity mode: fold accumulator set 1 (odd KV tiles) into set 0 inside the CTA ----
                // set 1's rows go through the (now idle) K/V ring: block `quarter`, chunks XOR-swizzled by row
                constexpr int CPRm = D / 4;
                unsigned char* ring = smem_raw + (sKV - smem_u32(smem_raw));
                float* mrow = reinterpret_cast<float*>(ring) + (size_t)quarter * 32 * D + lane * D;
                float2* mml = reinterpret_cast<float2*>(ring + 8 * 32 * D * 4) + quarter * 32 + lane;
                if (t == 1 && warp_live) {
                    tc_fence_after();
                    *mml = make_float2(m_ref, l_sum);
                    if (my_tiles > 0) {
#pragma unroll 1
                        for (int c = 0; c < D / 32; ++c) {
                            uint32_t o[32];
                            tmem_ld32(aO + c * 32, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int x = 0; x < 32; x += 4)
                                *reinterpret_cast<float4*>(mrow + (((c * 8 + (x >> 2)) ^ (lane & (CPRm - 1))) * 4)) =
                                    make_float4(__uint_as_float(o[x]), __uint_as_float(o[x + 1]),
                                                __uint_as_float(o[x + 2]), __uint_as_float(o[x + 3]));
                        }
                    }
                }
                asm volatile("bar.sync 2, 256;" ::: "memory");  // the two softmax warpgroups
                if (t == 0 && warp_live) {
                    const float2 ml = *mml;
                    if (ml.x > -INFINITY) {             // set 1 saw at least one KV tile (so did set 0)
                        tc_fence_after();
                        const float m = fmaxf(m_ref, ml.x);
                        const float a0 = fast_exp2(m_ref - m), a1 = fast_exp2(ml.x - m);
#pragma unroll 1
                        for (int c = 0; c < D / 32; ++c) {
                            uint32_t o[32];
                            tmem_ld32(aO + c * 32, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int x = 0; x < 32; x += 4) {
                                const float4 v = *reinterpret_cast<const float4*>(mrow + (((c * 8 + (x >> 2)) ^ (lane & (CPRm - 1))) * 4));
                                o[x] = __float_as_uint(fmaf(a1, v.x, a0 * __uint_as_float(o[x])));
                                o[x + 1] = __float_as_uint(fmaf(a1, v.y, a0 * __uint_as_float(o[x + 1])));
                                o[x + 2] = __float_as_uint(fmaf(a1, v.z, a0 * __uint_as_float(o[x + 2])));
                                o[x + 3] = __float_as_uint(fmaf(a1, v.w, a0 * __uint_as_float(o[x + 3])));
                            }
                            tmem_st32(aO + c * 32, o);
                        }
                        tmem_wait_st();
                        l_sum = a0 * l_sum + a1 * ml.y;
                        m_ref = m;
                    }
                }
            }
            if (!FUSED && warp_live && !(parity && t == 1)) {
                tc_fence_after();
                // Each thread owns one O row (512 B), so direct stores would scatter 16-byte pieces over 32
                // rows per instruction (measured: 5.5 us for 17 MB).  Stage the warp's 32 rows in the (now
                // idle) K/V ring, 16-byte chunks XOR-swizzled by row, then write whole rows coalesced.
                constexpr int CPR = D / 4;              // 16-byte chunks per row
                float* stage = reinterpret_cast<float*>(smem_raw + (sKV - smem_u32(smem_raw))) + (size_t)(t * 4 + quarter) * 32 * D;
#pragma unroll
                for (int c = 0; c < D / 32; ++c) {
                    uint32_t o[32];
                    tmem_ld32(aO + c * 32, o);
                    tmem_wait_ld();
#pragma unroll
                    for (int x = 0; x < 32; x += 4) {
                        const int ch = (c * 8 + (x >> 2)) ^ (lane & (CPR - 1));
                        *reinterpret_cast<float4*>(stage + lane * D + ch * 4) =
                            make_float4(__uint_as_float(o[x]), __uint_as_float(o[x + 1]), __uint_as_float(o[x + 2]),
                                        __uint_as_float(o[x + 3]));
                    }
                }
                const size_t row_base = split * split_stride + (size_t)u * n_q * Hq + kv * G;
                if (live) { pm[row_base + (size_t)i * Hq + g] = m_ref * kLn2; pl[row_base + (size_t)i * Hq + g] = l_sum; }
                __syncwarp();
                for (int idx = lane; idx < 32 * CPR; idx += 32) {
                    const int l2 = idx / CPR, ch = idx % CPR;
                    const int r2 = quarter * 32 + l2;
                    const int i2 = (tile0 + (parity ? 0 : t)) * beams_per_tile + r2 / G, g2 = r2 % G;
                    if (i2 < n_q)
                        *reinterpret_cast<float4*>(po + (row_base + (size_t)i2 * Hq + g2) * D + ch * 4) =
                            *reinterpret_cast<const float4*>(stage + l2 * D + ((ch ^ (l2 & (CPR - 1))) * 4));
                }
                tc_fence_before();
            }
        }
        if constexpr (FUSED) {
            constexpr uint32_t SLOT = 32 * D * 4;                          // one block of fp32 O rows
            const uint32_t ml_base = sKV + 8 * SLOT;                       // (m, l) pairs: [slot][32][2]
            // B1: every CTA of the cluster is done with its K/V ring, which now becomes the exchange buffer
            if (n_splits > 1) cluster_sync_all();
            if (mine && owner != (int)me) {
                tc_fence_after();
                const uint32_t slot = (uint32_t)(ob * n_splits) + me;
                const uint32_t dst = map_to_rank(sKV + slot * SLOT + (uint32_t)lane * D * 4, (uint32_t)owner);
                constexpr int CPR = D / 4;
#pragma unroll 1
                for (int c = 0; c < D / 32; ++c) {
                    uint32_t o[32];
                    tmem_ld32(aO + c * 32, o);
                    tmem_wait_ld();
#pragma unroll
                    for (int x = 0; x < 32; x += 4) {
                        const int ch = (c * 8 + (x >> 2)) ^ (lane & (CPR - 1));
                        if (n_tiles > 0)
                            st_cluster_f4(dst + ch * 16, __uint_as_float(o[x]), __uint_as_float(o[x + 1]),
                                          __uint_as_float(o[x + 2]), __uint_as_float(o[x + 3]));
                        else
                            st_cluster_f4(dst + ch * 16, 0.f, 0.f, 0.f, 0.f);  // empty split: (-inf, 0, 0)
                    }
                }
                st_cluster_f2(map_to_rank(ml_base + slot * 256 + (uint32_t)lane * 8, (uint32_t)owner), m_ref, l_sum);
            }
            if (n_splits > 1) cluster_sync_all();                          // B2: all partial rows delivered
            if constexpr (SINGLE) {
                if (single)
                    fused_finish_single<D>(fa, smem_raw, sKV - smem_u32(smem_raw), blk, lane, aO, n_tiles > 0, m_ref,
                                           l_sum, u, n_q, Hq, G, kv, (tile0 + t) * beams_per_tile, quarter, m_c, l_c, vs,
                                           &tm_o);
            } else if (mine && owner == (int)me) {
                if (vpre) { asm volatile("cp.async.wait_group 0;" ::: "memory"); __syncwarp(); }
                fused_finish<D>(fa, smem_raw, sKV - smem_u32(smem_raw), ob, (int)me, n_splits, lane, aO, n_tiles > 0, m_ref,
                                l_sum, u, n_q, Hq, G, kv, (tile0 + (parity ? 0 : t)) * beams_per_tile, quarter, ch_y, ch_off,
                                vpre ? smem_raw + (sKV - smem_u32(smem_raw)) + (size_t)(4 + quarter) * (32 * D * 4) : nullptr,
                                &tm_o);
            }
            tc_fence_before();
        }
    }
    __syncthreads();
    if (warp == 1) {
        __syncwarp();
        tc_fence_after();
        tmem_dealloc(tmem, C::TMEM_COLS);
    }
}

// ---- host side ----------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        else
            (void)cudaGetLastError();
    }
    return fn;
}

// bf16 tensor [n2][n1][D] (D contiguous, rows of n1*D), box = 64 x box1 x box2, 128-byte swizzle
bool make_map(CUtensorMap* tm, const void* base, int D, int n1, long long n2, int box1, int box2) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return false;
    cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)n1, (cuuint64_t)n2};
    cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)n1 * D * 2};
    cuuint32_t box[3] = {64, (cuuint32_t)box1, (cuuint32_t)box2};
    cuuint32_t estr[3] = {1, 1, 1};
    return fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// bf16 tensor out[B][n_q][Hq][D] as a 4-d map; box = 64 columns x hb heads x bb beams x 1 user (the 32 rows a warp
// finishes), 128-byte swizzle
bool make_map_out(CUtensorMap* tm, const void* base, int D, int Hq, int n_q, int B, int G) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return false;
    const int hb = G < 32 ? G : 32, bb = 32 / hb;
    cuuint64_t dims[4] = {(cuuint64_t)D, (cuuint64_t)Hq, (cuuint64_t)n_q, (cuuint64_t)B};
    cuuint64_t strides[3] = {(cuuint64_t)D * 2, (cuuint64_t)Hq * D * 2, (cuuint64_t)n_q * Hq * D * 2};
    cuuint32_t box[4] = {64, (cuuint32_t)hb, (cuuint32_t)bb, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    return fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int D>
int launch_d(const Dims& p, const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv, int n_q,
             const int32_t* cu, int n_splits, int lpt, float* pm, float* pl, float* po, cudaStream_t st) {
    static PerDevice<bool> attr_done;
    if (!attr_done.here()) {
        STARK_CUDA_TRY(cudaFuncSetAttribute(prefix_tc_kernel<D, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            TcCfg<D>::SMEM_BYTES));
        attr_done.here() = true;
    }
    const int M = n_q * p.G;
    const int parity = prefix_tc_parity(p, n_q, n_splits) ? 1 : 0;
    const int rows_per_cta = parity ? BM : 2 * BM;                  // one Q tile, or a pair of them
    dim3 grid((M + rows_per_cta - 1) / rows_per_cta, p.Hkv * n_splits, p.B);
    prefix_tc_kernel<D, false><<<grid, kThreadsTC, TcCfg<D>::SMEM_BYTES, st>>>(
        tq, tk, tv, tq /*unused*/, cu, pm, pl, po, p.B, n_q, p.Hq, p.Hkv, p.G, n_splits, p.scale * kLog2e, parity, lpt,
        FusedArgs{});
    STARK_LAUNCH_CHECK();
    return STARK_OK;
}

// fused launch: the n_splits CTAs of one (pair, KV head, user) are a cluster along y
template <int D>
int launch_fused_d(const Dims& p, const CUtensorMap& tq, const CUtensorMap& tk, const CUtensorMap& tv,
                   const CUtensorMap& to, int n_q, const int32_t* cu, int n_splits, int lpt, const FusedArgs& fa, cudaStream_t st) {
    static PerDevice<bool> attr_done;
    if (!attr_done.here()) {
        STARK_CUDA_TRY(cudaFuncSetAttribute(prefix_tc_kernel<D, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            TcCfg<D>::SMEM_BYTES));
        STARK_CUDA_TRY(cudaFuncSetAttribute(prefix_tc_kernel<D, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            TcCfg<D>::SMEM_BYTES));
        attr_done.here() = true;
    }
    const int M = n_q * p.G;
    const int parity = prefix_tc_parity(p, n_q, n_splits) ? 1 : 0;
    const int rows_per_cta = parity ? BM : 2 * BM;
    const bool single = !parity && n_splits == 1 && fa.level > 0;   // see the kernel's template parameters
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((M + rows_per_cta - 1) / rows_per_cta, p.Hkv * n_splits, p.B);
    cfg.blockDim = dim3(kThreadsTC);
    cfg.dynamicSmemBytes = TcCfg<D>::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 1; at[0].val.clusterDim.y = n_splits; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = n_splits > 1 ? 1 : 0;   // a single split needs no cluster launch
    STARK_CUDA_TRY(cudaLaunchKernelEx(&cfg, single ? prefix_tc_kernel<D, true, true> : prefix_tc_kernel<D, true, false>,
                                      tq, tk, tv, to, cu, (float*)nullptr, (float*)nullptr, (float*)nullptr, p.B, n_q,
                                      p.Hq, p.Hkv, p.G, n_splits, p.scale * kLog2e, parity, lpt, fa));
    return STARK_OK;
}

}  // namespace

// Parity mode (one Q tile per CTA, KV tiles alternating between the two accumulator sets) whenever its
// doubled CTA count still fits the GPU in one wave, and always for a single Q tile; pair mode (K/V staged once
// per 256 rows) otherwise.
bool prefix_tc_parity(const Dims& p, int n_q, int n_splits) {
    const int sms = num_sms() > 0 ? num_sms() : 148;
    const long long tiles_m = ((long long)n_q * p.G + BM - 1) / BM;
    // a single Q tile (decode step 0 above all): pair mode would have the same CTA count and leave the second
    // accumulator set idle -- every KV tile strictly after the other (config 3 step 0: 58 us for a 21 us stream)
    if (tiles_m == 1) return true;
    return tiles_m * p.Hkv * p.B * n_splits <= sms;
}

// Longest-prefix-first CTA order pays only for ragged batches; the kernel's ranking handles up to 64 users.
static int ragged_batch(const Dims& p, int total_tokens, int max_len) {
    return (p.B >= 2 && p.B <= 64 && (long long)max_len * p.B != (long long)total_tokens) ? 1 : 0;
}

bool prefix_tc_supported(const Dims& p, int dtype, int n_q) {
    if (dtype != STARK_BF16) return false;
    if (p.D != 64 && p.D != 128) return false;
    (void)n_q;  // any number of queries: step 0 (M = G rows) streams the prefix through the same kernel
    return p.G <= BM && (BM % p.G) == 0;
}

int launch_prefix_tc(const Dims& p, const void* q, int n_q, const void* k, const void* v, const int32_t* cu,
                     int total_tokens, int max_len, int n_splits, float* pm, float* pl, float* po, cudaStream_t st) {
    if (total_tokens < 1)
        return launch_prefix_simt(p, STARK_BF16, q, n_q, k, v, cu, n_splits, pm, pl, po, st);
    CUtensorMap tq, tk, tv;
    if (!make_map(&tq, q, p.D, p.Hq, (long long)p.B * n_q, p.G, BM / p.G) ||
        !make_map(&tk, k, p.D, p.Hkv, total_tokens, 1, BN) || !make_map(&tv, v, p.D, p.Hkv, total_tokens, 1, BN)) {
        last_cuda_error_ref() = (int)cudaErrorInvalidValue;
        return STARK_ERR_CUDA;
    }
    const int lpt = ragged_batch(p, total_tokens, max_len);
    if (p.D == 128) return launch_d<128>(p, tq, tk, tv, n_q, cu, n_splits, lpt, pm, pl, po, st);
    return launch_d<64>(p, tq, tk, tv, n_q, cu, n_splits, lpt, pm, pl, po, st);
}

// A1 + A2 in one launch (bf16): n_splits in {1, 2, 4, 8} = cluster size along the prefix.
int launch_decode_fused(const Dims& p, const void* q, int n_q, int level, const void* k, const void* v,
                        const int32_t* cu, int total_tokens, int max_len, int n_splits, const void* ks, const void* vs,
                        const int32_t* anc_level, void* out, cudaStream_t st, const void* kn, const void* vn,
                        const int32_t* parent, int32_t* anc_new) {
    CUtensorMap tq, tk, tv, to;
    if (!make_map(&tq, q, p.D, p.Hq, (long long)p.B * n_q, p.G, BM / p.G) ||
        !make_map(&tk, k, p.D, p.Hkv, total_tokens, 1, BN) || !make_map(&tv, v, p.D, p.Hkv, total_tokens, 1, BN) ||
        !make_map_out(&to, out, p.D, p.Hq, n_q, p.B, p.G)) {
        last_cuda_error_ref() = (int)cudaErrorInvalidValue;
        return STARK_ERR_CUDA;
    }
    FusedArgs fa;
    fa.q = (const __nv_bfloat16*)q; fa.ks = (const __nv_bfloat16*)ks; fa.vs = (const __nv_bfloat16*)vs;
    fa.anc = anc_level; fa.out = (__nv_bfloat16*)out;
    fa.level = level; fa.Wmax = p.Wmax; fa.d = p.d; fa.scale = p.scale;
    fa.kn = (const __nv_bfloat16*)kn; fa.vn = (const __nv_bfloat16*)vn; fa.parent = parent; fa.anc_new = anc_new;
    const int lpt = ragged_batch(p, total_tokens, max_len);
    if (p.D == 128) return launch_fused_d<128>(p, tq, tk, tv, to, n_q, cu, n_splits, lpt, fa, st);
    return launch_fused_d<64>(p, tq, tk, tv, to, n_q, cu, n_splits, lpt, fa, st);
}

}  // namespace stark

#ifdef STARK_TC_PROF
extern "C" int stark_debug_tc_prof(long long* host_out) {
    return (int)cudaMemcpyFromSymbol(host_out, stark::g_tc_prof, sizeof(stark::g_tc_prof));
}
#endif
