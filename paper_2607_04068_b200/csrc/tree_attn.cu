// A2: stark_tree_attn_step -- suffix tree attention + log-sum-exp merge with the
// shared-prefix partials.
//
// PAPER.md:263-268 (Eq. 14): "Each token can only attend to its ancestor nodes
// in the decoding tree and itself."  The mask is never materialised: each
// (query, head) walks its <= d ancestor slots through the pre-computed index
// mapping `anc` and reads K/V rows that are stored once per
// tree node.  The scores of those <= d rows are merged with the n_splits
// prefix partials (m, l, o) by log-sum-exp and the result is normalised.
//
// Byte-bound (<= 4*level*D flops per (query, head)): q + partials + chain rows
// + out, and at these sizes latency-bound: a cold
// dependent global access costs > 1 us on B200, so the kernel is built to have
// exactly two of them in sequence (anc -> K/V row) and to keep every other byte
// in flight at once without spending registers on it:
//   * one WARP per (user, beam, KV head); it serves all G query heads of the
//     GQA group, so the chain's K/V rows are fetched once per group;
//   * the G q rows and the G partial-o rows of split 0 (both contiguous in
//     memory) and the chain rows are copied global -> shared with cp.async
//     (16 bytes per lane, no register staging), into a private per-warp
//     region; only warp-level synchronisation is used;
//   * lane owns EPL = D/32 consecutive head-dim elements; dot products reduce
//     with xor-shuffles across the warp;
//   * further prefix splits (n_splits > 1 happens only when there are few
//     queries) are streamed straight from global memory.
#include "common.cuh"

namespace stark {

namespace {

constexpr int kThreads = 256;
constexpr int kWarpsPerCta = kThreads / 32;
constexpr int kMaxLevels = 8;

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
    asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}

// EPL consecutive elements of T (shared or global) -> float[EPL]; float[EPL] -> EPL elements of T
template <typename T, int EPL> struct Pack;
template <> struct Pack<float, 4> {
    static __device__ __forceinline__ void ld(const float* p, float (&o)[4]) {
        const float4 r = *reinterpret_cast<const float4*>(p);
        o[0] = r.x; o[1] = r.y; o[2] = r.z; o[3] = r.w;
    }
    static __device__ __forceinline__ void st(float* p, const float (&o)[4]) {
        *reinterpret_cast<float4*>(p) = make_float4(o[0], o[1], o[2], o[3]);
    }
};
template <> struct Pack<float, 2> {
    static __device__ __forceinline__ void ld(const float* p, float (&o)[2]) {
        const float2 r = *reinterpret_cast<const float2*>(p);
        o[0] = r.x; o[1] = r.y;
    }
    static __device__ __forceinline__ void st(float* p, const float (&o)[2]) {
        *reinterpret_cast<float2*>(p) = make_float2(o[0], o[1]);
    }
};
template <> struct Pack<__nv_bfloat16, 4> {
    static __device__ __forceinline__ void ld(const __nv_bfloat16* p, float (&o)[4]) {
        const float4 r = ld4(p);
        o[0] = r.x; o[1] = r.y; o[2] = r.z; o[3] = r.w;
    }
    static __device__ __forceinline__ void st(__nv_bfloat16* p, const float (&o)[4]) {
        st4(p, make_float4(o[0], o[1], o[2], o[3]));
    }
};
template <> struct Pack<__nv_bfloat16, 2> {
    static __device__ __forceinline__ void ld(const __nv_bfloat16* p, float (&o)[2]) {
        const uint32_t r = *reinterpret_cast<const uint32_t*>(p);
        o[0] = __uint_as_float(r << 16); o[1] = __uint_as_float(r & 0xffff0000u);
    }
    static __device__ __forceinline__ void st(__nv_bfloat16* p, const float (&o)[2]) {
        *reinterpret_cast<__nv_bfloat162*>(p) = __floats2bfloat162_rn(o[0], o[1]);
    }
};

// bytes of the per-warp shared-memory region
__host__ __device__ inline size_t warp_region_bytes(int G, int D, int eb, int level) {
    return (size_t)G * D * 4 + (size_t)G * D * eb + (size_t)2 * level * D * eb;
}

template <typename T, int D, int ML>
__global__ void __launch_bounds__(kThreads)
tree_attn_kernel(const T* __restrict__ q, const T* __restrict__ ks, const T* __restrict__ vs,
                 const int32_t* __restrict__ anc, const float* __restrict__ pm,
                 const float* __restrict__ pl, const float* __restrict__ po, T* __restrict__ out,
                 int B, int n_q, int Hq, int Hkv, int G, int HPW, int Wmax, int d, int level, int n_splits,
                 float scale) {
    // HPW = query heads served by one warp: the whole GQA group (HPW = G) when the chain's K/V rows
    // dominate, a single head (HPW = 1) when many prefix splits are merged for few queries.
    constexpr int EPL = D / 32;
    constexpr int ROW_CHUNKS = D * (int)sizeof(T) / 16;  // 16-byte chunks per K/V/q row
    using PT = Pack<T, EPL>;
    using PF = Pack<float, EPL>;
    extern __shared__ __align__(16) unsigned char smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wpq = Hq / HPW;  // warps per query
    const long long n_warps = (long long)B * n_q * wpq;
    const long long w = (long long)blockIdx.x * kWarpsPerCta + warp;
    if (w >= n_warps) return;  // whole warps leave together; there is no block-level barrier below

    const int h0 = (int)(w % wpq) * HPW;
    const int kv = h0 / G;
    const long long ui = w / wpq;  // u * n_q + i
    const int i = (int)(ui % n_q);
    const int u = (int)(ui / n_q);
    const long long row0 = ui * Hq + h0;  // first of the HPW consecutive (query, head) rows
    const size_t split_stride = (size_t)B * n_q * Hq;
    const int col = lane * EPL;

    unsigned char* region = smem + (size_t)warp * warp_region_bytes(HPW, D, (int)sizeof(T), level);
    float* sO = reinterpret_cast<float*>(region);
    T* sQ = reinterpret_cast<T*>(sO + HPW * D);
    T* sK = sQ + HPW * D;
    T* sV = sK + level * D;

    // ---- everything independent goes in flight first ---------------------------------
    const int a_l = lane < level ? __ldg(anc + ((size_t)u * Wmax + i) * d + lane) : 0;
    float m0 = -INFINITY, l0 = 0.f;
    if (lane < HPW) { m0 = __ldg(pm + row0 + lane); l0 = __ldg(pl + row0 + lane); }
    {
        const unsigned char* gq = reinterpret_cast<const unsigned char*>(q + row0 * D);
        const unsigned char* go = reinterpret_cast<const unsigned char*>(po + row0 * D);
        for (int c = lane; c < HPW * ROW_CHUNKS; c += 32) cp_async16(reinterpret_cast<unsigned char*>(sQ) + c * 16, gq + c * 16);
        for (int c = lane; c < HPW * (D / 4); c += 32) cp_async16(reinterpret_cast<unsigned char*>(sO) + c * 16, go + c * 16);
    }
    // ---- the one dependent fetch: ancestor slot -> K/V row ---------------------------------
    const size_t level_stride = (size_t)B * Wmax * Hkv * D;
    for (int t = 0; t < level; ++t) {
        int at = __shfl_sync(0xffffffffu, a_l, t);
        at = min(max(at, 0), Wmax - 1);  // memory safety on garbage input
        const size_t row = (size_t)t * level_stride + (((size_t)u * Wmax + at) * Hkv + kv) * D;
        const unsigned char* gk = reinterpret_cast<const unsigned char*>(ks + row);
        const unsigned char* gv = reinterpret_cast<const unsigned char*>(vs + row);
        for (int c = lane; c < 2 * ROW_CHUNKS; c += 32) {
            const bool is_v = c >= ROW_CHUNKS;
            const int off = (is_v ? c - ROW_CHUNKS : c) * 16;
            cp_async16(reinterpret_cast<unsigned char*>(is_v ? sV : sK) + (size_t)t * D * sizeof(T) + off,
                       (is_v ? gv : gk) + off);
        }
    }
    cp_async_wait_all();
    __syncwarp();

    for (int g = 0; g < HPW; ++g) {
        float qv[EPL];
        PT::ld(sQ + g * D + col, qv);
        // chain scores
        float y[ML];
#pragma unroll
        for (int t = 0; t < ML; ++t) {
            y[t] = -INFINITY;
            if (t < level) {
                float kr[EPL], dot = 0.f;
                PT::ld(sK + t * D + col, kr);
#pragma unroll
                for (int e = 0; e < EPL; ++e) dot = fmaf(qv[e], kr[e], dot);
                y[t] = warp_sum(dot) * scale;
            }
        }
        // global maximum over prefix splits and chain
        const float mg0 = __shfl_sync(0xffffffffu, m0, g), lg0 = __shfl_sync(0xffffffffu, l0, g);
        float m_tot = mg0;
        if (n_splits > 1) {
            for (int s = 1 + lane; s < n_splits; s += 32) m_tot = fmaxf(m_tot, __ldg(pm + s * split_stride + row0 + g));
            m_tot = warp_max(m_tot);
        }
#pragma unroll
        for (int t = 0; t < ML; ++t) m_tot = fmaxf(m_tot, y[t]);

        // merge: prefix splits by log-sum-exp, then the chain.  Empty split: (m, l, o) = (-inf, 0, 0),
        // reading R18 -- the guards only avoid (-inf) - (-inf).
        float acc[EPL];
        PF::ld(sO + g * D + col, acc);
        const float w0 = mg0 > -INFINITY ? __expf(mg0 - m_tot) : 0.f;
        float denom = w0 * lg0;
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] *= w0;
        for (int s0 = 1; s0 < n_splits; s0 += 8) {  // 8 splits in flight: their loads do not depend on each other
            float ms[8], ls[8], os[8][EPL];
#pragma unroll
            for (int x = 0; x < 8; ++x) {
                const size_t r = (size_t)min(s0 + x, n_splits - 1) * split_stride + row0 + g;
                ms[x] = __ldg(pm + r); ls[x] = __ldg(pl + r);
                PF::ld(po + r * D + col, os[x]);
            }
#pragma unroll
            for (int x = 0; x < 8; ++x) {
                const float ws = (s0 + x < n_splits && ms[x] > -INFINITY) ? __expf(ms[x] - m_tot) : 0.f;
                denom = fmaf(ws, ls[x], denom);
#pragma unroll
                for (int e = 0; e < EPL; ++e) acc[e] = fmaf(ws, os[x][e], acc[e]);
            }
        }
#pragma unroll
        for (int t = 0; t < ML; ++t) {
            if (t < level) {
                const float e_ = __expf(y[t] - m_tot);  // m_tot >= y[t] > -inf here
                float vr[EPL];
                PT::ld(sV + t * D + col, vr);
                denom += e_;
#pragma unroll
                for (int e = 0; e < EPL; ++e) acc[e] = fmaf(e_, vr[e], acc[e]);
            }
        }
        const float inv = denom > 0.f ? 1.0f / denom : 0.f;
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] *= inv;
        PT::st(out + (row0 + g) * D + col, acc);
    }
}

template <typename T, int D, int ML>
int launch_m(const Dims& p, const void* q, int n_q, int level, const void* ks, const void* vs,
             const int32_t* anc_l, const float* pm, const float* pl, const float* po, int n_splits,
             void* out, cudaStream_t st) {
    // few queries with many prefix splits (decode step 0): one head per warp, for parallelism over the
    // split partials; otherwise the whole GQA group per warp (the chain rows are fetched once per group)
    const int hpw = (n_splits > 1 && (long long)p.B * n_q * p.Hkv < 2048) ? 1 : p.G;
    const long long warps = (long long)p.B * n_q * (p.Hq / hpw);
    const unsigned nb = (unsigned)((warps + kWarpsPerCta - 1) / kWarpsPerCta);
    const size_t smem = kWarpsPerCta * warp_region_bytes(hpw, D, (int)sizeof(T), level);
    if (smem > 48 * 1024) {
        static PerDevice<size_t> opted_dev;  // idempotent; a benign race at worst repeats the call
        size_t& opted = opted_dev.here();
        if (smem > 227 * 1024) return STARK_ERR_UNSUPPORTED;
        if (smem > opted) {
            STARK_CUDA_TRY(cudaFuncSetAttribute(tree_attn_kernel<T, D, ML>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                (int)smem));
            opted = smem;
        }
    }
    tree_attn_kernel<T, D, ML><<<nb, kThreads, smem, st>>>((const T*)q, (const T*)ks, (const T*)vs, anc_l, pm, pl,
                                                           po, (T*)out, p.B, n_q, p.Hq, p.Hkv, p.G, hpw, p.Wmax,
                                                           p.d, level, n_splits, p.scale);
    STARK_LAUNCH_CHECK();
    return STARK_OK;
}

template <typename T>
int launch_t(const Dims& p, const void* q, int n_q, int level, const void* ks, const void* vs,
             const int32_t* anc, const float* pm, const float* pl, const float* po, int n_splits,
             void* out, cudaStream_t st) {
    const int32_t* anc_l = anc ? anc + (size_t)(level & 1) * p.B * p.Wmax * p.d : nullptr;
    if (p.G > 32) return STARK_ERR_UNSUPPORTED;  // per-head (m, l) of split 0 live one per lane
    // ML = compile-time bound of the chain length (score registers)
    if (p.D == 128) {
        if (level <= 4) return launch_m<T, 128, 4>(p, q, n_q, level, ks, vs, anc_l, pm, pl, po, n_splits, out, st);
        return launch_m<T, 128, kMaxLevels>(p, q, n_q, level, ks, vs, anc_l, pm, pl, po, n_splits, out, st);
    }
    if (level <= 4) return launch_m<T, 64, 4>(p, q, n_q, level, ks, vs, anc_l, pm, pl, po, n_splits, out, st);
    return launch_m<T, 64, kMaxLevels>(p, q, n_q, level, ks, vs, anc_l, pm, pl, po, n_splits, out, st);
}

}  // namespace

int launch_tree_attn(const Dims& p, int dtype, const void* q, int n_q, int level, const void* ks,
                     const void* vs, const int32_t* anc, const float* pm, const float* pl,
                     const float* po, int n_splits, void* out, cudaStream_t st) {
    if (dtype == STARK_F32)
        return launch_t<float>(p, q, n_q, level, ks, vs, anc, pm, pl, po, n_splits, out, st);
    return launch_t<__nv_bfloat16>(p, q, n_q, level, ks, vs, anc, pm, pl, po, n_splits, out, st);
}

}  // namespace stark
