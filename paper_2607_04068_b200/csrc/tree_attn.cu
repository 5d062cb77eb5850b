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
// + out.  Mapping: D/4 lanes per (query, head), each
// lane owns 4 consecutive head-dim elements (16-byte fp32 / 8-byte bf16
// accesses, fully coalesced rows); dot products reduce with warp shuffles.
#include "common.cuh"

namespace stark {

namespace {

constexpr int kThreads = 256;
constexpr int kMaxLevels = 8;

template <typename T, int D>
__global__ void __launch_bounds__(kThreads)
tree_attn_kernel(const T* __restrict__ q, const T* __restrict__ ks, const T* __restrict__ vs,
                 const int32_t* __restrict__ anc, const float* __restrict__ pm,
                 const float* __restrict__ pl, const float* __restrict__ po, T* __restrict__ out,
                 int B, int n_q, int Hq, int Hkv, int G, int Wmax, int d, int level, int n_splits,
                 float scale) {
    constexpr int LPH = D / 4;  // lanes per (query, head)
    const long long n_groups = (long long)B * n_q * Hq;
    const long long group = ((long long)blockIdx.x * kThreads + threadIdx.x) / LPH;
    const int sub = threadIdx.x % LPH;
    // whole LPH-lane groups are in or out together, shuffles below stay inside a group
    const bool live = group < n_groups;
    const long long g = live ? group : n_groups - 1;

    const int h = (int)(g % Hq);
    const long long ui = g / Hq;  // u * n_q + i
    const int i = (int)(ui % n_q);
    const int u = (int)(ui / n_q);
    const int kv = h / G;

    const float4 q4 = ld4(q + g * D + sub * 4);

    // ---- suffix chain scores --------------------------------------------------
    float y[kMaxLevels];
    float4 v4[kMaxLevels];
    const size_t level_stride = (size_t)B * Wmax * Hkv * D;
#pragma unroll
    for (int t = 0; t < kMaxLevels; ++t) {
        y[t] = -INFINITY;
        v4[t] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (t < level) {
            int a = __ldg(anc + ((size_t)u * Wmax + i) * d + t);
            a = min(max(a, 0), Wmax - 1);
            const size_t row = (size_t)t * level_stride + (((size_t)u * Wmax + a) * Hkv + kv) * D + sub * 4;
            const float4 k4 = ld4(ks + row);
            v4[t] = ld4(vs + row);
            float dot = q4.x * k4.x + q4.y * k4.y + q4.z * k4.z + q4.w * k4.w;
#pragma unroll
            for (int o = LPH / 2; o > 0; o >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, o);
            y[t] = dot * scale;
        }
    }

    // ---- global maximum over prefix splits and chain --------------------------
    float m_tot = -INFINITY;
    const size_t split_stride = (size_t)B * n_q * Hq;
    for (int s = 0; s < n_splits; ++s) m_tot = fmaxf(m_tot, __ldg(pm + s * split_stride + g));
#pragma unroll
    for (int t = 0; t < kMaxLevels; ++t) m_tot = fmaxf(m_tot, y[t]);

    float denom = 0.f;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    if (m_tot > -INFINITY) {
        for (int s = 0; s < n_splits; ++s) {
            const float ms = __ldg(pm + s * split_stride + g);
            if (ms == -INFINITY) continue;  // empty split: (m,l,o) = (-inf,0,0), reading R18
            const float w = __expf(ms - m_tot);
            denom += w * __ldg(pl + s * split_stride + g);
            const float4 o4 = *reinterpret_cast<const float4*>(po + (s * split_stride + g) * D + sub * 4);
            acc.x += w * o4.x; acc.y += w * o4.y; acc.z += w * o4.z; acc.w += w * o4.w;
        }
#pragma unroll
        for (int t = 0; t < kMaxLevels; ++t) {
            if (t < level) {
                const float e = __expf(y[t] - m_tot);
                denom += e;
                acc.x += e * v4[t].x; acc.y += e * v4[t].y; acc.z += e * v4[t].z; acc.w += e * v4[t].w;
            }
        }
    }
    const float inv = denom > 0.f ? 1.0f / denom : 0.f;
    if (live) st4(out + g * D + sub * 4, make_float4(acc.x * inv, acc.y * inv, acc.z * inv, acc.w * inv));
}

template <typename T>
int launch_t(const Dims& p, const void* q, int n_q, int level, const void* ks, const void* vs,
             const int32_t* anc, const float* pm, const float* pl, const float* po, int n_splits,
             void* out, cudaStream_t st) {
    const long long groups = (long long)p.B * n_q * p.Hq;
    const int lph = p.D / 4;
    const long long threads = groups * lph;
    const unsigned nb = (unsigned)((threads + kThreads - 1) / kThreads);
    const int32_t* anc_l = anc ? anc + (size_t)(level & 1) * p.B * p.Wmax * p.d : nullptr;
    if (p.D == 128)
        tree_attn_kernel<T, 128><<<nb, kThreads, 0, st>>>((const T*)q, (const T*)ks, (const T*)vs, anc_l, pm,
                                                          pl, po, (T*)out, p.B, n_q, p.Hq, p.Hkv, p.G,
                                                          p.Wmax, p.d, level, n_splits, p.scale);
    else
        tree_attn_kernel<T, 64><<<nb, kThreads, 0, st>>>((const T*)q, (const T*)ks, (const T*)vs, anc_l, pm,
                                                         pl, po, (T*)out, p.B, n_q, p.Hq, p.Hkv, p.G,
                                                         p.Wmax, p.d, level, n_splits, p.scale);
    STARK_LAUNCH_CHECK();
    return STARK_OK;
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
