// A1 (streaming form): stark_prefix_attn for SMALL M -- decode step 0 (one query
// per user, M = G rows) and the fp32 configuration.
//
// attention over the shared user-history prefix is computed
// once for all beams of a user.  When only a handful of query rows exist per
// (user, KV head) the contraction has ~4 flop per KV byte: it is a pure HBM
// stream of the prefix K/V and tensor cores are irrelevant (SURVEY.md section
// 8(d): "step 0 and cfg 1 HBM/latency-bound").  This kernel therefore streams
// K/V rows with 16-byte loads straight into registers (no shared-memory
// staging: there is no reuse to capture), keeps MQ query rows and their
// running (m, l, o) in registers, flash-decoding style, and splits the prefix
// over CTAs (n_splits) so that the grid fills all 148 SMs.
//
// Thread mapping: a row of D elements is covered by LPR = D/EPL lanes (EPL = 8
// bf16 or 4 fp32 elements = one 16-byte load per lane); a warp therefore holds
// 32/LPR rows at once and every lane keeps kUnroll rows in flight.
// Dot products reduce with xor-shuffles inside the LPR-lane subgroup.
// Output: split-softmax partials (m, l, o), see stark.h.
#include "common.cuh"

namespace stark {

namespace {

constexpr int kWarps = 4;
constexpr int kThreads = kWarps * 32;
constexpr int kUnroll = 4;

template <typename T> struct Vec;
template <> struct Vec<float> {
    static constexpr int EPL = 4;
    static __device__ __forceinline__ void load(const float* p, float (&o)[4]) {
        float4 r = __ldg(reinterpret_cast<const float4*>(p));
        o[0] = r.x; o[1] = r.y; o[2] = r.z; o[3] = r.w;
    }
};
template <> struct Vec<__nv_bfloat16> {
    static constexpr int EPL = 8;
    static __device__ __forceinline__ void load(const __nv_bfloat16* p, float (&o)[8]) {
        uint4 r = __ldg(reinterpret_cast<const uint4*>(p));
        const uint32_t w[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            o[2 * j] = __uint_as_float(w[j] << 16);
            o[2 * j + 1] = __uint_as_float(w[j] & 0xffff0000u);
        }
    }
};

template <typename T, int D, int MQ>
__global__ void __launch_bounds__(kThreads)
prefix_simt_kernel(const T* __restrict__ q, const T* __restrict__ kp, const T* __restrict__ vp,
                   const int32_t* __restrict__ cu, float* __restrict__ pm, float* __restrict__ pl,
                   float* __restrict__ po, int B, int n_q, int Hq, int Hkv, int G, int n_splits,
                   float scale_log2) {
    constexpr int EPL = Vec<T>::EPL;
    constexpr int LPR = D / EPL;    // lanes per row
    constexpr int SG = 32 / LPR;    // rows per warp-load
    const int mt = blockIdx.x;
    const int kv = blockIdx.y % Hkv;
    const int split = blockIdx.y / Hkv;
    const int u = blockIdx.z;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int sg = lane / LPR, sub = lane % LPR;
    const int M = n_q * G;

    const int row_begin = cu[u];
    const int L = cu[u + 1] - row_begin;
    int chunk = (L + n_splits - 1) / n_splits;
    chunk = ((chunk + 127) / 128) * 128;
    const int r0 = split * chunk;
    const int r1 = min(L, r0 + chunk);

    // query rows of this m-tile -> registers (pre-scaled into the log2 domain)
    float qr[MQ][EPL];
#pragma unroll
    for (int j = 0; j < MQ; ++j) {
        const int mrow = min(mt * MQ + j, M - 1);
        const int i = mrow / G, g = mrow % G;
        Vec<T>::load(q + (((size_t)u * n_q + i) * Hq + kv * G + g) * D + sub * EPL, qr[j]);
#pragma unroll
        for (int e = 0; e < EPL; ++e) qr[j][e] *= scale_log2;
    }

    float m[MQ], l[MQ], o[MQ][EPL];
#pragma unroll
    for (int j = 0; j < MQ; ++j) {
        m[j] = -INFINITY; l[j] = 0.f;
#pragma unroll
        for (int e = 0; e < EPL; ++e) o[j][e] = 0.f;
    }

    const size_t row_stride = (size_t)Hkv * D;
    const T* kbase = kp + ((size_t)row_begin * Hkv + kv) * D + sub * EPL;
    const T* vbase = vp + ((size_t)row_begin * Hkv + kv) * D + sub * EPL;
    constexpr int ROWS_PER_ITER = kWarps * SG * kUnroll;
    for (int rb = r0; rb < r1; rb += ROWS_PER_ITER) {
        float kr[kUnroll][EPL], vr[kUnroll][EPL];
        bool ok[kUnroll];
#pragma unroll
        for (int x = 0; x < kUnroll; ++x) {
            const int r = rb + (x * kWarps + warp) * SG + sg;
            ok[x] = r < r1;
            const int rr = ok[x] ? r : r0;  // r0 < r1 inside the loop: always a legal row
            Vec<T>::load(kbase + (size_t)rr * row_stride, kr[x]);
            Vec<T>::load(vbase + (size_t)rr * row_stride, vr[x]);
        }
#pragma unroll
        for (int j = 0; j < MQ; ++j) {
            float s[kUnroll];
            float mn = m[j];
#pragma unroll
            for (int x = 0; x < kUnroll; ++x) {
                float dot = 0.f;
#pragma unroll
                for (int e = 0; e < EPL; ++e) dot = fmaf(qr[j][e], kr[x][e], dot);
#pragma unroll
                for (int off = LPR / 2; off > 0; off >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, off);
                s[x] = ok[x] ? dot : -INFINITY;
                mn = fmaxf(mn, s[x]);
            }
            if (mn > -INFINITY) {
                const float corr = exp2f(m[j] - mn);
                float padd = 0.f;
#pragma unroll
                for (int e = 0; e < EPL; ++e) o[j][e] *= corr;
#pragma unroll
                for (int x = 0; x < kUnroll; ++x) {
                    const float p = exp2f(s[x] - mn);
                    padd += p;
#pragma unroll
                    for (int e = 0; e < EPL; ++e) o[j][e] = fmaf(p, vr[x][e], o[j][e]);
                }
                l[j] = l[j] * corr + padd;
                m[j] = mn;
            }
        }
    }

    // ---- merge the SG subgroups of a warp (shuffles), then the warps (smem) ----
    __shared__ float sm_m[kWarps][MQ], sm_l[kWarps][MQ];
    __shared__ float sm_o[kWarps][MQ][D];
#pragma unroll
    for (int j = 0; j < MQ; ++j) {
#pragma unroll
        for (int off = LPR; off < 32; off <<= 1) {
            const float m2 = __shfl_xor_sync(0xffffffffu, m[j], off);
            const float l2 = __shfl_xor_sync(0xffffffffu, l[j], off);
            const float mn = fmaxf(m[j], m2);
            const float c1 = mn > -INFINITY ? exp2f(m[j] - mn) : 0.f;
            const float c2 = mn > -INFINITY ? exp2f(m2 - mn) : 0.f;
            l[j] = l[j] * c1 + l2 * c2;
#pragma unroll
            for (int e = 0; e < EPL; ++e) {
                const float o2 = __shfl_xor_sync(0xffffffffu, o[j][e], off);
                o[j][e] = o[j][e] * c1 + o2 * c2;
            }
            m[j] = mn;
        }
        if (sg == 0) {
            if (sub == 0) { sm_m[warp][j] = m[j]; sm_l[warp][j] = l[j]; }
#pragma unroll
            for (int e = 0; e < EPL; ++e) sm_o[warp][j][sub * EPL + e] = o[j][e];
        }
    }
    __syncthreads();
    const size_t split_stride = (size_t)B * n_q * Hq;
    for (int idx = threadIdx.x; idx < MQ * D; idx += kThreads) {
        const int j = idx / D, col = idx % D;
        const int mrow = mt * MQ + j;
        if (mrow >= M) continue;
        const int i = mrow / G, g = mrow % G;
        float mn = -INFINITY;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) mn = fmaxf(mn, sm_m[w][j]);
        float lt = 0.f, ot = 0.f;
        if (mn > -INFINITY) {
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                const float c = exp2f(sm_m[w][j] - mn);
                lt += c * sm_l[w][j];
                ot += c * sm_o[w][j][col];
            }
        }
        const size_t row = split * split_stride + ((size_t)u * n_q + i) * Hq + kv * G + g;
        po[row * D + col] = ot;
        if (col == 0) { pm[row] = mn * kLn2; pl[row] = lt; }
    }
}

template <typename T, int D>
int launch_t(const Dims& p, const void* q, int n_q, const void* k, const void* v, const int32_t* cu,
             int n_splits, float* pm, float* pl, float* po, cudaStream_t st) {
    constexpr int MQ = 4;
    const int M = n_q * p.G;
    dim3 grid((M + MQ - 1) / MQ, p.Hkv * n_splits, p.B);
    prefix_simt_kernel<T, D, MQ><<<grid, kThreads, 0, st>>>((const T*)q, (const T*)k, (const T*)v, cu, pm, pl,
                                                            po, p.B, n_q, p.Hq, p.Hkv, p.G, n_splits,
                                                            p.scale * kLog2e);
    STARK_LAUNCH_CHECK();
    return STARK_OK;
}

}  // namespace

int launch_prefix_simt(const Dims& p, int dtype, const void* q, int n_q, const void* k, const void* v,
                       const int32_t* cu, int n_splits, float* pm, float* pl, float* po,
                       cudaStream_t st) {
    if (dtype == STARK_F32) {
        if (p.D == 128) return launch_t<float, 128>(p, q, n_q, k, v, cu, n_splits, pm, pl, po, st);
        return launch_t<float, 64>(p, q, n_q, k, v, cu, n_splits, pm, pl, po, st);
    }
    if (p.D == 128) return launch_t<__nv_bfloat16, 128>(p, q, n_q, k, v, cu, n_splits, pm, pl, po, st);
    return launch_t<__nv_bfloat16, 64>(p, q, n_q, k, v, cu, n_splits, pm, pl, po, st);
}

}  // namespace stark
