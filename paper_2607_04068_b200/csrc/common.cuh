// Shared device/host helpers for the STARK kernels (sm_100a only).
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "stark.h"

namespace stark {

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

// ---- launch parameters resolved on the host --------------------------------
struct Dims {
    int B, Hq, Hkv, G, D, d, Wmax;
    float scale;  // softmax scale (already defaulted)
};

inline Dims make_dims(const stark_shape_t* s) {
    Dims p;
    p.B = s->B; p.Hq = s->Hq; p.Hkv = s->Hkv; p.G = s->Hq / s->Hkv; p.D = s->D;
    p.d = s->d; p.Wmax = s->Wmax;
    p.scale = s->softmax_scale != 0.f ? s->softmax_scale : 1.0f / sqrtf((float)s->D);
    return p;
}

// Last CUDA error seen by the library (host side, set by CUDA_TRY).
int& last_cuda_error_ref();

#define STARK_CUDA_TRY(expr)                                          \
    do {                                                              \
        cudaError_t _e = (expr);                                      \
        if (_e != cudaSuccess) {                                      \
            ::stark::last_cuda_error_ref() = (int)_e;                 \
            (void)cudaGetLastError();                                 \
            return STARK_ERR_CUDA;                                    \
        }                                                             \
    } while (0)

#define STARK_LAUNCH_CHECK() STARK_CUDA_TRY(cudaGetLastError())

// cudaFuncSetAttribute, occupancy and SM count are PER DEVICE: every cached value is keyed by the current
// device (cudaGetDevice), so that a process driving several GPUs gets each of them set up.
constexpr int kMaxDevices = 64;
int current_device();  // cudaGetDevice(), clamped to [0, kMaxDevices); 0 if the call fails
template <typename T>
struct PerDevice {
    T v[kMaxDevices] = {};
    T& here() { return v[current_device()]; }
};
int num_sms();  // cudaDevAttrMultiProcessorCount of the current device, cached per device (148 on B200)

// ---- element access ---------------------------------------------------------
template <typename T> struct Elem;
template <> struct Elem<float> {
    static __device__ __forceinline__ float ld(const float* p) { return *p; }
    static __device__ __forceinline__ void st(float* p, float v) { *p = v; }
};
template <> struct Elem<__nv_bfloat16> {
    static __device__ __forceinline__ float ld(const __nv_bfloat16* p) { return __bfloat162float(*p); }
    static __device__ __forceinline__ void st(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }
};

// 4 consecutive elements -> float4 (16-byte load for fp32, 8-byte for bf16).
__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ float4 ld4(const __nv_bfloat16* p) {
    uint2 r = *reinterpret_cast<const uint2*>(p);
    float4 o;
    o.x = __uint_as_float(r.x << 16);
    o.y = __uint_as_float(r.x & 0xffff0000u);
    o.z = __uint_as_float(r.y << 16);
    o.w = __uint_as_float(r.y & 0xffff0000u);
    return o;
}
__device__ __forceinline__ void st4(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ void st4(__nv_bfloat16* p, float4 v) {
    __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y);
    __nv_bfloat162 b = __floats2bfloat162_rn(v.z, v.w);
    uint2 r;
    r.x = *reinterpret_cast<uint32_t*>(&a);
    r.y = *reinterpret_cast<uint32_t*>(&b);
    *reinterpret_cast<uint2*>(p) = r;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// ---- kernel launchers (one per .cu) -----------------------------------------
int launch_prefix_simt(const Dims& p, int dtype, const void* q, int n_q, const void* k, const void* v,
                       const int32_t* cu, int n_splits, float* pm, float* pl, float* po,
                       cudaStream_t st);
// returns STARK_ERR_UNSUPPORTED when the shape has no tensor-core path
int launch_prefix_tc(const Dims& p, const void* q, int n_q, const void* k, const void* v,
                     const int32_t* cu, int total_tokens, int max_len, int n_splits, float* pm, float* pl,
                     float* po, cudaStream_t st);
bool prefix_tc_supported(const Dims& p, int dtype, int n_q);
bool prefix_tc_parity(const Dims& p, int n_q, int n_splits);
int launch_decode_fused(const Dims& p, const void* q, int n_q, int level, const void* k, const void* v,
                        const int32_t* cu, int total_tokens, int max_len, int n_splits, const void* ks, const void* vs,
                        const int32_t* anc_level, void* out, cudaStream_t st, const void* kn = nullptr,
                        const void* vn = nullptr, const int32_t* parent = nullptr, int32_t* anc_new = nullptr);
int launch_tree_attn(const Dims& p, int dtype, const void* q, int n_q, int level, const void* ks,
                     const void* vs, const int32_t* anc, const float* pm, const float* pl,
                     const float* po, int n_splits, void* out, cudaStream_t st);
int launch_append(const Dims& p, int dtype, int level, int n_new, const void* kn, const void* vn,
                  const int32_t* parent, void* ks, void* vs, int32_t* anc, cudaStream_t st);
int launch_topk(const float* logp, const float* score, int B, int W_in, int C, int W_out,
                float* out_score, int32_t* out_parent, int32_t* out_code, void* ws, size_t ws_bytes,
                cudaStream_t st, bool fold_lse = false);
// fold_lse: `logp` holds RAW logits and the kernel folds the row's log-sum-exp into the score itself (reading
// R22); only where topk_can_fold_lse() says so (one row per user, small enough for the one-CTA kernel).
bool topk_can_fold_lse(int W_in, int C);
size_t topk_workspace_bytes(int B, int W_in, int C);
// topk_grid.cu: large candidate sets on the whole GPU; STARK_ERR_UNSUPPORTED = not served, use launch_topk's kernels
size_t topk_grid_workspace_bytes(int B, int W_in, int C);
int launch_topk_grid(const float* logp, const float* score, int B, int W_in, int C, int W_out,
                     float* out_score, int32_t* out_parent, int32_t* out_code, void* ws, size_t ws_bytes,
                     cudaStream_t st);
// topk_grid.cu: wide selections (W_out <= 1024) over small candidate sets (N <= 8192): R independent CTAs per user
bool topk_wide_serves(long long N, int W_out);
int launch_topk_wide(const float* logp, const float* score, int B, int W_in, int C, int W_out,
                     float* out_score, int32_t* out_parent, int32_t* out_code, cudaStream_t st);
int launch_row_offset(const float* logits, const float* score, long long rows, int C, float* offset,
                      cudaStream_t st);

}  // namespace stark
