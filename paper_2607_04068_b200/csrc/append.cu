// A4: stark_kv_append_reorg -- append the K/V of one new tree level to the
// compact per-level suffix buffer and extend the ancestor index mapping.
//
// PAPER.md:284-286 (section 3.6): "both the tree mask and KV cache remapping can
// be prepared as lightweight index operations rather than repeated data
// copies ... candidate expansion primarily appends newly selected semantic
// tokens to the tree rather than duplicating the entire prefix cache".
//
// Pure data movement, HBM-bound: 2*(2*D*eb) bytes per (new node, KV head) plus
// 8*d bytes of index per node.  The prefix is never
// touched.  One launch: blockIdx.y = 0 copies K, 1 copies V, 2 builds `anc`.
#include "common.cuh"

namespace stark {

namespace {

constexpr int kThreads = 256;
constexpr int kUnroll = 4;  // 16-byte vectors in flight per thread

__global__ void __launch_bounds__(kThreads)
append_kernel(const uint4* __restrict__ kn, const uint4* __restrict__ vn, uint4* __restrict__ ks,
              uint4* __restrict__ vs, const int32_t* __restrict__ parent,
              const int32_t* __restrict__ anc_prev, int32_t* __restrict__ anc_new, int B, int n_new,
              int Wmax, int d, int level, long long vec_per_user_src, long long vec_per_user_dst) {
    if (blockIdx.y < 2) {
        const uint4* __restrict__ src = blockIdx.y == 0 ? kn : vn;
        uint4* __restrict__ dst = blockIdx.y == 0 ? ks : vs;
        const long long total = (long long)B * vec_per_user_src;
        const long long stride = (long long)gridDim.x * kThreads * kUnroll;
        for (long long base = (long long)blockIdx.x * kThreads * kUnroll + threadIdx.x; base < total;
             base += stride) {
            uint4 r[kUnroll];
#pragma unroll
            for (int j = 0; j < kUnroll; ++j) {
                long long i = base + (long long)j * kThreads;
                if (i < total) r[j] = __ldg(src + i);
            }
#pragma unroll
            for (int j = 0; j < kUnroll; ++j) {
                long long i = base + (long long)j * kThreads;
                if (i < total) {
                    long long u = i / vec_per_user_src;
                    long long off = i - u * vec_per_user_src;
                    dst[u * vec_per_user_dst + off] = r[j];
                }
            }
        }
    } else if (anc_new != nullptr) {
        // one thread per (user, new beam): gather the parent's chain, append self
        const int total = B * n_new;
        for (int i = blockIdx.x * kThreads + threadIdx.x; i < total; i += gridDim.x * kThreads) {
            int u = i / n_new, s = i - u * n_new;
            int32_t* row = anc_new + ((long long)u * Wmax + s) * d;
            if (level >= 2) {
                int p = parent[i];
                p = min(max(p, 0), Wmax - 1);  // memory safety on garbage input
                const int32_t* prow = anc_prev + ((long long)u * Wmax + p) * d;
                for (int t = 0; t < level - 1; ++t) row[t] = prow[t];
            }
            row[level - 1] = s;
        }
    }
}

}  // namespace

int launch_append(const Dims& p, int dtype, int level, int n_new, const void* kn, const void* vn,
                  const int32_t* parent, void* ks, void* vs, int32_t* anc, cudaStream_t st) {
    const int eb = dtype == STARK_F32 ? 4 : 2;
    const long long row_vec = (long long)p.Hkv * p.D * eb / 16;  // D in {64,128}: always whole vectors
    const long long vps = (long long)n_new * row_vec, vpd = (long long)p.Wmax * row_vec;
    const size_t level_elems = (size_t)p.B * p.Wmax * p.Hkv * p.D;
    char* ksl = (char*)ks + (size_t)(level - 1) * level_elems * eb;
    char* vsl = (char*)vs + (size_t)(level - 1) * level_elems * eb;
    const long long total = (long long)p.B * vps;
    long long nb = (total + (long long)kThreads * kUnroll - 1) / ((long long)kThreads * kUnroll);
    long long nb_anc = ((long long)p.B * n_new + kThreads - 1) / kThreads;
    if (nb < nb_anc) nb = nb_anc;
    if (nb > 148 * 8) nb = 148 * 8;
    if (nb < 1) nb = 1;
    const size_t half = (size_t)p.B * p.Wmax * p.d;
    int32_t* anc_new = anc ? anc + (size_t)(level & 1) * half : nullptr;
    const int32_t* anc_prev = anc ? anc + (size_t)((level - 1) & 1) * half : nullptr;
    dim3 grid((unsigned)nb, anc ? 3 : 2);
    append_kernel<<<grid, kThreads, 0, st>>>((const uint4*)kn, (const uint4*)vn, (uint4*)ksl,
                                             (uint4*)vsl, parent, anc_prev, anc_new, p.B, n_new,
                                             p.Wmax, p.d, level, vps, vpd);
    STARK_LAUNCH_CHECK();
    return STARK_OK;
}

}  // namespace stark
