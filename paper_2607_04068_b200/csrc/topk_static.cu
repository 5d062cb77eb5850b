// stark_beam_topk_static: stark_beam_topk (A3; Eq. 1, 257, 263, 306) for callers that cannot
// allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Same kernels,
// same result bit for bit; the workspace of the whole-GPU kernel (topk_grid.cu) is a file-scope device array of
// this library instead of a caller buffer.
//
//  * The array costs STARK_TOPK_STATIC_SCRATCH_BYTES (9 MiB) of device memory on every GPU that loads the library,
//    until the process exits.  Problems whose workspace (stark_workspace_bytes(STARK_CALL_BEAM_TOPK)) is larger are
//    rejected with STARK_ERR_WORKSPACE (on B200: more than 29 users at >= 131 072 candidates per user).
//  * In host code `g_topk_scratch` is a host-side stand-in, not a device address: the device address is taken once
//    per device, with that device current, by cudaGetSymbolAddress (scratch_here()) and that pointer is what the
//    kernels get.
//  * All calls on one GPU share the array, and it keeps what the last call left.  The kernels need the counters in it
//    zero at launch and leave them zero, but a call that was aborted (a fault, a device reset by another library
//    call) would break that for everybody after it, so every call clears the part it uses first (one
//    cudaMemsetAsync on the caller's stream, ordered before the kernel).
//  * For the same reason two calls that OVERLAP on the GPU (different streams without an ordering between them, or
//    two host threads) RACE on the array: results are undefined.  Such callers use stark_beam_topk with a workspace
//    each.
//  * No cudaMalloc / cudaFree / allocating library routine on this path: argument checks, cudaGetSymbolAddress (first
//    call per device), cudaMemsetAsync, kernel launches.
#include "common.cuh"

namespace stark {
namespace {

static __device__ __align__(256) unsigned char g_topk_scratch[STARK_TOPK_STATIC_SCRATCH_BYTES];

// Device address of g_topk_scratch on the current device (nullptr + STARK_ERR_CUDA recorded on failure).
void* scratch_here() {
    static PerDevice<void*> addr;
    void*& p = addr.here();
    if (p == nullptr) {
        void* q = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&q, g_topk_scratch);
        if (e != cudaSuccess) {
            last_cuda_error_ref() = (int)e;
            (void)cudaGetLastError();
            return nullptr;
        }
        p = q;
    }
    return p;
}

// per device: 0 = unknown, 1 = sm_100, -1 = something else (the same rule as the other entry points)
int static_device_status() {
    static PerDevice<int> state;
    int& s = state.here();
    if (s == 0) {
        int dev = 0, major = 0;
        if (cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
            last_cuda_error_ref() = (int)cudaGetLastError();
            return STARK_ERR_CUDA;
        }
        s = major == 10 ? 1 : -1;
    }
    return s == 1 ? STARK_OK : STARK_ERR_UNSUPPORTED;
}

}  // namespace
}  // namespace stark

using namespace stark;

extern "C" int stark_beam_topk_static(const float* logp, const float* score_or_null, int B, int W_in, int C,
                                      int W_out, float* out_score, int32_t* out_parent, int32_t* out_code,
                                      void* stream) {
    if (!logp || !out_score || !out_parent || !out_code) return STARK_ERR_INVALID_ARG;
    if (B < 1 || W_in < 1 || C < 1 || W_out < 1) return STARK_ERR_INVALID_ARG;
    if ((long long)W_in * C >= (1ll << 31)) return STARK_ERR_INVALID_ARG;
    if ((long long)W_out > (long long)W_in * C || W_out > 4096) return STARK_ERR_INVALID_ARG;
    const size_t need = topk_workspace_bytes(B, W_in, C);
    if (need > (size_t)STARK_TOPK_STATIC_SCRATCH_BYTES) return STARK_ERR_WORKSPACE;   // beyond the static maximum
    const int rc = static_device_status();
    if (rc != STARK_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    void* ws = nullptr;
    if (need > 0) {
        ws = scratch_here();
        if (ws == nullptr) return STARK_ERR_CUDA;
        STARK_CUDA_TRY(cudaMemsetAsync(ws, 0, need, st));
    }
    return launch_topk(logp, score_or_null, B, W_in, C, W_out, out_score, out_parent, out_code, ws, need, st);
}
