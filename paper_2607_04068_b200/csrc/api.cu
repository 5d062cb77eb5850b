// C-ABI boundary of the STARK decode library (declared in include/stark.h).
// Argument validation first (no CUDA call), then dispatch to the launchers.
#include <math.h>

#include "common.cuh"

namespace stark {

int& last_cuda_error_ref() {
    static int e = 0;
    return e;
}

int current_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return 0; }
    return dev < 0 ? 0 : (dev >= kMaxDevices ? kMaxDevices - 1 : dev);
}

int num_sms() {
    static PerDevice<int> n;
    int& c = n.here();
    if (c == 0) {
        int dev = 0, v = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0)
            c = v;
        else {
            (void)cudaGetLastError();
            return 148;  // B200; used for planning only
        }
    }
    return c;
}

namespace {

// per device: 0 = unknown, 1 = sm_100, -1 = something else; -2 (not cached) = no device
int device_ok() {
    static PerDevice<int> state;
    int& s = state.here();
    if (s == 0) {
        int dev = 0, major = 0;
        if (cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
            last_cuda_error_ref() = (int)cudaGetLastError();
            return -2;
        }
        s = major == 10 ? 1 : -1;
    }
    return s;
}

int check_shape(const stark_shape_t* s) {
    if (!s) return STARK_ERR_INVALID_ARG;
    if (s->B < 1 || s->Hq < 1 || s->Hkv < 1 || s->D < 1 || s->d < 1 || s->Wmax < 1)
        return STARK_ERR_INVALID_ARG;
    if (s->Hq % s->Hkv != 0) return STARK_ERR_INVALID_ARG;
    if (s->d > 8) return STARK_ERR_INVALID_ARG;
    if (!(s->softmax_scale >= 0.f) || isinf(s->softmax_scale)) return STARK_ERR_INVALID_ARG;
    if (s->dtype != STARK_F32 && s->dtype != STARK_BF16) return STARK_ERR_UNSUPPORTED;
    if (s->D != 64 && s->D != 128) return STARK_ERR_UNSUPPORTED;
    return STARK_OK;
}

int check_device() {
    const int ok = device_ok();
    if (ok == 1) return STARK_OK;
    return ok == -2 ? STARK_ERR_CUDA : STARK_ERR_UNSUPPORTED;
}

// Per-beam offsets of stark_beam_topk_logits, at the front of its workspace (256-byte multiple).
size_t offset_bytes(int B, int W_in) { return (((size_t)B * W_in * sizeof(float)) + 255) / 256 * 256; }

int ceil_div(long long a, long long b) { return (int)((a + b - 1) / b); }

// Shape-only split choice.  Cost model: waves of CTAs x (KV tiles per CTA + a
// fixed per-CTA overhead of ~1 tile, ~2 for the tensor-core kernel whose
// prologue allocates TMEM and fills the TMA ring); ties go to the smaller
// split count (less partial traffic).
int plan_splits(const Dims& p, int dtype, int n_q, int max_len) {
    const int sms = num_sms() > 0 ? num_sms() : 148;
    const int tiles = ceil_div(max_len, 128);
    const bool tc = prefix_tc_supported(p, dtype, n_q);
    const long long M = (long long)n_q * p.G;
    int best = 1;
    double best_cost = 1e300;
    for (int n = 1; n <= 64 && n <= tiles; ++n) {
        double cost;
        if (tc) {
            // tensor-core kernel: an iteration handles one KV tile for a Q-tile pair, or (parity mode, when the
            // doubled CTA count still fits one wave) two KV tiles for one Q tile; ~2 iterations of prologue /
            // epilogue; every extra split adds a partial set (fp32, written and re-read through HBM)
            const bool parity = prefix_tc_parity(p, n_q, n);
            const long long ctas = (long long)p.B * p.Hkv * n * ceil_div(M, parity ? 128 : 256);
            const double iters = parity ? ceil_div(ceil_div(tiles, n), 2) + 0.5 : ceil_div(tiles, n);
            cost = (double)ceil_div(ctas, sms) * (iters + 2.0) + 0.75 * (n - 1);
        } else {
            const long long ctas = (long long)p.B * p.Hkv * n * ceil_div(M, 4);
            cost = (double)ceil_div(ctas, (long long)sms * 4) * (ceil_div(tiles, n) + 1.0);
        }
        if (cost < best_cost * 0.97) { best_cost = cost; best = n; }
    }
    return best;
}

// Cluster size (= prefix splits) of the fused decode-attention kernel: 1, 2, 4 or 8.  Same cost model; the
// exchange through distributed shared memory (~17 B/clk per SM) costs up to ~3.5 iterations when all 256
// rows are live; resident CTAs: one per SM, whole clusters only (B200 co-schedules 15 clusters of 8).
// A RAGGED batch (prefix lengths differ: total_tokens < B * max_len) is not a sequence of equal waves: its CTAs are
// handed out longest user first, so the launch takes about max(longest CTA, total work / resident CTAs).  (Measured at
// config 5 step 0, lengths 1.2-8.2 K: the wave model chose 4 splits, 160 us; 1 split: see profiles.)
int plan_cluster_splits(const Dims& p, int n_q, int max_len, int total_tokens) {
    const int sms = num_sms() > 0 ? num_sms() : 148;
    const int tiles = ceil_div(max_len, 128);
    const long long M = (long long)n_q * p.G;
    const bool ragged = p.B >= 2 && (long long)max_len * p.B != (long long)total_tokens;
    const double avg_tiles = (double)total_tokens / (128.0 * p.B);
    int best = 1;
    double best_cost = 1e300;
    for (int n = 1; n <= 8 && n <= tiles; n *= 2) {
        const bool parity = prefix_tc_parity(p, n_q, n);
        const long long ctas = (long long)p.B * p.Hkv * n * ceil_div(M, parity ? 128 : 256);
        const int resident = n == 8 ? (sms / 8 - 3) * 8 : sms / n * n;
        const double iters = parity ? ceil_div(ceil_div(tiles, n), 2) + 0.5 : ceil_div(tiles, n);
        const double live = (double)(M < 256 ? M : 256) / 256.0;
        double cost = (double)ceil_div(ctas, resident > 0 ? resident : n) * (iters + 2.0) + (n > 1 ? 3.5 * live : 0.0);
        if (ragged) {
            const double avg_iters = (parity ? 0.5 : 1.0) * avg_tiles / n;
            const double fluid = (double)ctas * (avg_iters + 2.0) / (double)(resident > 0 ? resident : n);
            cost = (fluid > iters + 2.0 ? fluid : iters + 2.0) + (n > 1 ? 3.5 * live : 0.0);
        }
        if (cost < best_cost * 0.97) { best_cost = cost; best = n; }
    }
    return best;
}

}  // namespace
}  // namespace stark

using namespace stark;

extern "C" {

int stark_version(void) { return STARK_VERSION; }

const char* stark_status_string(int status) {
    switch (status) {
        case STARK_OK: return "STARK_OK";
        case STARK_ERR_INVALID_ARG: return "STARK_ERR_INVALID_ARG: invalid argument";
        case STARK_ERR_UNSUPPORTED: return "STARK_ERR_UNSUPPORTED: dtype, head_dim or device not supported";
        case STARK_ERR_WORKSPACE: return "STARK_ERR_WORKSPACE: workspace missing or too small";
        case STARK_ERR_CUDA: return "STARK_ERR_CUDA: a CUDA call failed (see stark_last_cuda_error)";
        default: return "unknown stark status";
    }
}

int stark_last_cuda_error(void) { return last_cuda_error_ref(); }

size_t stark_suffix_bytes(const stark_shape_t* s) {
    if (check_shape(s) != STARK_OK) return 0;
    return (size_t)s->d * s->B * s->Wmax * s->Hkv * s->D * (s->dtype == STARK_F32 ? 4 : 2);
}

size_t stark_anc_bytes(const stark_shape_t* s) {
    if (check_shape(s) != STARK_OK) return 0;
    return (size_t)2 * s->B * s->Wmax * s->d * sizeof(int32_t);
}

size_t stark_workspace_bytes(const stark_shape_t* s, int call, int n_q, int total_tokens) {
    if (!s) return 0;
    if (call == STARK_CALL_BEAM_TOPK) {
        if (s->B < 1 || n_q < 1 || total_tokens < 1) return 0;
        return topk_workspace_bytes(s->B, n_q, total_tokens);
    }
    if (call == STARK_CALL_BEAM_TOPK_LOGITS) {
        if (s->B < 1 || n_q < 1 || total_tokens < 1) return 0;
        return offset_bytes(s->B, n_q) + topk_workspace_bytes(s->B, n_q, total_tokens);
    }
    return 0;
}

int stark_prefix_attn_plan(const stark_shape_t* shape, int n_q, int total_tokens, int max_prefix_len,
                           int* n_splits) {
    int rc = check_shape(shape);
    if (rc != STARK_OK) return rc;
    if (!n_splits || n_q < 1 || total_tokens < 0 || max_prefix_len < 1) return STARK_ERR_INVALID_ARG;
    *n_splits = plan_splits(make_dims(shape), shape->dtype, n_q, max_prefix_len);
    return STARK_OK;
}

int stark_prefix_attn(const stark_shape_t* shape, const void* q, int n_q, const void* k_prefix,
                      const void* v_prefix, const int32_t* cu_seqlens, int total_tokens,
                      int max_prefix_len, int n_splits, float* part_m, float* part_l, float* part_o,
                      void* ws, size_t ws_bytes, void* stream) {
    (void)ws; (void)ws_bytes;
    int rc = check_shape(shape);
    if (rc != STARK_OK) return rc;
    if (!q || !cu_seqlens || !part_m || !part_l || !part_o) return STARK_ERR_INVALID_ARG;
    if (n_q < 1 || total_tokens < 0 || max_prefix_len < 1 || n_splits < 0 || n_splits > 64)
        return STARK_ERR_INVALID_ARG;
    if (total_tokens > 0 && (!k_prefix || !v_prefix)) return STARK_ERR_INVALID_ARG;
    rc = check_device();
    if (rc != STARK_OK) return rc;
    const Dims p = make_dims(shape);
    if (n_splits == 0) n_splits = plan_splits(p, shape->dtype, n_q, max_prefix_len);
    cudaStream_t st = (cudaStream_t)stream;
    if (prefix_tc_supported(p, shape->dtype, n_q))
        return launch_prefix_tc(p, q, n_q, k_prefix, v_prefix, cu_seqlens, total_tokens, max_prefix_len, n_splits, part_m,
                                part_l, part_o, st);
    return launch_prefix_simt(p, shape->dtype, q, n_q, k_prefix, v_prefix, cu_seqlens, n_splits, part_m,
                              part_l, part_o, st);
}

int stark_tree_attn_step(const stark_shape_t* shape, const void* q, int n_q, int level,
                         const void* k_suffix, const void* v_suffix, const int32_t* anc,
                         const float* part_m, const float* part_l, const float* part_o, int n_splits,
                         void* out, void* stream) {
    int rc = check_shape(shape);
    if (rc != STARK_OK) return rc;
    if (!q || !part_m || !part_l || !part_o || !out) return STARK_ERR_INVALID_ARG;
    if (n_q < 1 || n_splits < 1 || level < 0 || level > shape->d) return STARK_ERR_INVALID_ARG;
    if (level >= 1 && (!k_suffix || !v_suffix || !anc || n_q > shape->Wmax)) return STARK_ERR_INVALID_ARG;
    rc = check_device();
    if (rc != STARK_OK) return rc;
    return launch_tree_attn(make_dims(shape), shape->dtype, q, n_q, level, k_suffix, v_suffix, anc, part_m,
                            part_l, part_o, n_splits, out, (cudaStream_t)stream);
}

int stark_decode_attn(const stark_shape_t* shape, const void* q, int n_q, int level, const void* k_prefix,
                      const void* v_prefix, const int32_t* cu_seqlens, int total_tokens, int max_prefix_len,
                      const void* k_suffix, const void* v_suffix, const int32_t* anc, void* out, void* stream) {
    int rc = check_shape(shape);
    if (rc != STARK_OK) return rc;
    if (!q || !cu_seqlens || !out) return STARK_ERR_INVALID_ARG;
    if (n_q < 1 || total_tokens < 0 || max_prefix_len < 1 || level < 0 || level > shape->d) return STARK_ERR_INVALID_ARG;
    if (total_tokens > 0 && (!k_prefix || !v_prefix)) return STARK_ERR_INVALID_ARG;
    if (level >= 1 && (!k_suffix || !v_suffix || !anc || n_q > shape->Wmax)) return STARK_ERR_INVALID_ARG;
    const Dims p = make_dims(shape);
    if (!prefix_tc_supported(p, shape->dtype, n_q) || total_tokens < 1) return STARK_ERR_UNSUPPORTED;
    rc = check_device();
    if (rc != STARK_OK) return rc;
    const int32_t* anc_l = anc ? anc + (size_t)(level & 1) * p.B * p.Wmax * p.d : nullptr;
    return launch_decode_fused(p, q, n_q, level, k_prefix, v_prefix, cu_seqlens, total_tokens, max_prefix_len,
                               plan_cluster_splits(p, n_q, max_prefix_len, total_tokens), k_suffix, v_suffix, anc_l, out,
                               (cudaStream_t)stream);
}

int stark_decode_step(const stark_shape_t* shape, const void* q, int n_q, int level, const void* k_prefix,
                      const void* v_prefix, const int32_t* cu_seqlens, int total_tokens, int max_prefix_len,
                      const void* k_new, const void* v_new, const int32_t* parent, void* k_suffix, void* v_suffix,
                      int32_t* anc, int write_anc, void* out, void* stream) {
    int rc = check_shape(shape);
    if (rc != STARK_OK) return rc;
    if (!q || !cu_seqlens || !out) return STARK_ERR_INVALID_ARG;
    if (n_q < 1 || total_tokens < 0 || max_prefix_len < 1 || level < 0 || level > shape->d) return STARK_ERR_INVALID_ARG;
    if (total_tokens > 0 && (!k_prefix || !v_prefix)) return STARK_ERR_INVALID_ARG;
    if (level >= 1 && (!k_new || !v_new || !k_suffix || !v_suffix || !anc || n_q > shape->Wmax)) return STARK_ERR_INVALID_ARG;
    if (level >= 2 && !parent) return STARK_ERR_INVALID_ARG;
    const Dims p = make_dims(shape);
    if (!prefix_tc_supported(p, shape->dtype, n_q) || total_tokens < 1) return STARK_ERR_UNSUPPORTED;
    rc = check_device();
    if (rc != STARK_OK) return rc;
    const size_t half = (size_t)p.B * p.Wmax * p.d;
    const int32_t* anc_prev = level >= 1 ? anc + (size_t)((level - 1) & 1) * half : nullptr;
    int32_t* anc_new = (level >= 1 && write_anc) ? anc + (size_t)(level & 1) * half : nullptr;
    return launch_decode_fused(p, q, n_q, level, k_prefix, v_prefix, cu_seqlens, total_tokens, max_prefix_len,
                               plan_cluster_splits(p, n_q, max_prefix_len, total_tokens), k_suffix, v_suffix, anc_prev, out,
                               (cudaStream_t)stream, level >= 1 ? k_new : nullptr, level >= 1 ? v_new : nullptr, parent,
                               anc_new);
}

int stark_beam_topk(const float* logp, const float* score_or_null, int B, int W_in, int C, int W_out,
                    float* out_score, int32_t* out_parent, int32_t* out_code, void* ws, size_t ws_bytes,
                    void* stream) {
    if (!logp || !out_score || !out_parent || !out_code) return STARK_ERR_INVALID_ARG;
    if (B < 1 || W_in < 1 || C < 1 || W_out < 1) return STARK_ERR_INVALID_ARG;
    if ((long long)W_in * C >= (1ll << 31)) return STARK_ERR_INVALID_ARG;
    if ((long long)W_out > (long long)W_in * C || W_out > 4096) return STARK_ERR_INVALID_ARG;
    const size_t need = topk_workspace_bytes(B, W_in, C);
    if (need > 0 && (!ws || ws_bytes < need)) return STARK_ERR_WORKSPACE;
    int rc = check_device();
    if (rc != STARK_OK) return rc;
    return launch_topk(logp, score_or_null, B, W_in, C, W_out, out_score, out_parent, out_code, ws, ws_bytes,
                       (cudaStream_t)stream);
}

int stark_logits_row_offset(const float* logits, const float* score_or_null, int64_t rows, int C,
                            float* offset, void* stream) {
    if (!logits || !offset || rows < 1 || C < 1) return STARK_ERR_INVALID_ARG;
    const int rc = check_device();
    if (rc != STARK_OK) return rc;
    return launch_row_offset(logits, score_or_null, (long long)rows, C, offset, (cudaStream_t)stream);
}

int stark_beam_topk_logits(const float* logits, const float* score_or_null, int B, int W_in, int C, int W_out,
                           float* out_score, int32_t* out_parent, int32_t* out_code, void* ws,
                           size_t ws_bytes, void* stream) {
    if (!logits || !out_score || !out_parent || !out_code) return STARK_ERR_INVALID_ARG;
    if (B < 1 || W_in < 1 || C < 1 || W_out < 1) return STARK_ERR_INVALID_ARG;
    if ((long long)W_in * C >= (1ll << 31)) return STARK_ERR_INVALID_ARG;
    if ((long long)W_out > (long long)W_in * C || W_out > 4096) return STARK_ERR_INVALID_ARG;
    const size_t off_bytes = offset_bytes(B, W_in), tk_bytes = topk_workspace_bytes(B, W_in, C);
    if (!ws || ws_bytes < off_bytes + tk_bytes) return STARK_ERR_WORKSPACE;
    int rc = check_device();
    if (rc != STARK_OK) return rc;
    if (topk_can_fold_lse(W_in, C))  // decode step 0: the one-CTA kernel normalises its single row itself
        return launch_topk(logits, score_or_null, B, W_in, C, W_out, out_score, out_parent, out_code,
                           static_cast<char*>(ws) + off_bytes, ws_bytes - off_bytes, (cudaStream_t)stream, true);
    float* offset = static_cast<float*>(ws);
    rc = launch_row_offset(logits, score_or_null, (long long)B * W_in, C, offset, (cudaStream_t)stream);
    if (rc != STARK_OK) return rc;
    return launch_topk(logits, offset, B, W_in, C, W_out, out_score, out_parent, out_code,
                       static_cast<char*>(ws) + off_bytes, ws_bytes - off_bytes, (cudaStream_t)stream);
}

int stark_kv_append_reorg(const stark_shape_t* shape, int level, int n_new, const void* k_new,
                          const void* v_new, const int32_t* parent, void* k_suffix, void* v_suffix,
                          int32_t* anc_or_null, void* stream) {
    int rc = check_shape(shape);
    if (rc != STARK_OK) return rc;
    if (!k_new || !v_new || !k_suffix || !v_suffix) return STARK_ERR_INVALID_ARG;
    if (level < 1 || level > shape->d || n_new < 1 || n_new > shape->Wmax) return STARK_ERR_INVALID_ARG;
    if (level >= 2 && anc_or_null && !parent) return STARK_ERR_INVALID_ARG;
    rc = check_device();
    if (rc != STARK_OK) return rc;
    return launch_append(make_dims(shape), shape->dtype, level, n_new, k_new, v_new, parent, k_suffix,
                         v_suffix, anc_or_null, (cudaStream_t)stream);
}

}  // extern "C"
