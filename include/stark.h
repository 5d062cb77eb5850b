/*
 * stark.h -- C ABI of the B200-native STARK decode library.
 *
 * STARK = Semantic Tree Attention with Reorganized KV cache, the inference
 * scheme of UniSGR (arxiv/paper_2607_04068, section 3.6).
 * The library implements the per-step hot path of semantic-ID (SID) beam
 * search in which all beams of a user share ONE user-history prefix KV cache,
 * stored once, plus a tiny per-beam suffix of generated SID tokens tied
 * together by parent pointers.
 *
 * Conventions common to every call
 * --------------------------------
 *  - Every buffer argument is a DEVICE pointer allocated and owned by the
 *    caller unless the comment says "host".  The library allocates no device
 *    memory, keeps no state between calls (except the last CUDA error code),
 *    never synchronises the host with the device and never copies to the host.
 *  - Scalars and shapes are host values.
 *  - `stream` is a `cudaStream_t` passed as `void*` (NULL = legacy default
 *    stream).  Every call only enqueues work on it and returns; all calls are
 *    CUDA-graph capturable (shapes are static per step).
 *  - Return value: STARK_OK (0) or a negative stark_status_t.  Argument
 *    validation happens BEFORE any CUDA call, so it can be exercised on a
 *    machine without a GPU.  No exceptions, no aborts, nothing printed.
 *  - Inputs are assumed NaN-free; `-inf` log-probabilities are legal.
 *    Behaviour on NaN is unspecified but memory-safe.
 *  - Element type of q / K / V / out is `shape->dtype`: STARK_F32 (4 bytes) or
 *    STARK_BF16 (2 bytes, fp32 accumulation).  Partials, scores and log-probs
 *    are always fp32; indices are int32.
 *
 * Step indexing (reading R2): decode step t = 0..d-1 produces the
 * logits of SID level t+1.  Step 0 has n_q = 1 query per user (the last
 * prefix position; empty suffix).  Step t >= 1 has n_q = W_t queries per user
 * sitting at tree depth t; each sees the whole prefix of its user plus its
 * ancestor chain of t suffix nodes, itself included (Eq. 14 "or j = i",
 * PAPER.md:265-268).  The optional step t = d (ranking features,
 * PAPER.md:215) has chain length d.
 *
 * Layouts (all contiguous, innermost dimension last)
 *   q, out          [B, n_q, Hq, D]
 *   k_prefix,
 *   v_prefix        [total_tokens, Hkv, D]  users packed back to back
 *   cu_seqlens      [B+1] int32, cu_seqlens[0] = 0, user u owns rows
 *                   cu_seqlens[u] .. cu_seqlens[u+1]-1
 *   k_suffix,
 *   v_suffix        [d, B, Wmax, Hkv, D]    level l (1..d) lives at index l-1
 *   anc             [2, B, Wmax, d] int32   ping-pong by level parity: the
 *                   entries of the beams of level l are in half (l & 1);
 *                   anc[l&1][u][i][tau-1] = slot, at depth tau, of the
 *                   depth-tau ancestor of the beam in slot i (tau = 1..l;
 *                   entry l-1 is i itself)
 *   part_m, part_l  [n_splits, B, n_q, Hq] fp32
 *   part_o          [n_splits, B, n_q, Hq, D] fp32
 *   logp            [B, W_in, C] fp32;  score [B, W_in] fp32
 * Alignment: every tensor pointer is 16-byte aligned (bf16 q / k_prefix /
 * v_prefix / out are read and written through TMA tensor maps and 16-byte
 * vectors; a misaligned bf16 pointer makes the call return STARK_ERR_CUDA with
 * cudaErrorInvalidValue, nothing is launched).
 */
#ifndef STARK_H_
#define STARK_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define STARK_VERSION 100  /* major*10000 + minor*100 + patch */

typedef enum stark_status {
    STARK_OK = 0,
    STARK_ERR_INVALID_ARG = -1, /* null pointer, non-positive dim, Hq % Hkv != 0,
                                   W_out > W_in*C, level out of range, n_q > Wmax ... */
    STARK_ERR_UNSUPPORTED = -2, /* dtype / head_dim / device not supported */
    STARK_ERR_WORKSPACE = -3,   /* workspace pointer null or too small */
    STARK_ERR_CUDA = -4         /* a CUDA call failed; see stark_last_cuda_error() */
} stark_status_t;

typedef enum stark_dtype { STARK_F32 = 0, STARK_BF16 = 1 } stark_dtype_t;

/* Identifies a call in stark_workspace_bytes(). */
typedef enum stark_call {
    STARK_CALL_PREFIX_ATTN = 0,
    STARK_CALL_TREE_ATTN_STEP = 1,
    STARK_CALL_BEAM_TOPK = 2,
    STARK_CALL_KV_APPEND_REORG = 3,
    STARK_CALL_BEAM_TOPK_LOGITS = 4
} stark_call_t;

/* Static shape of one attention layer's decode problem. */
typedef struct stark_shape {
    int32_t B;     /* users in the batch (>= 1) */
    int32_t Hq;    /* query heads */
    int32_t Hkv;   /* KV heads; Hq % Hkv == 0, GQA group G = Hq / Hkv */
    int32_t D;     /* head_dim, 64 or 128 */
    int32_t d;     /* number of SID levels = maximum suffix chain length (1..8) */
    int32_t Wmax;  /* capacity (beams per user) of one suffix level */
    int32_t dtype; /* stark_dtype_t of q / K / V / out */
    float softmax_scale; /* 0 => 1/sqrt(D) (reading R3) */
} stark_shape_t;

/* ---------------------------------------------------------------------------
 * A1. Shared-prefix attention partials
 *
 * the conventional path recomputes attention over the shared
 * user-history prefix once per beam; STARK computes it "exactly once".  All
 * n_q beams x G group heads of a (user, KV head) are packed into the M
 * dimension of one contraction against that user's prefix K/V, so every prefix
 * byte is read from HBM once per step instead of once per beam.
 *
 * For every (split s, user u, query i < n_q, head h) with kv = h / G and
 * J_s(u) the prefix rows of user u that split s owns:
 *     x_j    = scale * <q[u,i,h,:], k_prefix[cu[u]+j, kv, :]>        j in J_s(u)
 *     part_m = max_j x_j                      (natural-log units; -inf if J empty)
 *     part_l = sum_j exp(x_j - part_m)        (0 if J empty)
 *     part_o = sum_j exp(x_j - part_m) * v_prefix[cu[u]+j, kv, :]   (unnormalised)
 * (split-softmax partials; merging them by log-sum-exp gives exact softmax
 * attention over the prefix.)  Split s of user u owns rows
 * [s*chunk_u, min((s+1)*chunk_u, L_u)), chunk_u = ceil(ceil(L_u/n_splits)/128)*128.
 * The library may keep a reference maximum m' >= true max - 8*ln2 instead of
 * the exact maximum in part_m (part_l, part_o are then relative to m'); the
 * merged result is unchanged.
 *
 * q            in   [B, n_q, Hq, D]          dtype
 * k_prefix,
 * v_prefix     in   [total_tokens, Hkv, D]   dtype; never written
 * cu_seqlens   in   [B+1] int32
 * total_tokens      host: number of rows of k_prefix / v_prefix
 * max_prefix_len    host: upper bound of L_u over the batch (>= 1)
 * n_splits          host: >= 1, or 0 to use stark_prefix_attn_plan()'s choice
 * part_m/l/o   out  fp32, sized for the n_splits actually used
 * ws, ws_bytes      workspace of stark_workspace_bytes(STARK_CALL_PREFIX_ATTN, ...)
 *                   bytes (may be NULL when that size is 0)
 * Errors: INVALID_ARG (null pointers, n_q < 1, total_tokens < 0,
 * max_prefix_len < 1, n_splits < 0 or > 64), UNSUPPORTED (D not in {64,128},
 * dtype), WORKSPACE, CUDA.
 */
int stark_prefix_attn(const stark_shape_t* shape, const void* q, int n_q,
                      const void* k_prefix, const void* v_prefix,
                      const int32_t* cu_seqlens, int total_tokens, int max_prefix_len,
                      int n_splits, float* part_m, float* part_l, float* part_o,
                      void* ws, size_t ws_bytes, void* stream);

/* Deterministic choice of n_splits from the shapes and the SM count of the
 * CURRENT device (one cudaGetDevice / cudaDeviceGetAttribute query, cached per
 * device; 148 is assumed when no device is present; no launch, no
 * synchronisation): 1 when the (user, KV head, M tile) grid alone fills the
 * GPU, more when it does not (step 0, small batches).  Writes *n_splits (host).
 * Call it with the device current on which stark_prefix_attn will run. */
int stark_prefix_attn_plan(const stark_shape_t* shape, int n_q, int total_tokens,
                           int max_prefix_len, int* n_splits);

/* ---------------------------------------------------------------------------
 * A2. Suffix tree attention + merge
 *
 * PAPER.md:263-268 (Eq. 14): a candidate token attends only to its ancestors
 * in the decoding tree and itself -- realised by walking the beam's ancestor
 * index instead of materialising the mask.  For each (u, i < n_q, h):
 *     chain: a_tau = anc[level&1][u][i][tau-1], tau = 1..level
 *     y_tau = scale * <q[u,i,h,:], k_suffix[tau-1][u][a_tau][kv][:]>
 *     out   = softmax over {prefix rows (through the partials), y_1..y_level}
 *             applied to the matching V rows, i.e. the log-sum-exp merge of
 *             all n_splits prefix partials with the chain's scores.
 * level = 0: no suffix; merge the splits and normalise (this also serves the
 * encoder-decoder cross-attention form, reading R1).  A query with
 * no visible key at all (empty prefix, level 0) yields zeros.
 *
 * q       in  [B, n_q, Hq, D] dtype     level  host, 0..d
 * k_suffix, v_suffix in [d, B, Wmax, Hkv, D] dtype (NULL allowed when level = 0)
 * anc     in  [2, B, Wmax, d] int32 (NULL allowed when level = 0)
 * part_*  in  as written by stark_prefix_attn with the same n_splits
 * out     out [B, n_q, Hq, D] dtype
 * Errors: INVALID_ARG (null pointers, level outside [0,d], n_q < 1,
 * n_q > Wmax when level >= 1, n_splits < 1), UNSUPPORTED, CUDA.
 */
int stark_tree_attn_step(const stark_shape_t* shape, const void* q, int n_q, int level,
                         const void* k_suffix, const void* v_suffix, const int32_t* anc,
                         const float* part_m, const float* part_l, const float* part_o,
                         int n_splits, void* out, void* stream);

/* ---------------------------------------------------------------------------
 * A1 + A2 fused: decode attention in ONE launch
 *
 * Same result as stark_prefix_attn followed by stark_tree_attn_step
 * (every query attends to its user's whole prefix
 * plus its own ancestor chain), but the split-softmax partials never leave the
 * chip: the CTAs that share one (query tile pair, KV head, user) form a
 * thread-block cluster over the prefix splits, exchange their partial rows
 * through distributed shared memory, and the owner of each 32-row block merges
 * them, adds the suffix chain and writes the normalised output.  Saves the
 * fp32 partial round trip through HBM (2 * n_splits * B*n_q*Hq*(D+2)*4 bytes),
 * the second read of q and one launch per step.
 *
 * Arguments as in the two separate calls; the split count (cluster size 1, 2,
 * 4 or 8) is chosen from shapes only.  bf16 only: returns
 * STARK_ERR_UNSUPPORTED for fp32 shapes (compose the two calls instead).
 * Errors: INVALID_ARG (null pointers, level outside [0,d], n_q < 1, n_q > Wmax
 * when level >= 1, total_tokens < 0, max_prefix_len < 1), UNSUPPORTED, CUDA.
 */
int stark_decode_attn(const stark_shape_t* shape, const void* q, int n_q, int level,
                      const void* k_prefix, const void* v_prefix, const int32_t* cu_seqlens,
                      int total_tokens, int max_prefix_len, const void* k_suffix,
                      const void* v_suffix, const int32_t* anc, void* out, void* stream);

/* ---------------------------------------------------------------------------
 * A4 + A1 + A2 fused: one whole decode step of a layer in ONE launch
 *
 * Same result, in `out`, in level `level` of k_suffix / v_suffix and in
 * anc[level&1], as
 *     stark_kv_append_reorg(shape, level, n_q, k_new, v_new, parent,
 *                           k_suffix, v_suffix, write_anc ? anc : NULL)
 *     stark_decode_attn(shape, q, n_q, level, ..., k_suffix, v_suffix, anc, out)
 * (PAPER.md:263-268 and 284-286).  A query's own K/V row is read from k_new /
 * v_new, its ancestors' slots from the PREVIOUS level's index through `parent`
 * (anc[(level-1)&1][u][parent[u,i]][0..level-2]), so nothing this launch writes
 * is read by it: the append is done by warps of the attention kernel that are
 * otherwise idle, and the step costs one launch instead of two.
 *
 * level 0 (the root queries its prefix) appends nothing: k_new, v_new, parent,
 * k_suffix, v_suffix and anc may be NULL.  level >= 1: all of them are needed,
 * except parent at level 1.  write_anc = 0 for layers > 0 of a decoder (the
 * tree is shared, layer 0 extends the index; `parent` is still read).
 * k_new, v_new  in [B, n_q, Hkv, D];  parent in [B, n_q] int32;  the rest as in
 * the separate calls.  bf16 only (UNSUPPORTED for fp32: compose the calls).
 * Errors: INVALID_ARG, UNSUPPORTED, CUDA.
 */
int stark_decode_step(const stark_shape_t* shape, const void* q, int n_q, int level,
                      const void* k_prefix, const void* v_prefix, const int32_t* cu_seqlens,
                      int total_tokens, int max_prefix_len, const void* k_new,
                      const void* v_new, const int32_t* parent, void* k_suffix, void* v_suffix,
                      int32_t* anc, int write_anc, void* out, void* stream);

/* ---------------------------------------------------------------------------
 * A3. Per-level beam selection
 *
 * Beam score = sum of per-level log-probabilities (Eq. 1);
 * each level keeps the top-W candidate paths.  For
 * every user u independently:
 *     key[i*C + c] = fl32(score[u,i] + logp[u,i,c])   -- ONE fp32 addition
 *     select the W_out entries first in the order (key descending, flat index
 *     i*C + c ascending; IEEE comparison: -0.0 == +0.0, -inf legal and last)
 *     slot r:  out_score = key, out_parent = idx / C, out_code = idx % C
 * The result is bit-exact and deterministic (no dependence on thread timing).
 *
 * logp       in  [B, W_in, C] fp32      score  in [B, W_in] fp32, NULL => zeros
 * out_score  out [B, W_out] fp32        out_parent, out_code out [B, W_out] int32
 * Caller passes W_out = min(W, W_in*C); widths may differ per level
 * (512, 512, 1024).
 * ws, ws_bytes   workspace of stark_workspace_bytes(STARK_CALL_BEAM_TOPK, ...)
 *                bytes (0 for small candidate sets: ws may then be NULL).  Large
 *                candidate sets are spread over all SMs of the GPU; the CTAs of a
 *                user meet through counters and lists in the workspace.  THE
 *                WORKSPACE MUST BE ZERO-FILLED BEFORE ITS FIRST USE (one
 *                cudaMemset after allocation); every call leaves it zero-filled
 *                again, so it can be reused by any later call that is ordered
 *                after this one (same stream / same graph); calls that may run
 *                concurrently need a workspace each.
 * Errors: INVALID_ARG (null pointers, non-positive dims, W_out > W_in*C,
 * W_out > 4096 -- reading R7: PAPER.md:306 needs at most 1024 --, W_in*C >= 2^31),
 * WORKSPACE (ws NULL or smaller than stark_workspace_bytes says), CUDA.
 */
int stark_beam_topk(const float* logp, const float* score_or_null, int B, int W_in, int C,
                    int W_out, float* out_score, int32_t* out_parent, int32_t* out_code,
                    void* ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------
 * A3 without a caller workspace: stark_beam_topk_static
 *
 * stark_beam_topk (same definition: Eq. 1, 257, 263, 306; same
 * kernels, same arguments, bit-identical result) for callers that cannot
 * allocate device memory: code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc.  The workspace is a static device array
 * inside the library:
 *   - it takes STARK_TOPK_STATIC_SCRATCH_BYTES of device memory on every GPU
 *     that loads the library, until the process exits;
 *   - a problem whose stark_workspace_bytes(STARK_CALL_BEAM_TOPK, ...) exceeds
 *     it is rejected with STARK_ERR_WORKSPACE (nothing is launched); on B200
 *     that is B > 29 users with W_in*C >= 131072 -- use stark_beam_topk then;
 *   - the call allocates nothing (no cudaMalloc / cudaFree / allocating
 *     library routine): argument checks, one cudaMemsetAsync that clears the
 *     part of the array this call uses, the kernel launches, all on `stream`;
 *   - ALL CALLS ON ONE GPU SHARE THE ARRAY: calls that may overlap on the GPU
 *     (streams without an ordering between them, several host threads) race
 *     and give undefined results.  Order them, or use stark_beam_topk with a
 *     workspace each;
 *   - the first call on a device looks the array's address up
 *     (cudaGetSymbolAddress): make it outside stream capture; every later call
 *     may be captured into a CUDA graph.
 * logp, score_or_null, out_*: device pointers, as for stark_beam_topk.
 * Errors: INVALID_ARG as stark_beam_topk, WORKSPACE (beyond the static
 * maximum), UNSUPPORTED (not an sm_100 device), CUDA.
 */
#define STARK_TOPK_STATIC_SCRATCH_BYTES (9u << 20)
int stark_beam_topk_static(const float* logp, const float* score_or_null, int B, int W_in, int C,
                           int W_out, float* out_score, int32_t* out_parent, int32_t* out_code,
                           void* stream);

/* ---------------------------------------------------------------------------
 * A3'. Beam selection straight from raw logits  (
 *      DESIGN.md reading R22)
 *
 * Eq. 1 needs log P(c | ...) = logit_c - logsumexp(logits of
 * the parent beam).  The normaliser is one scalar per parent beam; it is folded
 * into the beam's running score, the candidates are never rewritten:
 *     lse[u,i]    = fl32( logsumexp_c logits[u,i,c] )   fp64 arithmetic, rounded once
 *     offset[u,i] = fl32( score[u,i] - lse[u,i] )       ONE fp32 subtraction;
 *                   -inf if every logit of the beam is -inf (no legal continuation)
 *     key[i*C + c] = fl32( offset[u,i] + logits[u,i,c] ) ONE fp32 addition
 * followed by exactly stark_beam_topk's selection and outputs (out_score = key,
 * the new cumulative log-probability).  Equal to score + log-softmax(logits) up
 * to the rounding of the two fp32 operations; +inf logits are undefined.
 * Rounding guarantee: the log-sum-exp is evaluated in fp64 (error of a few
 * 1e-16 relative, depending on the summation order) and rounded ONCE to fp32, so
 * lse is the correctly rounded fp32 value of the exact log-sum-exp unless the
 * exact value lies within ~64 fp64 ulps (1.2e-7 of an fp32 ulp) of the midpoint
 * of two neighbouring fp32 numbers -- for logits without special structure a
 * probability of ~2.4e-7 per beam that the row is that close, and only then may
 * lse (hence the beam's keys, all together) differ by one fp32 ulp from another
 * correctly implemented fp64 evaluation.  The selection that follows is
 * bit-exact GIVEN the offsets (total order on (key, index)).
 *
 * stark_logits_row_offset is the first half on its own (rows = B*W_in beams,
 * logits [rows, C] fp32, score [rows] fp32 or NULL => zeros, offset out [rows]).
 * stark_beam_topk_logits runs both (one launch when W_in == 1 and C <= 512, i.e.
 * decode step 0: the one-CTA selection kernel normalises its single row itself;
 * two launches otherwise); ws, ws_bytes = workspace of
 * stark_workspace_bytes(shape (B only), STARK_CALL_BEAM_TOPK_LOGITS, W_in, C),
 * zero-filled before its first use like stark_beam_topk's (left zero-filled
 * except for the per-beam offsets at its front, which every call rewrites).
 * Errors: as stark_beam_topk; the workspace is always required.
 */
int stark_logits_row_offset(const float* logits, const float* score_or_null, int64_t rows, int C,
                            float* offset, void* stream);
int stark_beam_topk_logits(const float* logits, const float* score_or_null, int B, int W_in, int C,
                           int W_out, float* out_score, int32_t* out_parent, int32_t* out_code,
                           void* ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------
 * A4. KV append + index reorganisation
 *
 * K/V are stored once per tree node and referenced by
 * descendants through a pre-computed index mapping; expansion "appends newly
 * selected semantic tokens to the tree rather than duplicating the entire
 * prefix cache for every beam".  This call
 *   (1) copies k_new / v_new [B, n_new, Hkv, D] into slots 0..n_new-1 of level
 *       `level` of the suffix buffers, and
 *   (2) if anc != NULL, writes the ancestor index of the new level:
 *         anc[level&1][u][i][0..level-2] = anc[(level-1)&1][u][parent[u,i]][0..level-2]
 *         anc[level&1][u][i][level-1]    = i
 * The prefix region is neither read nor written.  The tree is shared by all
 * layers of a decoder while K/V are per layer: pass anc = NULL for layers > 0
 * of the same step.  level = 1 ignores `parent` (the root is the last prefix
 * row) and `parent` may be NULL.
 *
 * level  host, 1..d        n_new  host, 1..Wmax
 * parent in [B, n_new] int32, values in [0, Wmax) (slot at level-1)
 * Errors: INVALID_ARG, UNSUPPORTED, CUDA.
 */
int stark_kv_append_reorg(const stark_shape_t* shape, int level, int n_new,
                          const void* k_new, const void* v_new, const int32_t* parent,
                          void* k_suffix, void* v_suffix, int32_t* anc_or_null, void* stream);

/* ---------------------------------------------------------------------------
 * Sizes the caller must allocate (host arithmetic only).
 */
/* Workspace bytes for `call`.  For STARK_CALL_BEAM_TOPK and
 * STARK_CALL_BEAM_TOPK_LOGITS pass n_q = W_in, total_tokens = C and
 * shape->B = B (other shape fields ignored; the size does not depend on
 * W_out); the other calls currently need none and return 0.  Returns 0 on
 * invalid input.  See stark_beam_topk for the zero-fill rule. */
size_t stark_workspace_bytes(const stark_shape_t* shape, int call, int n_q, int total_tokens);
/* Bytes of ONE of k_suffix / v_suffix: d*B*Wmax*Hkv*D*elem. */
size_t stark_suffix_bytes(const stark_shape_t* shape);
/* Bytes of anc: 2*B*Wmax*d*4. */
size_t stark_anc_bytes(const stark_shape_t* shape);

int stark_version(void);
/* Static string describing a stark_status_t. */
const char* stark_status_string(int status);
/* cudaError_t (as int) of the most recent failing CUDA call in this thread's
 * process, 0 if none. */
int stark_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* STARK_H_ */
