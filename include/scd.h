/* scd.h -- C ABI of the B200-native SCD KV state codec (arxiv/paper_2606_07684).
 *
 * Semantic Cache Distillation replaces raw KV transmission between a producer model
 * M_A and a weight-mismatched consumer M_B of the same architecture by per-layer
 * low-rank "semantic codes".  This library is the data-parallel hot
 * path of that method on one B200 (sm_100a):
 *
 *   scd_plan          static routing table + artifact store   (Alg.1 :174)
 *   scd_encode        producer:  Z_K = deRoPE(K_A) W_enc,K ; Z_V = V_A W_enc,V   (Eq. 5, Eq. 8 :145)
 *                                Z_H = x_norm,A W_enc,H on PATCH layers          (Eq. 10, :165)
 *   scd_reuse_decode  consumer:  K_B = RoPE(Z_K W_dec,K) ; V_B = Z_V W_dec,V     (Eq. 9 :150, :152)
 *   scd_patch         consumer:  H^ = g_theta(Z_H) ; K^ = RoPE(H^ W_k) ; V^ = H^ W_v   (Eq. 11 :171, Eq. 12 :190-193)
 *
 * Results are written straight into a paged KV cache (the "cache container" of
 * PAPER.md:610, here a pool of `block_size`-token pages; build extension).
 *
 * Conventions
 *  - extern "C", plain pointers and sizes; no exceptions, no global mutable state.
 *  - Unless a comment says HOST, every data pointer is a DEVICE pointer that the caller
 *    owns ("borrowed"); the library never frees or keeps it past the call, except that
 *    scd_plan keeps its own repacked copies of the artifacts.
 *  - Hot calls (scd_encode / scd_reuse_decode / scd_patch) enqueue kernels on `stream`
 *    (a cudaStream_t passed as void*) and return without synchronising or allocating.
 *  - Argument / shape / alignment problems are detected on the host and returned as a
 *    status before anything is enqueued; scd_last_error() gives a thread-local message.
 *  - Layer indices are 0-based.  All matrices are row-major.
 *  - Alignment: every base pointer 16 B (128 B recommended), code buffer 128 B; strides
 *    of bf16 tensors multiples of 8 elements (TMA needs 16-B pitches).
 *  - Writes: exactly the slots { page_table[b][t/bs]*bs + t%bs : 0 <= t < len_b } of the
 *    addressed layers' pools, nothing else.
 */
#ifndef SCD_H_
#define SCD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SCD_MAX_LAYERS 128

typedef struct scd_plan scd_plan_t;          /* opaque; immutable after creation */

typedef enum {
  SCD_OK = 0,
  SCD_E_ARG = 1,          /* NULL / out-of-range argument                         */
  SCD_E_SHAPE = 2,        /* inconsistent shapes                                  */
  SCD_E_UNSUPPORTED = 3,  /* legal but not implemented combination */
  SCD_E_ALIGN = 4,        /* pointer / stride alignment                            */
  SCD_E_WORKSPACE = 5,    /* workspace too small                                   */
  SCD_E_CUDA = 6,         /* CUDA runtime / driver error                           */
  SCD_E_NOMEM = 7
} scd_status_t;

typedef enum { SCD_F32 = 0, SCD_BF16 = 1, SCD_E4M3_ROWSCALE = 2 } scd_dtype_t;
typedef enum { SCD_REUSE = 0, SCD_PATCH = 1 } scd_kind_t;
typedef enum { SCD_BRANCH_K = 0, SCD_BRANCH_V = 1, SCD_BRANCH_H = 2 } scd_branch_t;
/* HALF = HF rotate_half, pairs (j, j + d_h/2); INTERLEAVED pairs (2j, 2j+1). */
typedef enum { SCD_ROPE_HALF = 0, SCD_ROPE_INTERLEAVED = 1 } scd_rope_t;
typedef enum { SCD_ACT_IDENTITY = 0, SCD_ACT_SILU = 1 } scd_act_t;
/* NORM_NONE is the paper-literal Eq. 11-12; NORM_RMS: h = gamma * u / sqrt(mean(u^2)+eps). */
typedef enum { SCD_NORM_NONE = 0, SCD_NORM_RMS = 1 } scd_norm_t;

/* Model-pair geometry; producer and consumer share the architecture. */
typedef struct {
  int32_t n_layers;        /* 1 .. SCD_MAX_LAYERS                                        */
  int32_t d_model;
  int32_t n_kv_heads;
  int32_t head_dim;        /* 32, 64 or 128                                              */
  int32_t block_size;      /* tokens per KV page (16)                                    */
  int32_t max_position;    /* RoPE table length; every position id must be < this        */
  int32_t state_dtype;     /* scd_dtype_t F32 | BF16: K/V/hidden, artifacts, pools       */
  int32_t code_dtype;      /* scd_dtype_t F32 | BF16 | E4M3_ROWSCALE                     */
  double  rope_theta_producer;
  double  rope_theta_consumer;
  int32_t rope_style;      /* scd_rope_t                                                 */
  int32_t k_is_roped;      /* producer K is post-RoPE: encode applies deRoPE (Eq. 5)     */
  int32_t rope_on_reuse_k; /* decode re-applies RoPE to K; 0 for tests    */
  int32_t patch_act;       /* scd_act_t                                                  */
  int32_t patch_norm;      /* scd_norm_t                                                 */
  float   rms_eps;
  /* REUSE translator reading.  0: one basis per layer over all heads, enc [D, r], dec [r, D],
   * means [D] (the shapes BASELINE.json's configs use).  1: the paper's own Sec. 4.1
   * form: batch x heads x tokens are one sample axis and ONE map per
   * layer and branch serves every KV head -- enc [d_h, r], dec [r, d_h], means [d_h].  A token's
   * code row is then its heads' codes side by side: scd_plan_code_segment reports rank
   * n_kv_heads * r, and r_k / r_v below are the per-head ranks.  PATCH layers are unaffected. */
  int32_t reuse_per_head;
} scd_model_desc_t;

/* One per layer.  Artifacts are in state_dtype unless typed float. NULL means "absent"
 * (mean / bias = 0).  REUSE fields are read when kind == SCD_REUSE, PATCH fields when
 * kind == SCD_PATCH.  D = n_kv_heads * head_dim. */
typedef struct {
  int32_t kind;                      /* scd_kind_t                                       */
  int32_t r_k, r_v;                  /* REUSE ranks, independent          */
  const void *enc_k, *enc_v;         /* [D, r]  producer encoders  (Eq. 7-8); [d_h, r] if reuse_per_head */
  const void *dec_k, *dec_v;         /* [r, D]  consumer decoders  (Eq. 6, 9); [r, d_h] if reuse_per_head */
  const float *mean_src_k, *mean_src_v;   /* [D] ([d_h] if reuse_per_head) subtracted before encode, or NULL */
  const float *mean_dst_k, *mean_dst_v;   /* [D] ([d_h] if reuse_per_head) added after decode, or NULL      */
  int32_t r_h, d_aligner;            /* PATCH: code rank r_H, aligner hidden width d_a   */
  const void *enc_h;                 /* [d_model, r_h]                   */
  const float *mean_src_h;           /* [d_model] or NULL                                */
  const void *w1, *b1;               /* [r_h, d_a], [d_a]     aligner layer 1 (Eq. 11)   */
  const void *w2, *b2;               /* [d_a, d_model], [d_model]  aligner layer 2       */
  const void *norm_gamma;            /* [d_model] consumer RMSNorm weight (NORM_RMS)     */
  const void *w_k, *w_v;             /* [D, d_model]  HF layout [out, in]  (Eq. 12)      */
  const void *b_k, *b_v;             /* [D] or NULL                                      */
} scd_layer_desc_t;

/* A ragged batch.  Packed row n = cu_seqlens[b] + t; position id = pos_offset[b] + t. */
typedef struct {
  int32_t n_seqs, total_tokens, max_seqlen, max_pages_per_seq;
  const int32_t *cu_seqlens;         /* [n_seqs + 1]                                     */
  const int32_t *page_table;         /* [n_seqs, max_pages_per_seq] block ids, unused -1; the table lives on the
                                        device and is not validated by the host: a token whose page id is outside
                                        [0, n_blocks) is skipped (its row is not written), never stored out of the pool */
  const int32_t *pos_offset;         /* [n_seqs] first position id, or NULL (= 0)        */
  int32_t max_pos_offset;            /* HOST upper bound on pos_offset[] (0 if NULL)     */
} scd_batch_t;

/* Producer states.  k, v, h are HOST arrays of n_layers DEVICE pointers. */
typedef struct {
  const void *const *k;              /* [n_layers] -> [total_tokens, H_kv, d_h]; REUSE layers read */
  const void *const *v;
  const void *const *h;              /* [n_layers] -> [total_tokens, d_model]; PATCH layers read   */
  int64_t kv_token_stride, kv_head_stride, h_token_stride;   /* in elements              */
  /* Paged producer cache ("native cache semantics"): when page_table is not
   * NULL, k[l] / v[l] point to the PRODUCER's paged pools [n_blocks, block_size, H_kv, d_h] (dense heads;
   * kv_token_stride = elements between slots) and token t of request b is read from slot
   * page_table[b][t / bs] * bs + t % bs -- the encode gathers rows through the table (TMA tile::gather4), no
   * packed copy is made.  h stays packed [total_tokens, d_model].  The table lives on the device and is trusted:
   * a page id outside [0, n_blocks) reads slot 0 instead (that token's codes are then meaningless, nothing is
   * read out of bounds).  bf16 states only. */
  const int32_t *page_table;         /* DEVICE [n_seqs, max_pages_per_seq] or NULL (packed rows) */
  int32_t max_pages_per_seq, n_blocks;
} scd_src_t;

/* Consumer paged pool.  k_pool, v_pool are HOST arrays of n_layers DEVICE pointers, each
 * -> [n_blocks, block_size, H_kv, d_h] in state_dtype.
 * fp8 pools (build extension, DESIGN.md section 2 U20): pool_e4m3 != 0 makes the pools
 * [n_blocks, block_size, H_kv, d_h] e4m3fn BYTES with one fp32 scale per (slot, head) in k_scale[l] / v_scale[l]
 * -> [n_blocks, block_size, H_kv]: for each head of a token, x = the bf16 value the codec would have stored,
 * s = amax_head / 448 (1 if the head is all zero), stored byte = e4m3_rne_sat(x * (1 / s)) in IEEE fp32.
 * bf16 states, head_dim 128, HALF RoPE only (else SCD_E_UNSUPPORTED). */
typedef struct {
  void *const *k_pool;
  void *const *v_pool;
  int32_t n_blocks;
  int32_t pool_e4m3;                 /* 0: pools in state_dtype; 1: e4m3 bytes + per-(slot, head) fp32 scales */
  float *const *k_scale;             /* HOST arrays of n_layers DEVICE pointers, used when pool_e4m3 != 0 */
  float *const *v_scale;
} scd_paged_kv_t;

/* Create a plan: validates, classifies layers (REUSE | PATCH), copies and repacks the
 * artifacts into plan-owned device memory (transposes to K-major, folds gamma into
 * W_k|W_v, precomputes c = mu_src W_enc in fp64 and the RoPE tables), builds the TMA
 * descriptors of the plan-owned operands.  Work is enqueued on `stream`; the caller may
 * free its artifact buffers after synchronising it.  *out is NULL on failure. */
scd_status_t scd_plan(const scd_model_desc_t* model, const scd_layer_desc_t* layers /* HOST [n_layers] */,
                      void* stream, scd_plan_t** out);
scd_status_t scd_plan_destroy(scd_plan_t* plan);

/* Sizes for a call over `total_tokens` packed rows: code buffer bytes (with padding),
 * the workspace scd_patch prefers (the intermediates of as many PATCH layers as it runs
 * per launch: up to 2 GiB, never more than all of them), and the transport payload |Z| of
 * Eq. 3 (codes + e4m3 scales, no padding).  Any out pointer may be NULL. */
scd_status_t scd_plan_query(const scd_plan_t* plan, int32_t total_tokens,
                            size_t* code_bytes, size_t* patch_workspace_bytes, size_t* payload_bytes);

/* Where the codes of (layer, branch) live in the code buffer: [total_tokens, rank]
 * row-major in code_dtype at `offset`; for E4M3_ROWSCALE the fp32 row scales
 * [total_tokens] at `scale_offset` (else (size_t)-1).  REUSE layers have branches K, V;
 * PATCH layers branch H; anything else is SCD_E_ARG. */
scd_status_t scd_plan_code_segment(const scd_plan_t* plan, int32_t layer, int32_t branch,
                                   int32_t total_tokens, size_t* offset, size_t* scale_offset,
                                   int32_t* rank);

/* The same layout arithmetic as a pure HOST function (no plan, no CUDA): used to size
 * buffers before a plan exists and by the CPU tests.  Only kind, r_k, r_v, r_h of each
 * layer are read.  layer < 0 skips the per-segment outputs. */
scd_status_t scd_code_layout(const scd_model_desc_t* model, const scd_layer_desc_t* layers,
                             int32_t total_tokens, int32_t layer, int32_t branch,
                             size_t* offset, size_t* scale_offset, int32_t* rank,
                             size_t* code_bytes, size_t* payload_bytes);

/* Producer side (Alg. 1 :176-180).  Reads K, V of every REUSE layer and H of every PATCH
 * layer, writes every code segment of `codes` (size >= code_bytes). */
scd_status_t scd_encode(const scd_plan_t* plan, const scd_batch_t* batch, const scd_src_t* src,
                        void* codes, void* stream);

/* Consumer side, REUSE layers only (Alg. 1 :182-184): codes x basis (+ mean), RoPE on K,
 * cast, paged write. */
scd_status_t scd_reuse_decode(const scd_plan_t* plan, const scd_batch_t* batch, const void* codes,
                              const scd_paged_kv_t* kv, void* stream);

/* Consumer side, PATCH layers only (Eq. 11-12): aligner -> RMS-consistent scaling ->
 * [W_k | W_v] -> RoPE on K -> paged write.  `workspace` (DEVICE, 128-byte aligned, caller
 * owned, contents undefined afterwards): patch_workspace_bytes of scd_plan_query is the
 * preferred size; anything that holds one PATCH layer's intermediates is accepted (fewer
 * layers per launch), less returns SCD_E_WORKSPACE before anything is enqueued. */
scd_status_t scd_patch(const scd_plan_t* plan, const scd_batch_t* batch, const void* codes,
                       const scd_paged_kv_t* kv, void* workspace, size_t workspace_bytes, void* stream);

/* Layer-streamed variants: the same three calls restricted to layers [layer_begin, layer_end)
 * (0 <= begin <= end <= n_layers, else SCD_E_ARG).  Code segments are per (layer, branch)
 * (scd_plan_code_segment), so a producer can encode a group of layers, hand their segments
 * to the transport, and go on with the next group while the consumer decodes / patches the
 * groups that have arrived: the three terms of Eq. 3 pipelined instead of
 * summed.  Source states, code segments and pools of layers outside the window are neither
 * read, written nor validated (their pointers may be NULL); a window without REUSE (PATCH)
 * layers makes scd_reuse_decode_layers (scd_patch_layers) a no-op returning SCD_OK. */
scd_status_t scd_encode_layers(const scd_plan_t* plan, const scd_batch_t* batch, const scd_src_t* src,
                               void* codes, int32_t layer_begin, int32_t layer_end, void* stream);
scd_status_t scd_reuse_decode_layers(const scd_plan_t* plan, const scd_batch_t* batch, const void* codes,
                                     const scd_paged_kv_t* kv, int32_t layer_begin, int32_t layer_end,
                                     void* stream);
scd_status_t scd_patch_layers(const scd_plan_t* plan, const scd_batch_t* batch, const void* codes,
                              const scd_paged_kv_t* kv, void* workspace, size_t workspace_bytes,
                              int32_t layer_begin, int32_t layer_end, void* stream);

/* ---------------------------------------------------------------------------------------------
 * scd_patch without a caller workspace and without any allocation: for callers that cannot call
 * cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  The same
 * operation as scd_patch (Eq. 11, 12a/b), the same kernels; the intermediates
 * (aligner activations a [T, d_a], u [T, d_model], sum-of-squares partials) live in a file-scope
 * `static __device__` array of SCD_PATCH_STATIC_WORKSPACE_BYTES inside the library, which every GPU that
 * loads the library holds until the process exits.  The caller passes inputs and outputs only.
 *   - Limit: one PATCH layer's intermediates of the batch must fit: scd_plan_query's workspace for ONE layer,
 *     about total_tokens * (d_aligner + d_model) * sizeof(state) bytes (32 MiB = ~2000 tokens at d_model 4096
 *     in bf16).  Larger batches return SCD_E_WORKSPACE with the sizes in scd_last_error(); nothing is
 *     enqueued.  Layers are grouped per launch by what the array holds, exactly as scd_patch does with a
 *     small caller workspace (bit-identical results).
 *   - The plan's device must be the current device.
 *   - Calls no cudaMalloc / cudaFree / allocating library routine (the array's device address is looked up once
 *     per device with cudaGetSymbolAddress).  Enqueues on `stream` and returns, like scd_patch.
 *   - ALL calls on a device share the one array, which keeps the previous call's contents.  Nothing in it has to
 *     start at zero (every byte a call reads was written earlier by the same call), so nothing is cleared; but two
 *     calls that overlap on the GPU (different streams, no ordering between them) RACE on it -- serialise them,
 *     or use scd_patch with separate workspaces. */
#define SCD_PATCH_STATIC_WORKSPACE_BYTES (32u << 20)
scd_status_t scd_patch_static(const scd_plan_t* plan, const scd_batch_t* batch, const void* codes,
                              const scd_paged_kv_t* kv, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Group-wise INT4 KV codec -- the paper's fastest transport baseline ("Quantized KV: transmits 4-bit
 * quantized KV caches (group-wise INT4) and dequantizes on the consumer"; Table 4
 * :352-359), built as the same-box comparison codec.  The paper fixes neither group
 * size nor range convention; reading (U19): a group is `group` consecutive channels
 * of one token row (32, 64 or 128, dividing head_dim), lo = min, hi = max of the group,
 * s = bf16((hi - lo) / 15) (1 if that is 0), q = clamp(rint((x - lo) * (1 / s)), 0, 15), all in IEEE fp32;
 * byte j of a row = q[2j] | q[2j+1] << 4; metadata per group = {bf16 s, bf16 lo} (4 bytes);
 * dequantised x^ = bf16(q * s + lo).  Bit-exact against oracle/int4_oracle.py.
 *
 * Packed buffer (DEVICE, 128-byte aligned, caller owned): tensor i at i * tensor_stride holds the nibbles
 * [T, W/2] at 0 and the metadata [T, W/group] x {bf16 scale, bf16 zero point} at meta_offset
 * (W = n_kv_heads * head_dim).  A "tensor" is one layer's K or V; the caller chooses the order.
 * Both calls enqueue on `stream` and return; no allocation, no synchronisation; statuses as above.
 * --------------------------------------------------------------------------------------------- */
typedef struct {
  int32_t n_kv_heads, head_dim, block_size, group;
} scd_int4_desc_t;

/* Layout arithmetic (pure host).  payload_bytes = |Z| of Eq. 3: nibbles + metadata, no padding.
 * Any out pointer may be NULL. */
scd_status_t scd_int4_layout(const scd_int4_desc_t* desc, int32_t total_tokens, int32_t n_tensors,
                             size_t* tensor_stride, size_t* meta_offset, size_t* total_bytes, size_t* payload_bytes);

/* Producer: src = HOST array of n_tensors DEVICE pointers -> [total_tokens, H_kv, d_h] bf16 with dense heads
 * and `token_stride` elements between token rows (multiple of 8, >= W); writes every tensor's segment of
 * `packed`. */
scd_status_t scd_int4_quantize(const scd_int4_desc_t* desc, int32_t total_tokens, int32_t n_tensors,
                               const void* const* src, int64_t token_stride, void* packed, void* stream);

/* Consumer: dequantises tensor i into pools[i] (HOST array of DEVICE pointers ->
 * [n_blocks, block_size, H_kv, d_h] bf16) at slot = page_table[b][t / bs] * bs + t % bs; slots outside the
 * batch are not written; a page id outside [0, n_blocks) skips the token.  pos_offset is not used. */
scd_status_t scd_int4_dequantize_paged(const scd_int4_desc_t* desc, const scd_batch_t* batch, int32_t n_tensors,
                                       const void* packed, void* const* pools, int32_t n_blocks, void* stream);


/* ---------------------------------------------------------------------------------------------
 * Offline REUSE calibration fit: "Layer-wise Stack-SVD with Ridge Regression"
 * (section 4.3.1, Eq. 6-7; App. F.1 :583-586; Table 6 :602 "Reuse fitting").  For one
 * (layer, branch): paired samples A (producer), B (consumer), both [n_rows, width] bf16 row-major with
 * `row_stride` elements between rows (keys in content space, i.e. deRoPE'd, Eq. 5); X = [A B];
 *   V_r   = top-`rank` right singular vectors of X (of X minus its column means when center != 0)
 *   W_dec = V_r^T = [W_dec,A | W_dec,B]  ([rank, width] each; Eq. 6 with Z = X V_r, reading U4)
 *   W_enc = (A^T A + lam I)^-1 A^T Z,  lam = lam_rel * trace(A^T A) / width      (Eq. 7, reading U4)
 *   sigma = the top singular values; mu_a, mu_b = column means (center != 0; reading U2).
 * V_r is unique only up to the sign of each direction: compare V_r V_r^T, sigma and W_enc W_dec, never entries.
 * Outputs (DEVICE) are written in out_dtype (F32 or BF16; sigma and means always fp32); w_dec_a, sigma may be NULL.
 * The per-head reading is width = head_dim with the heads flattened into n_rows.
 * NOT a hot call: it enqueues on `stream` and SYNCHRONISES it once per Jacobi sweep (convergence test);
 * sweeps (HOST [2], may be NULL) receives the sweeps of the joint and of the ridge eigen-solve (at most 60 each).  Workspace (DEVICE,
 * 256-byte aligned, scd_fit_query bytes: the K-major copy of X dominates, 4 * width * n_rows bytes).
 * width: multiple of 8, <= 1024; bf16 states only (else SCD_E_UNSUPPORTED).
 * --------------------------------------------------------------------------------------------- */
typedef struct {
  int32_t width, rank, center;
  float lam_rel;
  scd_dtype_t state_dtype, out_dtype;
} scd_fit_desc_t;

scd_status_t scd_fit_query(const scd_fit_desc_t* desc, int64_t n_rows, size_t* workspace_bytes);
scd_status_t scd_fit_reuse(const scd_fit_desc_t* desc, const void* a, const void* b, int64_t n_rows, int64_t row_stride,
                           void* w_enc /* [width, rank] */, void* w_dec_a /* [rank, width] */, void* w_dec_b /* [rank, width] */,
                           float* mu_a /* [width] */, float* mu_b /* [width] */, float* sigma /* [rank] */,
                           void* workspace, size_t workspace_bytes, int32_t* sweeps, void* stream);

/* Number of kernels the last hot call on this thread enqueued (for bench accounting). */
int32_t scd_last_launch_count(void);

/* Per-kernel timing for measurement harnesses.  While enabled (on != 0) every kernel a hot
 * call on this thread enqueues is bracketed by CUDA events on the caller's stream.
 * scd_profile_fetch synchronises those events and returns, for up to `max` launches since
 * the last fetch, the elapsed milliseconds and a kernel id
 * (100*path + 10*epilogue + a_mode; path 0 = SIMT, 1 = tcgen05; epilogue 0 codes, 1 paged KV,
 * 2 aligner-in, 3 aligner-out; a_mode 0 plain, 1 deRoPE, 2 codes).  Returns the number of
 * launches recorded (may exceed max).  Off by default; adds two event records per launch. */
scd_status_t scd_profile_enable(int32_t on);
int32_t scd_profile_fetch(float* ms /* HOST [max] */, int32_t* kernel_id /* HOST [max] */, int32_t max);

/* Thread-local message for the last non-OK status returned on this thread ("" if none). */
const char* scd_last_error(void);

/* sizeof() of the ABI structs as this library was compiled (0 model, 1 layer, 2 batch, 3 src, 4 paged_kv, 5 int4 desc,
 * 6 fit desc; -1 otherwise): lets a binding verify its struct layouts before the first call. */
int32_t scd_struct_size(int32_t which);

/* Library version string. */
const char* scd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SCD_H_ */
