// Internal declarations shared by the host side (scd_host.cu) and the kernels.
// Nothing here is part of the C ABI (include/scd.h).
#pragma once

#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda.h>
#include <stdint.h>

#include <string>
#include <atomic>
#include <vector>

#include "scd.h"

namespace scd {

constexpr int SCD_MAX_DEVICES = 64;

// ---------------------------------------------------------------------------------
// Epilogue kinds of the one GEMM shape the whole path reduces to:
//     C[M, N] = A[M, K] * Bt[N, K]^T      (A, Bt both K-major)
// ---------------------------------------------------------------------------------
enum EpiKind : int {
  EPI_CODES = 0,   // encode:  z = acc - c[n]            -> codes (f32 | bf16 | e4m3 + row scale)
  EPI_KV = 1,      // decode / patch GEMM-3: y = acc * rowscale + add[n]; RoPE on K cols; paged write
  EPI_ACT = 2,     // patch GEMM-1: y = act(acc * rowscale + b1[n])     -> row-major state dtype
  EPI_U = 3        // patch GEMM-2: y = acc + b2[n]; partial sum of squares per (n-tile, row)
};

// ids under which scd_profile_fetch reports the launches of the tensor-core path
enum ProfId : int {
  SCD_PROF_ENCODE = 100, SCD_PROF_ENCODE_K = 101, SCD_PROF_REUSE_DECODE = 110, SCD_PROF_PATCH_GEMM1 = 120,
  SCD_PROF_PATCH_GEMM2 = 130, SCD_PROF_PATCH_GEMM3 = 140, SCD_PROF_INT4_QUANT = 200, SCD_PROF_INT4_DEQUANT = 201,
  SCD_PROF_FIT_GRAM = 300
};

enum AMode : int {
  A_PLAIN = 0,     // A is state dtype, used as is
  A_DEROPE = 1,    // A is the producer's post-RoPE K: rotate by -pos on load (Eq. 5)
  A_CODES = 2      // A is a code segment (code dtype; e4m3 carries row scales)
};

// Batch geometry as the kernels see it (device pointers).
struct BatchDev {
  const int32_t* cu_seqlens;
  const int32_t* page_table;
  const int32_t* pos_offset;   // may be null
  int32_t n_seqs, total_tokens, max_pages_per_seq, block_size;
  int32_t n_blocks;            // pages in the pool (0 = not checked): a page id outside [0, n_blocks) makes the row's slot -1
};

// RoPE geometry.  Tables hold (cos, sin) of p * theta^(-2j/d_h), [max_position][d_h/2].
struct RopeDev {
  const float2* table;
  int32_t head_dim, style, max_position;
};

// One GEMM problem ("segment"): a (layer, branch) slice of a hot call.
struct GemmSeg {
  const void* a;            // [M, K], row pitch lda elements (head-strided K/V: see a_head_stride)
  int64_t lda;
  int64_t a_head_stride;    // elements between heads of A (A_PLAIN/A_DEROPE on K/V); 0 = dense rows
  const float* a_scale;     // e4m3 codes: [M] row scales, else null
  const float* a_sub;       // SIMT path: [K] mean subtracted from A on load (exact (x - mu) W), else null
  const void* bt;           // [N, K] K-major, state dtype
  const float* col_vec;     // EPI_CODES: c[n] (subtracted); others: mean / bias [N] (added); may be null
  void* out0;               // EPI_CODES: codes; EPI_KV: pool for cols < split; EPI_ACT/EPI_U: [M, N]
  void* out1;               // EPI_KV: pool for cols >= split (or null)
  float* aux;               // EPI_CODES e4m3: row scales out; EPI_U: sumsq partials [ceil(N/tile)][M]
  const float* rowscale_in; // EPI_KV with NORM_RMS: sumsq partials [n_partials][M]; else null
  int32_t n_partials;       // number of partial rows to sum for NORM_RMS
  int32_t M, N, K;
  int32_t split;            // EPI_KV: first column that goes to out1 (N if none)
  int32_t pool_width;       // EPI_KV: elements per pool slot (D)
  int32_t rope_cols;        // EPI_KV: columns [0, rope_cols) get RoPE (multiple of head_dim)
  int32_t act;              // EPI_ACT: scd_act_t
  float rms_eps;            // EPI_KV NORM_RMS
  int32_t rms_dim;          // divisor of the sum of squares (d_model)
};

struct DevAlloc {
  void* ptr;
  size_t bytes;
};

// Plan-owned, repacked artifacts of one code segment (layer, branch).
struct SegPlan {
  int32_t layer, branch, rank, width;   // width = D (K, V) or d_model (H)
  void* enc_t;        // [rank, width]   W_enc^T, K-major B operand of encode
  float* enc_c;       // [rank]          c = mu_src * W_enc (fp64 -> fp32), zeros when no mean
  float* mean_src;    // [width] fp32 copy of mu_src, or null when absent (SIMT path subtracts it on load)
  void* dec_t;        // [D, rank]       W_dec^T, K-major B operand of decode (REUSE only)
  float* mean_dst;    // [D] fp32, zeros when absent (REUSE only)
  int32_t seg_index;  // order in the code buffer
};

struct PatchPlan {
  int32_t layer, r_h, d_a;
  void* w1_t;         // [d_a, r_h]
  float* b1;          // [d_a]
  void* w2_t;         // [d_model, d_a]
  float* b2;          // [d_model]
  void* wkv;          // [2D, d_model]  rows 0..D-1 = gamma (.) W_k, rows D..2D-1 = gamma (.) W_v
  float* bkv;         // [2D]
  int32_t h_seg;      // index into segs of this layer's H segment
};

}  // namespace scd

struct scd_plan {
  scd_model_desc_t model;
  std::vector<int32_t> kind, r_k, r_v, r_h, d_a;      // per layer
  std::vector<scd::SegPlan> segs;                     // code-buffer order: all K, all V, all H
  std::vector<int32_t> seg_of;                        // [layer * 3 + branch] -> seg index or -1
  std::vector<scd::PatchPlan> patches;
  float2* rope_prod = nullptr;                        // [max_position][d_h/2]
  float2* rope_cons = nullptr;
  std::vector<void*> allocs;                          // everything cudaMalloc'ed by the plan
  int32_t D = 0, sm_count = 0, device = 0;            // device: ordinal the plan was created on
  bool use_tc = false;                                // bf16 state -> tcgen05 kernels
  // tcgen05 path: plan-owned TMA descriptors of the B operands in device memory
  // ([0,nseg) encoders, [nseg,2nseg) decoders, then 3 per PATCH layer)
  void* tc_bmaps = nullptr;
  // tile-scheduler counters of the persistent paged-KV kernel: KV_SCHED_SETS pairs {next chunk, CTAs done},
  // zero between launches (the last CTA of a launch resets its pair); launches take the sets round-robin
  std::vector<int32_t> head_rank_k, head_rank_v;       // per layer: per-head ranks when model.reuse_per_head, else 0
  int32_t* kv_sched = nullptr;
  mutable std::atomic<uint32_t> kv_sched_next{0};
};

namespace scd {

// ---- error plumbing (scd_host.cu) -------------------------------------------------
scd_status_t fail(scd_status_t st, const char* fmt, ...);
void count_launch();
void reset_launch_count();               // at the top of every hot call (scd_last_launch_count)
// layer window of the running hot call: the *_layers entry points restrict a call to [layer_begin, layer_end)
bool layer_in_window(int layer);
// profiling hooks (scd_profile_enable): bracket one launch with events on `s`
void prof_begin(cudaStream_t s);
void prof_end(cudaStream_t s, int kernel_id);

// ---- layout (scd_host.cu) ---------------------------------------------------------
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline int code_elem_bytes(int code_dtype) { return code_dtype == SCD_F32 ? 4 : (code_dtype == SCD_BF16 ? 2 : 1); }
inline int state_elem_bytes(int state_dtype) { return state_dtype == SCD_F32 ? 4 : 2; }

// ---- plan-time repack kernels (scd_prep.cu) ----------------------------------------
cudaError_t prep_transpose(const void* src, void* dst, int rows, int cols, int state_dtype, cudaStream_t s);
// dst[n, k] = w[n, k] * gamma[k] (gamma may be null -> copy), rows = N, cols = K
cudaError_t prep_fold_gamma(const void* w, const void* gamma, void* dst, int rows, int cols, int state_dtype,
                            cudaStream_t s);
// c[n] = sum_k mu[k] * w_enc[k, n]  in fp64, stored fp32 (mu null -> zeros)
cudaError_t prep_mean_proj(const float* mu, const void* w_enc, float* c, int width, int rank, int state_dtype,
                           cudaStream_t s);
// dst[i] = (float) src[i] (src state dtype, may be null -> zeros)
cudaError_t prep_to_f32(const void* src, float* dst, int n, int state_dtype, cudaStream_t s);
cudaError_t prep_copy_f32(const float* src, float* dst, int n, cudaStream_t s);   // null -> zeros
// per-head REUSE reading: dst [H*rows, H*cols] = I_H (x) src [rows, cols] (state dtype); dst [H*n] = src [n] tiled H times
cudaError_t prep_block_diag(const void* src, void* dst, int rows, int cols, int heads, int state_dtype, cudaStream_t s);
cudaError_t prep_tile_f32(const float* src, float* dst, int n, int heads, cudaStream_t s);
// (cos, sin)(p * theta^(-2j/d_h)) evaluated in fp64, rounded to fp32
cudaError_t prep_rope_table(float2* table, int max_position, int head_dim, double theta, cudaStream_t s);

// ---- SIMT kernels (scd_simt.cu): fp32 path and debug path --------------------------
cudaError_t simt_gemm(const GemmSeg& seg, int epi, int a_mode, int state_dtype, int code_dtype,
                      const BatchDev& batch, const RopeDev& rope, cudaStream_t s);

}  // namespace scd
