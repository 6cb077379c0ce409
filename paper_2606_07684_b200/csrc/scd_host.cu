// Host side of the C ABI (include/scd.h): validation, the static routing table and
// artifact store (scd_plan), code-buffer layout, and the launch logic of the three hot
// calls.  No arithmetic of the method happens on the host.
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "scd_internal.h"
#include "scd_tc.h"

namespace scd {

static thread_local char g_err[512] = "";
static thread_local int g_launches = 0;

scd_status_t fail(scd_status_t st, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return st;
}
void count_launch() { ++g_launches; }
void reset_launch_count() { g_launches = 0; }
static thread_local int g_layer_begin = 0, g_layer_end = 1 << 30;
bool layer_in_window(int layer) { return layer >= g_layer_begin && layer < g_layer_end; }
struct LayerWindow {                       // scoped: set by the *_layers entry points
  LayerWindow(int b, int e) { g_layer_begin = b; g_layer_end = e; }
  ~LayerWindow() { g_layer_begin = 0; g_layer_end = 1 << 30; }
};

struct ProfRec { cudaEvent_t a, b; int id; };
static thread_local bool g_prof_on = false;
static thread_local std::vector<ProfRec>* g_prof = nullptr;
void prof_begin(cudaStream_t s) {
  if (!g_prof_on) return;
  if (!g_prof) g_prof = new std::vector<ProfRec>();
  ProfRec r{};
  cudaEventCreate(&r.a);
  cudaEventCreate(&r.b);
  cudaEventRecord(r.a, s);
  g_prof->push_back(r);
}
void prof_end(cudaStream_t s, int kernel_id) {
  if (!g_prof_on || !g_prof || g_prof->empty()) return;
  g_prof->back().id = kernel_id;
  cudaEventRecord(g_prof->back().b, s);
}

#define SCD_CUDA(expr)                                                                          \
  do {                                                                                          \
    cudaError_t _e = (expr);                                                                    \
    if (_e != cudaSuccess) return fail(SCD_E_CUDA, "%s: %s", #expr, cudaGetErrorString(_e));    \
  } while (0)

// ---------------------------------------------------------------------------------
// validation of the descriptors (host only)
// ---------------------------------------------------------------------------------
static scd_status_t check_model(const scd_model_desc_t* m) {
  if (!m) return fail(SCD_E_ARG, "model is NULL");
  if (m->n_layers < 1 || m->n_layers > SCD_MAX_LAYERS)
    return fail(SCD_E_ARG, "n_layers %d outside [1, %d]", m->n_layers, SCD_MAX_LAYERS);
  if (m->d_model < 1 || m->n_kv_heads < 1) return fail(SCD_E_SHAPE, "d_model / n_kv_heads must be positive");
  if (m->head_dim != 32 && m->head_dim != 64 && m->head_dim != 128)
    return fail(SCD_E_UNSUPPORTED, "head_dim %d (supported: 32, 64, 128)", m->head_dim);
  if (m->block_size < 1) return fail(SCD_E_ARG, "block_size must be positive");
  if (m->max_position < 1) return fail(SCD_E_ARG, "max_position must be positive");
  if (m->state_dtype != SCD_F32 && m->state_dtype != SCD_BF16)
    return fail(SCD_E_ARG, "state_dtype must be F32 or BF16");
  if (m->code_dtype != SCD_F32 && m->code_dtype != SCD_BF16 && m->code_dtype != SCD_E4M3_ROWSCALE)
    return fail(SCD_E_ARG, "code_dtype must be F32, BF16 or E4M3_ROWSCALE");
  if (m->rope_style != SCD_ROPE_HALF && m->rope_style != SCD_ROPE_INTERLEAVED)
    return fail(SCD_E_ARG, "rope_style");
  if (m->patch_act != SCD_ACT_IDENTITY && m->patch_act != SCD_ACT_SILU) return fail(SCD_E_ARG, "patch_act");
  if (m->patch_norm != SCD_NORM_NONE && m->patch_norm != SCD_NORM_RMS) return fail(SCD_E_ARG, "patch_norm");
  if (!(m->rope_theta_producer > 0.0) || !(m->rope_theta_consumer > 0.0))
    return fail(SCD_E_ARG, "rope theta must be positive");
  return SCD_OK;
}

static scd_status_t check_layer_ranks(const scd_model_desc_t* m, const scd_layer_desc_t* l, int i) {
  if (l->kind == SCD_REUSE) {
    if (l->r_k < 1 || l->r_v < 1) return fail(SCD_E_SHAPE, "layer %d: REUSE ranks must be positive", i);
  } else if (l->kind == SCD_PATCH) {
    if (l->r_h < 1) return fail(SCD_E_SHAPE, "layer %d: r_h must be positive", i);
  } else {
    return fail(SCD_E_ARG, "layer %d: kind %d", i, l->kind);
  }
  // 16-byte row pitches of the code segments (TMA) on the tensor-core path
  if (m->state_dtype == SCD_BF16) {
    int q = m->code_dtype == SCD_E4M3_ROWSCALE ? 16 : 8;
    int ranks[3] = {l->kind == SCD_REUSE ? l->r_k : 0, l->kind == SCD_REUSE ? l->r_v : 0,
                    l->kind == SCD_PATCH ? l->r_h : 0};
    for (int r : ranks)
      if (r % q) return fail(SCD_E_UNSUPPORTED, "layer %d: rank %d not a multiple of %d on the bf16 path", i, r, q);
  }
  return SCD_OK;
}

// ---------------------------------------------------------------------------------
// code-buffer layout: segments in the order all-K, all-V, all-H (layers ascending), each
// [T, r] row-major padded to 128 B; e4m3 row scales follow in the same order.
// ---------------------------------------------------------------------------------
struct Layout {
  size_t code_bytes = 0, payload = 0;
  size_t off[SCD_MAX_LAYERS * 3], soff[SCD_MAX_LAYERS * 3];
  int32_t rank[SCD_MAX_LAYERS * 3];
};

static void compute_layout(const scd_model_desc_t* m, const int32_t* kind, const int32_t* r_k, const int32_t* r_v,
                           const int32_t* r_h, int32_t T, Layout* lay) {
  const size_t cb = code_elem_bytes(m->code_dtype);
  const bool sc = m->code_dtype == SCD_E4M3_ROWSCALE;
  size_t at = 0;
  for (int i = 0; i < m->n_layers * 3; ++i) { lay->off[i] = lay->soff[i] = (size_t)-1; lay->rank[i] = 0; }
  lay->payload = 0;
  for (int br = 0; br < 3; ++br)
    for (int l = 0; l < m->n_layers; ++l) {
      int r = 0;
      if (kind[l] == SCD_REUSE && br == SCD_BRANCH_K) r = r_k[l];
      if (kind[l] == SCD_REUSE && br == SCD_BRANCH_V) r = r_v[l];
      if (kind[l] == SCD_PATCH && br == SCD_BRANCH_H) r = r_h[l];
      if (!r) continue;
      lay->off[l * 3 + br] = at;
      lay->rank[l * 3 + br] = r;
      at += align_up((size_t)T * r * cb, 128);
      lay->payload += (size_t)T * (r * cb + (sc ? 4 : 0));
    }
  if (sc)
    for (int br = 0; br < 3; ++br)
      for (int l = 0; l < m->n_layers; ++l)
        if (lay->rank[l * 3 + br]) {
          lay->soff[l * 3 + br] = at;
          at += align_up((size_t)T * 4, 128);
        }
  lay->code_bytes = at;
}

static void plan_layout(const scd_plan_t* p, int32_t T, Layout* lay) {
  compute_layout(&p->model, p->kind.data(), p->r_k.data(), p->r_v.data(), p->r_h.data(), T, lay);
}

// scd_patch workspace: `group` slices of {a [T, d_a], u [T, d], sum-of-squares partials}.  The tensor-core path runs
// each GEMM stage of up to `group` PATCH layers as one multi-segment launch (fewer launches, fuller last wave); the
// group is as many layers as fit in 2 GiB of workspace (at least 1, at most 16).
struct PatchWs {
  size_t act_stride = 0, u_stride = 0, ss_stride = 0;
  int group = 1;
  size_t total() const { return (size_t)group * (act_stride + u_stride + ss_stride); }
};
static PatchWs patch_ws(const scd_plan_t* p, int32_t T) {
  PatchWs w;
  if (p->patches.empty() || T <= 0) { w.group = 0; return w; }
  const size_t es = state_elem_bytes(p->model.state_dtype);
  int d_a = 0;
  for (auto& pp : p->patches) d_a = pp.d_a > d_a ? pp.d_a : d_a;
  const int d = p->model.d_model;
  w.act_stride = align_up((size_t)T * d_a * es, 128);
  w.u_stride = align_up((size_t)T * d * es, 128);
  w.ss_stride = align_up((size_t)(2 * ((d + 127) / 128)) * T * 4, 128);   // sum-of-squares partials
  const size_t per_layer = w.act_stride + w.u_stride + w.ss_stride;
  size_t g = p->use_tc ? ((size_t)2 << 30) / per_layer : 1;
  g = g < 1 ? 1 : g;
  g = g > 16 ? 16 : g;
  w.group = (int)(g > p->patches.size() ? p->patches.size() : g);
  return w;
}
static size_t patch_workspace(const scd_plan_t* p, int32_t T) { return patch_ws(p, T).total(); }

// ---------------------------------------------------------------------------------
// batch validation shared by the hot calls
// ---------------------------------------------------------------------------------
static scd_status_t check_batch(const scd_plan_t* p, const scd_batch_t* b, bool need_pages) {
  if (!p) return fail(SCD_E_ARG, "plan is NULL");
  if (!b) return fail(SCD_E_ARG, "batch is NULL");
  if (b->n_seqs < 0 || b->total_tokens < 0) return fail(SCD_E_ARG, "negative n_seqs / total_tokens");
  if (b->n_seqs == 0 || b->total_tokens == 0) return SCD_OK;
  if (!b->cu_seqlens) return fail(SCD_E_ARG, "cu_seqlens is NULL");
  if (need_pages && !b->page_table) return fail(SCD_E_ARG, "page_table is NULL");
  if (b->max_seqlen < 1 || b->max_seqlen > b->total_tokens) return fail(SCD_E_ARG, "max_seqlen out of range");
  if (need_pages) {
    int bs = p->model.block_size;
    if (b->max_pages_per_seq < (b->max_seqlen + bs - 1) / bs)
      return fail(SCD_E_SHAPE, "max_pages_per_seq %d too small for max_seqlen %d", b->max_pages_per_seq,
                  b->max_seqlen);
  }
  if (b->max_pos_offset < 0) return fail(SCD_E_ARG, "max_pos_offset negative");
  if ((int64_t)b->max_seqlen + b->max_pos_offset > p->model.max_position)
    return fail(SCD_E_ARG, "position ids up to %lld exceed max_position %d",
                (long long)b->max_seqlen + b->max_pos_offset - 1, p->model.max_position);
  return SCD_OK;
}

static BatchDev batch_dev(const scd_plan_t* p, const scd_batch_t* b, bool pages, int n_blocks = 0) {
  BatchDev d;
  d.cu_seqlens = b->cu_seqlens;
  d.page_table = pages ? b->page_table : nullptr;
  d.pos_offset = b->pos_offset;
  d.n_seqs = b->n_seqs;
  d.total_tokens = b->total_tokens;
  d.max_pages_per_seq = b->max_pages_per_seq;
  d.block_size = p->model.block_size;
  d.n_blocks = n_blocks;
  return d;
}

static RopeDev rope_dev(const scd_plan_t* p, bool producer) {
  RopeDev r;
  r.table = producer ? p->rope_prod : p->rope_cons;
  r.head_dim = p->model.head_dim;
  r.style = p->model.rope_style;
  r.max_position = p->model.max_position;
  return r;
}

static bool aligned(const void* p, size_t a) { return ((uintptr_t)p % a) == 0; }

// ---------------------------------------------------------------------------------
// plan construction
// ---------------------------------------------------------------------------------
// fp32 epilogue vectors are read with 16-byte loads up to one tile (256 columns) past N
static const size_t kVecPad = 256 * sizeof(float);

// zero-filled on the plan's stream: the repack kernels that write the same buffers are enqueued on that stream too, so
// the fill is ordered before them even when it is a non-blocking stream (a legacy-stream cudaMemset would not be)
template <typename T>
static scd_status_t dev_alloc(scd_plan_t* p, T** out, size_t bytes, cudaStream_t s) {
  void* ptr = nullptr;
  cudaError_t e = cudaMalloc(&ptr, bytes ? bytes : 16);
  if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? SCD_E_NOMEM : SCD_E_CUDA, "cudaMalloc(%zu): %s",
                                    bytes, cudaGetErrorString(e));
  p->allocs.push_back(ptr);
  e = cudaMemsetAsync(ptr, 0, bytes ? bytes : 16, s);
  if (e != cudaSuccess) return fail(SCD_E_CUDA, "cudaMemsetAsync(%zu): %s", bytes, cudaGetErrorString(e));
  *out = (T*)ptr;
  return SCD_OK;
}

static scd_status_t build_plan(scd_plan_t* p, const scd_layer_desc_t* layers, cudaStream_t s) {
  const scd_model_desc_t& m = p->model;
  const int sd = m.state_dtype;
  const size_t es = state_elem_bytes(sd);
  const int D = p->D, d = m.d_model;
  scd_status_t st;

  // RoPE tables (fp64 angles -> fp32 cos/sin)
  const size_t tbytes = (size_t)m.max_position * (m.head_dim / 2) * sizeof(float2);
  if ((st = dev_alloc(p, &p->rope_cons, tbytes, s)) != SCD_OK) return st;
  SCD_CUDA(prep_rope_table(p->rope_cons, m.max_position, m.head_dim, m.rope_theta_consumer, s));
  if (m.rope_theta_producer == m.rope_theta_consumer) {
    p->rope_prod = p->rope_cons;
  } else {
    if ((st = dev_alloc(p, &p->rope_prod, tbytes, s)) != SCD_OK) return st;
    SCD_CUDA(prep_rope_table(p->rope_prod, m.max_position, m.head_dim, m.rope_theta_producer, s));
  }

  // code segments in buffer order
  p->seg_of.assign((size_t)m.n_layers * 3, -1);
  for (int br = 0; br < 3; ++br)
    for (int l = 0; l < m.n_layers; ++l) {
      const scd_layer_desc_t& L = layers[l];
      int r = 0;
      const void *enc = nullptr, *dec = nullptr;
      const float *mu_s = nullptr, *mu_d = nullptr;
      int width = D;
      if (L.kind == SCD_REUSE && br == SCD_BRANCH_K) { r = L.r_k; enc = L.enc_k; dec = L.dec_k; mu_s = L.mean_src_k; mu_d = L.mean_dst_k; }
      if (L.kind == SCD_REUSE && br == SCD_BRANCH_V) { r = L.r_v; enc = L.enc_v; dec = L.dec_v; mu_s = L.mean_src_v; mu_d = L.mean_dst_v; }
      if (L.kind == SCD_PATCH && br == SCD_BRANCH_H) { r = L.r_h; enc = L.enc_h; mu_s = L.mean_src_h; width = d; }
      if (!r) continue;
      if (!enc) return fail(SCD_E_ARG, "layer %d branch %d: encoder is NULL", l, br);
      if (br != SCD_BRANCH_H && !dec) return fail(SCD_E_ARG, "layer %d branch %d: decoder is NULL", l, br);
      SegPlan sp{};
      sp.layer = l; sp.branch = br; sp.rank = r; sp.width = width; sp.seg_index = (int)p->segs.size();
      if ((st = dev_alloc(p, &sp.enc_t, (size_t)r * width * es, s)) != SCD_OK) return st;
      SCD_CUDA(prep_transpose(enc, sp.enc_t, width, r, sd, s));            // [width, r] -> [r, width]
      if ((st = dev_alloc(p, &sp.enc_c, (size_t)r * 4 + kVecPad, s)) != SCD_OK) return st;
      SCD_CUDA(prep_mean_proj(mu_s, enc, sp.enc_c, width, r, sd, s));
      if (mu_s) {
        if ((st = dev_alloc(p, &sp.mean_src, (size_t)width * 4, s)) != SCD_OK) return st;
        SCD_CUDA(prep_copy_f32(mu_s, sp.mean_src, width, s));
      }
      if (dec) {
        if ((st = dev_alloc(p, &sp.dec_t, (size_t)D * r * es, s)) != SCD_OK) return st;
        SCD_CUDA(prep_transpose(dec, sp.dec_t, r, D, sd, s));              // [r, D] -> [D, r]
        if ((st = dev_alloc(p, &sp.mean_dst, (size_t)D * 4 + kVecPad, s)) != SCD_OK) return st;
        SCD_CUDA(prep_copy_f32(mu_d, sp.mean_dst, D, s));
      }
      p->seg_of[(size_t)l * 3 + br] = sp.seg_index;
      p->segs.push_back(sp);
    }

  // PATCH layers: aligner + gamma-folded [W_k ; W_v]
  for (int l = 0; l < m.n_layers; ++l) {
    const scd_layer_desc_t& L = layers[l];
    if (L.kind != SCD_PATCH) continue;
    if (L.d_aligner < 1) return fail(SCD_E_SHAPE, "layer %d: d_aligner must be positive", l);
    if (!L.w1 || !L.w2 || !L.w_k || !L.w_v) return fail(SCD_E_ARG, "layer %d: PATCH weight is NULL", l);
    if (m.patch_norm == SCD_NORM_RMS && !L.norm_gamma) return fail(SCD_E_ARG, "layer %d: norm_gamma is NULL", l);
    PatchPlan pp{};
    pp.layer = l; pp.r_h = L.r_h; pp.d_a = L.d_aligner; pp.h_seg = p->seg_of[(size_t)l * 3 + SCD_BRANCH_H];
    if ((st = dev_alloc(p, &pp.w1_t, (size_t)pp.d_a * pp.r_h * es, s)) != SCD_OK) return st;
    SCD_CUDA(prep_transpose(L.w1, pp.w1_t, pp.r_h, pp.d_a, sd, s));        // [r_h, d_a] -> [d_a, r_h]
    if ((st = dev_alloc(p, &pp.b1, (size_t)pp.d_a * 4 + kVecPad, s)) != SCD_OK) return st;
    SCD_CUDA(prep_to_f32(L.b1, pp.b1, pp.d_a, sd, s));
    if ((st = dev_alloc(p, &pp.w2_t, (size_t)d * pp.d_a * es, s)) != SCD_OK) return st;
    SCD_CUDA(prep_transpose(L.w2, pp.w2_t, pp.d_a, d, sd, s));             // [d_a, d] -> [d, d_a]
    if ((st = dev_alloc(p, &pp.b2, (size_t)d * 4 + kVecPad, s)) != SCD_OK) return st;
    SCD_CUDA(prep_to_f32(L.b2, pp.b2, d, sd, s));
    if ((st = dev_alloc(p, &pp.wkv, (size_t)2 * D * d * es, s)) != SCD_OK) return st;
    const void* gamma = m.patch_norm == SCD_NORM_RMS ? L.norm_gamma : nullptr;
    SCD_CUDA(prep_fold_gamma(L.w_k, gamma, pp.wkv, D, d, sd, s));
    SCD_CUDA(prep_fold_gamma(L.w_v, gamma, (char*)pp.wkv + (size_t)D * d * es, D, d, sd, s));
    if ((st = dev_alloc(p, &pp.bkv, (size_t)2 * D * 4 + kVecPad, s)) != SCD_OK) return st;
    SCD_CUDA(prep_to_f32(L.b_k, pp.bkv, D, sd, s));
    SCD_CUDA(prep_to_f32(L.b_v, pp.bkv + D, D, sd, s));
    p->patches.push_back(pp);
  }

  if (p->use_tc) {
    if ((st = tc_plan_init(p, s)) != SCD_OK) return st;
  }
  return SCD_OK;
}

// I_H (x) W for the REUSE artifacts of every layer; `temps` owns the device buffers until the plan has repacked them
scd_status_t expand_per_head(const scd_model_desc_t* m, const scd_layer_desc_t* layers, cudaStream_t s,
                             std::vector<scd_layer_desc_t>& eff, std::vector<void*>& temps) {
  const int H = m->n_kv_heads, dh = m->head_dim;
  const size_t es = state_elem_bytes(m->state_dtype);
  eff.assign(layers, layers + m->n_layers);
  auto alloc = [&](size_t bytes) -> void* {
    void* d = nullptr;
    if (cudaMalloc(&d, bytes) != cudaSuccess) return nullptr;
    temps.push_back(d);
    return d;
  };
  for (int i = 0; i < m->n_layers; ++i) {
    scd_layer_desc_t& l = eff[i];
    if (l.kind != SCD_REUSE) continue;
    if (l.r_k < 1 || l.r_v < 1) return fail(SCD_E_SHAPE, "layer %d: REUSE ranks must be positive", i);
    if (!l.enc_k || !l.enc_v || !l.dec_k || !l.dec_v) return fail(SCD_E_ARG, "layer %d: REUSE artifacts missing", i);
    struct { const void** w; int rows, cols; } mats[4] = {
        {&l.enc_k, dh, l.r_k}, {&l.enc_v, dh, l.r_v}, {&l.dec_k, l.r_k, dh}, {&l.dec_v, l.r_v, dh}};
    for (auto& mt : mats) {
      void* d = alloc((size_t)H * mt.rows * H * mt.cols * es);
      if (!d) return fail(SCD_E_NOMEM, "cudaMalloc(per-head expansion)");
      SCD_CUDA(prep_block_diag(*mt.w, d, mt.rows, mt.cols, H, m->state_dtype, s));
      *mt.w = d;
    }
    const float** means[4] = {&l.mean_src_k, &l.mean_src_v, &l.mean_dst_k, &l.mean_dst_v};
    for (auto mp : means) {
      if (!*mp) continue;
      float* d = (float*)alloc((size_t)H * dh * sizeof(float));
      if (!d) return fail(SCD_E_NOMEM, "cudaMalloc(per-head expansion)");
      SCD_CUDA(prep_tile_f32(*mp, d, dh, H, s));
      *mp = d;
    }
    l.r_k *= H;
    l.r_v *= H;
  }
  return SCD_OK;
}

}  // namespace scd

using namespace scd;

// =================================================================================
// C ABI
// =================================================================================
extern "C" {

const char* scd_last_error(void) { return g_err; }
int32_t scd_last_launch_count(void) { return g_launches; }
int32_t scd_struct_size(int32_t which) {
  switch (which) {
    case 0: return (int32_t)sizeof(scd_model_desc_t);
    case 1: return (int32_t)sizeof(scd_layer_desc_t);
    case 2: return (int32_t)sizeof(scd_batch_t);
    case 3: return (int32_t)sizeof(scd_src_t);
    case 4: return (int32_t)sizeof(scd_paged_kv_t);
    case 5: return (int32_t)sizeof(scd_int4_desc_t);
    case 6: return (int32_t)sizeof(scd_fit_desc_t);
    default: return -1;
  }
}
const char* scd_version(void) { return "scd-b200 0.1 (sm_100a)"; }

scd_status_t scd_profile_enable(int32_t on) {
  g_prof_on = on != 0;
  return SCD_OK;
}
int32_t scd_profile_fetch(float* ms, int32_t* kernel_id, int32_t max) {
  if (!g_prof) return 0;
  int32_t n = (int32_t)g_prof->size();
  for (int32_t i = 0; i < n; ++i) {
    ProfRec& r = (*g_prof)[i];
    float t = 0.0f;
    cudaEventSynchronize(r.b);
    cudaEventElapsedTime(&t, r.a, r.b);
    if (i < max) {
      if (ms) ms[i] = t;
      if (kernel_id) kernel_id[i] = r.id;
    }
    cudaEventDestroy(r.a);
    cudaEventDestroy(r.b);
  }
  g_prof->clear();
  return n;
}

scd_status_t scd_code_layout(const scd_model_desc_t* model, const scd_layer_desc_t* layers, int32_t total_tokens,
                             int32_t layer, int32_t branch, size_t* offset, size_t* scale_offset, int32_t* rank,
                             size_t* code_bytes, size_t* payload_bytes) {
  scd_status_t st = check_model(model);
  if (st != SCD_OK) return st;
  if (!layers) return fail(SCD_E_ARG, "layers is NULL");
  if (total_tokens < 0) return fail(SCD_E_ARG, "total_tokens negative");
  int32_t kind[SCD_MAX_LAYERS], rk[SCD_MAX_LAYERS], rv[SCD_MAX_LAYERS], rh[SCD_MAX_LAYERS];
  const int hm = model->reuse_per_head ? model->n_kv_heads : 1;     // per-head reading: H * r codes per token
  for (int i = 0; i < model->n_layers; ++i) {
    scd_layer_desc_t le = layers[i];
    le.r_k *= hm; le.r_v *= hm;
    if ((st = check_layer_ranks(model, &le, i)) != SCD_OK) return st;
    kind[i] = le.kind; rk[i] = le.r_k; rv[i] = le.r_v; rh[i] = le.r_h;
  }
  Layout lay;
  compute_layout(model, kind, rk, rv, rh, total_tokens, &lay);
  if (code_bytes) *code_bytes = lay.code_bytes;
  if (payload_bytes) *payload_bytes = lay.payload;
  if (layer >= 0) {
    if (layer >= model->n_layers || branch < 0 || branch > 2) return fail(SCD_E_ARG, "layer / branch out of range");
    if (!lay.rank[layer * 3 + branch])
      return fail(SCD_E_ARG, "layer %d has no branch %d (REUSE: K, V; PATCH: H)", layer, branch);
    if (offset) *offset = lay.off[layer * 3 + branch];
    if (scale_offset) *scale_offset = lay.soff[layer * 3 + branch];
    if (rank) *rank = lay.rank[layer * 3 + branch];
  }
  return SCD_OK;
}

scd_status_t scd_plan(const scd_model_desc_t* model, const scd_layer_desc_t* layers, void* stream,
                      scd_plan_t** out) {
  if (out) *out = nullptr;
  if (!out) return fail(SCD_E_ARG, "out is NULL");
  scd_status_t st = check_model(model);
  if (st != SCD_OK) return st;
  if (!layers) return fail(SCD_E_ARG, "layers is NULL");
  // Per-head reading: the shared d_h x r map is expanded once, here, to the
  // block-diagonal per-layer operand I_H (x) W (means tiled over heads); everything below then sees a per-layer
  // plan of rank H * r, and the decode kernel skips the zero blocks (head_rank_k / head_rank_v).
  std::vector<scd_layer_desc_t> eff;
  std::vector<void*> temps;
  struct TempGuard {
    std::vector<void*>& t;
    ~TempGuard() { for (void* a : t) cudaFree(a); }
  } guard{temps};
  const scd_layer_desc_t* user_layers = layers;
  if (model->reuse_per_head) {
    if ((st = expand_per_head(model, layers, (cudaStream_t)stream, eff, temps)) != SCD_OK) return st;
    layers = eff.data();
  }
  for (int i = 0; i < model->n_layers; ++i)
    if ((st = check_layer_ranks(model, &layers[i], i)) != SCD_OK) return st;
  if (model->state_dtype == SCD_F32 && model->code_dtype != SCD_F32)
    return fail(SCD_E_UNSUPPORTED, "fp32 states require fp32 codes");
  if (model->state_dtype == SCD_BF16 && model->code_dtype == SCD_F32)
    return fail(SCD_E_UNSUPPORTED, "bf16 states require bf16 or e4m3 codes");

  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return fail(SCD_E_CUDA, "no CUDA device: %s", cudaGetErrorString(cudaGetLastError()));

  scd_plan_t* p = new (std::nothrow) scd_plan_t();
  if (!p) return fail(SCD_E_NOMEM, "host allocation failed");
  p->model = *model;
  p->D = model->n_kv_heads * model->head_dim;
  p->sm_count = sms;
  p->device = dev;
  if (dev < 0 || dev >= SCD_MAX_DEVICES) { delete p; return fail(SCD_E_UNSUPPORTED, "device ordinal %d >= %d", dev, SCD_MAX_DEVICES); }
  for (int i = 0; i < model->n_layers; ++i) {
    p->kind.push_back(layers[i].kind);
    p->r_k.push_back(layers[i].kind == SCD_REUSE ? layers[i].r_k : 0);
    p->r_v.push_back(layers[i].kind == SCD_REUSE ? layers[i].r_v : 0);
    p->r_h.push_back(layers[i].kind == SCD_PATCH ? layers[i].r_h : 0);
    p->d_a.push_back(layers[i].kind == SCD_PATCH ? layers[i].d_aligner : 0);
    const bool ph = model->reuse_per_head && layers[i].kind == SCD_REUSE;
    p->head_rank_k.push_back(ph ? user_layers[i].r_k : 0);
    p->head_rank_v.push_back(ph ? user_layers[i].r_v : 0);
  }
  p->use_tc = model->state_dtype == SCD_BF16;
  if (p->use_tc && (st = tc_supported(p, layers)) != SCD_OK) { scd_plan_destroy(p); return st; }

  st = build_plan(p, layers, (cudaStream_t)stream);
  if (st != SCD_OK) { scd_plan_destroy(p); return st; }
  if (!temps.empty() && cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) {   // the repacks read the temporaries
    scd_plan_destroy(p);
    return fail(SCD_E_CUDA, "plan: %s", cudaGetErrorString(cudaGetLastError()));
  }
  *out = p;
  return SCD_OK;
}

scd_status_t scd_plan_destroy(scd_plan_t* plan) {
  if (!plan) return SCD_OK;
  for (void* a : plan->allocs) cudaFree(a);
  delete plan;
  return SCD_OK;
}

scd_status_t scd_plan_query(const scd_plan_t* plan, int32_t total_tokens, size_t* code_bytes,
                            size_t* patch_workspace_bytes, size_t* payload_bytes) {
  if (!plan) return fail(SCD_E_ARG, "plan is NULL");
  if (total_tokens < 0) return fail(SCD_E_ARG, "total_tokens negative");
  Layout lay;
  plan_layout(plan, total_tokens, &lay);
  if (code_bytes) *code_bytes = lay.code_bytes;
  if (payload_bytes) *payload_bytes = lay.payload;
  if (patch_workspace_bytes) *patch_workspace_bytes = patch_workspace(plan, total_tokens);
  return SCD_OK;
}

scd_status_t scd_plan_code_segment(const scd_plan_t* plan, int32_t layer, int32_t branch, int32_t total_tokens,
                                   size_t* offset, size_t* scale_offset, int32_t* rank) {
  if (!plan) return fail(SCD_E_ARG, "plan is NULL");
  if (layer < 0 || layer >= plan->model.n_layers || branch < 0 || branch > 2 || total_tokens < 0)
    return fail(SCD_E_ARG, "layer / branch / total_tokens out of range");
  Layout lay;
  plan_layout(plan, total_tokens, &lay);
  if (!lay.rank[layer * 3 + branch])
    return fail(SCD_E_ARG, "layer %d has no branch %d (REUSE: K, V; PATCH: H)", layer, branch);
  if (offset) *offset = lay.off[layer * 3 + branch];
  if (scale_offset) *scale_offset = lay.soff[layer * 3 + branch];
  if (rank) *rank = lay.rank[layer * 3 + branch];
  return SCD_OK;
}

// ---------------------------------------------------------------------------------
// scd_encode  (Alg. 1 producer half)
// ---------------------------------------------------------------------------------
scd_status_t scd_encode(const scd_plan_t* plan, const scd_batch_t* batch, const scd_src_t* src, void* codes,
                        void* stream) {
  g_launches = 0;
  scd_status_t st = check_batch(plan, batch, false);
  if (st != SCD_OK) return st;
  if (batch->n_seqs == 0 || batch->total_tokens == 0) return SCD_OK;
  if (!src || !codes) return fail(SCD_E_ARG, "src / codes is NULL");
  if (!aligned(codes, 128)) return fail(SCD_E_ALIGN, "codes must be 128-byte aligned");
  const scd_model_desc_t& m = plan->model;
  const int T = batch->total_tokens;
  const bool has_reuse = plan->segs.size() > plan->patches.size();
  if (has_reuse && (!src->k || !src->v)) return fail(SCD_E_ARG, "src->k / src->v is NULL");
  if (!plan->patches.empty() && !src->h) return fail(SCD_E_ARG, "src->h is NULL");
  if (has_reuse && (src->kv_head_stride < m.head_dim || src->kv_token_stride < (int64_t)m.n_kv_heads * m.head_dim))
    return fail(SCD_E_SHAPE, "kv strides smaller than the tensor");
  if (!plan->patches.empty() && src->h_token_stride < m.d_model) return fail(SCD_E_SHAPE, "h_token_stride < d_model");
  if (src->page_table && has_reuse) {
    if (!plan->use_tc) return fail(SCD_E_UNSUPPORTED, "paged producer source: bf16 states only");
    if (src->kv_head_stride != m.head_dim) return fail(SCD_E_UNSUPPORTED, "paged producer source needs dense heads");
    if (src->n_blocks < 1 || src->max_pages_per_seq < 1) return fail(SCD_E_ARG, "paged producer source: n_blocks / max_pages_per_seq");
    if ((int64_t)src->max_pages_per_seq * m.block_size < batch->max_seqlen)
      return fail(SCD_E_SHAPE, "producer page table too narrow for max_seqlen");
  }
  for (const SegPlan& sp : plan->segs) {
    if (!layer_in_window(sp.layer)) continue;
    const void* a = sp.branch == SCD_BRANCH_K ? src->k[sp.layer] : sp.branch == SCD_BRANCH_V ? src->v[sp.layer] : src->h[sp.layer];
    if (!a) return fail(SCD_E_ARG, "source state of layer %d branch %d is NULL", sp.layer, sp.branch);
    if (!aligned(a, 16)) return fail(SCD_E_ALIGN, "source state of layer %d not 16-byte aligned", sp.layer);
  }
  Layout lay;
  plan_layout(plan, T, &lay);

  if (plan->use_tc) return tc_encode(plan, batch, src, codes, lay.off, lay.soff, (cudaStream_t)stream);

  BatchDev bd = batch_dev(plan, batch, false);
  RopeDev rd = rope_dev(plan, true);
  for (const SegPlan& sp : plan->segs) {
    if (!layer_in_window(sp.layer)) continue;
    GemmSeg g{};
    const int key = sp.layer * 3 + sp.branch;
    if (sp.branch == SCD_BRANCH_H) {
      g.a = src->h[sp.layer]; g.lda = src->h_token_stride; g.a_head_stride = 0;
    } else {
      g.a = sp.branch == SCD_BRANCH_K ? src->k[sp.layer] : src->v[sp.layer];
      g.lda = src->kv_token_stride;
      g.a_head_stride = src->kv_head_stride == m.head_dim ? 0 : src->kv_head_stride;
    }
    g.a_sub = sp.mean_src;
    g.bt = sp.enc_t;
    g.col_vec = nullptr;
    g.out0 = (char*)codes + lay.off[key];
    g.aux = m.code_dtype == SCD_E4M3_ROWSCALE ? (float*)((char*)codes + lay.soff[key]) : nullptr;
    g.M = T; g.N = sp.rank; g.K = sp.width;
    int a_mode = (sp.branch == SCD_BRANCH_K && m.k_is_roped) ? A_DEROPE : A_PLAIN;
    SCD_CUDA(simt_gemm(g, EPI_CODES, a_mode, m.state_dtype, m.code_dtype, bd, rd, (cudaStream_t)stream));
  }
  return SCD_OK;
}

// ---------------------------------------------------------------------------------
// scd_reuse_decode  (Alg. 1 consumer half; Eq. 9; RoPE :152)
// ---------------------------------------------------------------------------------
static scd_status_t check_pools(const scd_plan_t* plan, const scd_paged_kv_t* kv, int want_kind) {
  if (!kv || !kv->k_pool || !kv->v_pool) return fail(SCD_E_ARG, "kv pools are NULL");
  if (kv->n_blocks < 1) return fail(SCD_E_ARG, "n_blocks must be positive");
  for (int l = 0; l < plan->model.n_layers; ++l) {
    if (plan->kind[l] != want_kind || !layer_in_window(l)) continue;
    if (!kv->k_pool[l] || !kv->v_pool[l]) return fail(SCD_E_ARG, "pool of layer %d is NULL", l);
    if (!aligned(kv->k_pool[l], 16) || !aligned(kv->v_pool[l], 16))
      return fail(SCD_E_ALIGN, "pool of layer %d not 16-byte aligned", l);
    if (kv->pool_e4m3 && (!kv->k_scale || !kv->v_scale || !kv->k_scale[l] || !kv->v_scale[l]))
      return fail(SCD_E_ARG, "fp8 pools: scale array of layer %d is NULL", l);
  }
  if (kv->pool_e4m3) {
    const scd_model_desc_t& m = plan->model;
    if (!plan->use_tc || m.head_dim != 128 || m.rope_style != SCD_ROPE_HALF)
      return fail(SCD_E_UNSUPPORTED, "fp8 pools need bf16 states, head_dim 128 and HALF RoPE");
  }
  return SCD_OK;
}

scd_status_t scd_reuse_decode(const scd_plan_t* plan, const scd_batch_t* batch, const void* codes,
                              const scd_paged_kv_t* kv, void* stream) {
  g_launches = 0;
  scd_status_t st = check_batch(plan, batch, true);
  if (st != SCD_OK) return st;
  if (batch->n_seqs == 0 || batch->total_tokens == 0) return SCD_OK;
  if (!codes) return fail(SCD_E_ARG, "codes is NULL");
  if (!aligned(codes, 128)) return fail(SCD_E_ALIGN, "codes must be 128-byte aligned");
  if ((st = check_pools(plan, kv, SCD_REUSE)) != SCD_OK) return st;
  const scd_model_desc_t& m = plan->model;
  const int T = batch->total_tokens;
  Layout lay;
  plan_layout(plan, T, &lay);

  if (plan->use_tc) return tc_reuse_decode(plan, batch, codes, kv, lay.off, lay.soff, (cudaStream_t)stream);

  BatchDev bd = batch_dev(plan, batch, true, kv->n_blocks);
  RopeDev rd = rope_dev(plan, false);
  for (const SegPlan& sp : plan->segs) {
    if (sp.branch == SCD_BRANCH_H || !layer_in_window(sp.layer)) continue;
    const int key = sp.layer * 3 + sp.branch;
    GemmSeg g{};
    g.a = (const char*)codes + lay.off[key]; g.lda = sp.rank;
    g.a_scale = m.code_dtype == SCD_E4M3_ROWSCALE ? (const float*)((const char*)codes + lay.soff[key]) : nullptr;
    g.bt = sp.dec_t;
    g.col_vec = sp.mean_dst;
    g.out0 = sp.branch == SCD_BRANCH_K ? kv->k_pool[sp.layer] : kv->v_pool[sp.layer];
    g.M = T; g.N = plan->D; g.K = sp.rank;
    g.split = g.N; g.pool_width = plan->D;
    g.rope_cols = (sp.branch == SCD_BRANCH_K && m.rope_on_reuse_k) ? plan->D : 0;
    SCD_CUDA(simt_gemm(g, EPI_KV, A_CODES, m.state_dtype, m.code_dtype, bd, rd, (cudaStream_t)stream));
  }
  return SCD_OK;
}

// ---------------------------------------------------------------------------------
// scd_patch  (Eq. 11, Eq. 12a/b :190-193, cache assembly :612-616)
// ---------------------------------------------------------------------------------
scd_status_t scd_patch(const scd_plan_t* plan, const scd_batch_t* batch, const void* codes,
                       const scd_paged_kv_t* kv, void* workspace, size_t workspace_bytes, void* stream) {
  g_launches = 0;
  scd_status_t st = check_batch(plan, batch, true);
  if (st != SCD_OK) return st;
  if (batch->n_seqs == 0 || batch->total_tokens == 0 || plan->patches.empty()) return SCD_OK;
  if (!codes) return fail(SCD_E_ARG, "codes is NULL");
  if (!aligned(codes, 128)) return fail(SCD_E_ALIGN, "codes must be 128-byte aligned");
  if ((st = check_pools(plan, kv, SCD_PATCH)) != SCD_OK) return st;
  const scd_model_desc_t& m = plan->model;
  const int T = batch->total_tokens;
  // scd_plan_query reports the workspace for the preferred group of layers per launch; any workspace that holds at
  // least one layer's intermediates is accepted, and the group shrinks to what it holds
  PatchWs pw = patch_ws(plan, T);
  const size_t per_layer = pw.act_stride + pw.u_stride + pw.ss_stride;
  if (pw.group > 0 && (!workspace || workspace_bytes < per_layer))
    return fail(SCD_E_WORKSPACE, "scd_patch needs at least %zu workspace bytes (%zu preferred), got %zu", per_layer, pw.total(),
                workspace_bytes);
  if (pw.group > 0 && (size_t)pw.group * per_layer > workspace_bytes) pw.group = (int)(workspace_bytes / per_layer);
  if (!aligned(workspace, 128)) return fail(SCD_E_ALIGN, "workspace must be 128-byte aligned");
  Layout lay;
  plan_layout(plan, T, &lay);

  const size_t es = state_elem_bytes(m.state_dtype);
  int d_a_max = 0;
  for (auto& pp : plan->patches) d_a_max = pp.d_a > d_a_max ? pp.d_a : d_a_max;
  const int d = m.d_model, D = plan->D;
  char* ws_act = (char*)workspace;
  char* ws_u = ws_act + (size_t)pw.group * pw.act_stride;
  float* ws_ss = (float*)(ws_u + (size_t)pw.group * pw.u_stride);
  (void)es; (void)d_a_max;

  if (plan->use_tc)
    return tc_patch(plan, batch, codes, kv, ws_act, ws_u, ws_ss, pw.group, pw.act_stride, pw.u_stride, pw.ss_stride, lay.off,
                    lay.soff, (cudaStream_t)stream);

  BatchDev bd = batch_dev(plan, batch, true, kv->n_blocks);
  RopeDev rd = rope_dev(plan, false);
  const bool rms = m.patch_norm == SCD_NORM_RMS;
  for (const PatchPlan& pp : plan->patches) {
    if (!layer_in_window(pp.layer)) continue;
    const int key = pp.layer * 3 + SCD_BRANCH_H;
    GemmSeg g1{};
    g1.a = (const char*)codes + lay.off[key]; g1.lda = pp.r_h;
    g1.a_scale = m.code_dtype == SCD_E4M3_ROWSCALE ? (const float*)((const char*)codes + lay.soff[key]) : nullptr;
    g1.bt = pp.w1_t; g1.col_vec = pp.b1; g1.out0 = ws_act;
    g1.M = T; g1.N = pp.d_a; g1.K = pp.r_h; g1.act = m.patch_act;
    SCD_CUDA(simt_gemm(g1, EPI_ACT, A_CODES, m.state_dtype, m.code_dtype, bd, rd, (cudaStream_t)stream));
    GemmSeg g2{};
    g2.a = ws_act; g2.lda = pp.d_a; g2.bt = pp.w2_t; g2.col_vec = pp.b2; g2.out0 = ws_u;
    g2.aux = rms ? ws_ss : nullptr;
    g2.M = T; g2.N = d; g2.K = pp.d_a;
    SCD_CUDA(simt_gemm(g2, EPI_U, A_PLAIN, m.state_dtype, m.code_dtype, bd, rd, (cudaStream_t)stream));
    GemmSeg g3{};
    g3.a = ws_u; g3.lda = d; g3.bt = pp.wkv; g3.col_vec = pp.bkv;
    g3.out0 = kv->k_pool[pp.layer]; g3.out1 = kv->v_pool[pp.layer];
    g3.M = T; g3.N = 2 * D; g3.K = d; g3.split = D; g3.pool_width = D; g3.rope_cols = D;
    g3.rowscale_in = rms ? ws_ss : nullptr; g3.n_partials = (d + 127) / 128; g3.rms_eps = m.rms_eps; g3.rms_dim = d;
    SCD_CUDA(simt_gemm(g3, EPI_KV, A_PLAIN, m.state_dtype, m.code_dtype, bd, rd, (cudaStream_t)stream));
  }
  return SCD_OK;
}

// ---------------------------------------------------------------------------------
// layer-streamed variants: the same calls restricted to layers [layer_begin, layer_end), so
// that encode of later layers, transport of a layer's code segments (scd_plan_code_segment) and decode of earlier
// layers can overlap on different streams -- Eq. 3's three terms pipelined.  Segments and pools of
// layers outside the window are neither read, written nor validated.
// ---------------------------------------------------------------------------------
static scd_status_t check_window(const scd_plan_t* plan, int32_t b, int32_t e) {
  if (!plan) return fail(SCD_E_ARG, "plan is NULL");
  if (b < 0 || e < b || e > plan->model.n_layers) return fail(SCD_E_ARG, "layer window [%d, %d) outside [0, %d]", b, e, plan->model.n_layers);
  return SCD_OK;
}
scd_status_t scd_encode_layers(const scd_plan_t* plan, const scd_batch_t* batch, const scd_src_t* src, void* codes,
                               int32_t layer_begin, int32_t layer_end, void* stream) {
  scd_status_t st = check_window(plan, layer_begin, layer_end);
  if (st != SCD_OK) return st;
  LayerWindow w(layer_begin, layer_end);
  return scd_encode(plan, batch, src, codes, stream);
}
scd_status_t scd_reuse_decode_layers(const scd_plan_t* plan, const scd_batch_t* batch, const void* codes,
                                     const scd_paged_kv_t* kv, int32_t layer_begin, int32_t layer_end, void* stream) {
  scd_status_t st = check_window(plan, layer_begin, layer_end);
  if (st != SCD_OK) return st;
  LayerWindow w(layer_begin, layer_end);
  return scd_reuse_decode(plan, batch, codes, kv, stream);
}
scd_status_t scd_patch_layers(const scd_plan_t* plan, const scd_batch_t* batch, const void* codes, const scd_paged_kv_t* kv,
                              void* workspace, size_t workspace_bytes, int32_t layer_begin, int32_t layer_end, void* stream) {
  scd_status_t st = check_window(plan, layer_begin, layer_end);
  if (st != SCD_OK) return st;
  LayerWindow w(layer_begin, layer_end);
  return scd_patch(plan, batch, codes, kv, workspace, workspace_bytes, stream);
}

// ---------------------------------------------------------------------------------
// scd_patch_static: scd_patch with its intermediates in a static device array (no allocation, no caller workspace)
// ---------------------------------------------------------------------------------
}  // extern "C"  (the array and its address cache have internal linkage)

// In HOST code this name is a host-side stand-in, not a device address: it is only ever handed to
// cudaGetSymbolAddress below, never to a kernel.
static __device__ __align__(256) unsigned char g_patch_static_ws[SCD_PATCH_STATIC_WORKSPACE_BYTES];

// Device address of the array on `device`, looked up once per device with that device current.
static scd_status_t patch_static_ws(int device, void** out) {
  static std::atomic<void*> addr[scd::SCD_MAX_DEVICES];
  if (device < 0 || device >= scd::SCD_MAX_DEVICES) return scd::fail(SCD_E_UNSUPPORTED, "scd_patch_static: device ordinal %d", device);
  int cur = -1;
  cudaError_t e = cudaGetDevice(&cur);
  if (e != cudaSuccess) return scd::fail(SCD_E_CUDA, "scd_patch_static: cudaGetDevice: %s", cudaGetErrorString(e));
  if (cur != device)
    return scd::fail(SCD_E_ARG, "scd_patch_static: the plan lives on device %d but device %d is current", device, cur);
  void* ptr = addr[device].load(std::memory_order_acquire);
  if (!ptr) {
    e = cudaGetSymbolAddress(&ptr, g_patch_static_ws);
    if (e != cudaSuccess || !ptr)
      return scd::fail(SCD_E_CUDA, "scd_patch_static: cudaGetSymbolAddress(static workspace): %s", cudaGetErrorString(e));
    addr[device].store(ptr, std::memory_order_release);      // racing threads look up the same address
  }
  *out = ptr;
  return SCD_OK;
}

extern "C" scd_status_t scd_patch_static(const scd_plan_t* plan, const scd_batch_t* batch, const void* codes,
                                         const scd_paged_kv_t* kv, void* stream) {
  using namespace scd;
  reset_launch_count();
  scd_status_t st = check_batch(plan, batch, true);
  if (st != SCD_OK) return st;
  if (batch->n_seqs == 0 || batch->total_tokens == 0 || plan->patches.empty()) return SCD_OK;
  const PatchWs pw = patch_ws(plan, batch->total_tokens);
  const size_t per_layer = pw.act_stride + pw.u_stride + pw.ss_stride;
  if (per_layer > (size_t)SCD_PATCH_STATIC_WORKSPACE_BYTES)
    return fail(SCD_E_WORKSPACE,
                "scd_patch_static: one PATCH layer of %d tokens needs %zu bytes of intermediates, the static array holds %zu "
                "(SCD_PATCH_STATIC_WORKSPACE_BYTES); use scd_patch with a caller workspace",
                batch->total_tokens, per_layer, (size_t)SCD_PATCH_STATIC_WORKSPACE_BYTES);
  void* ws = nullptr;
  if ((st = patch_static_ws(plan->device, &ws)) != SCD_OK) return st;
  return scd_patch(plan, batch, codes, kv, ws, (size_t)SCD_PATCH_STATIC_WORKSPACE_BYTES, stream);
}
