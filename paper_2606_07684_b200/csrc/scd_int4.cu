// Group-wise INT4 KV codec: the paper's fastest transport baseline ("Quantized KV: transmits 4-bit quantized KV
// caches (group-wise INT4) and dequantizes on the consumer"; Table 4 :352-359) built as the same-box
// comparison codec of SURVEY 8(f) NEXT-3.  Definition: DESIGN.md section 2, U19 (oracle/int4_oracle.py restates it):
//
//   group = G consecutive channels of one token row (G in {32, 64, 128}, G | head_dim)
//   lo = min x, hi = max x;  s = bf16_rne((hi - lo) / 15) (1 if that is 0);  q = clamp(rint((x - lo) / s), 0, 15)
//   byte j = q[2j] | q[2j + 1] << 4;  metadata = bf16 s and bf16 lo per group;  x^ = bf16_rne(q * s + lo)
//
// Every decision is IEEE fp32 (div.rn, cvt.rni), so codes and dequantised values are bit-exact against the oracle.
// Both kernels are pure streams (read 2 B, write 0.5 + 4/G B per element, and the reverse): one 16-byte access per
// thread and element octet, many small CTAs (the write-only probe of this part prefers them to a persistent grid,
// profiles/r01_hbm_probe.md), evict-first stores, all tensors (layers x {K, V}) in one launch.
#include <algorithm>

#include "ptx.cuh"
#include "scd_device.cuh"

namespace scd {
namespace {

constexpr int Q4_THREADS = 256;
constexpr int Q4_ROWS = 16;          // token rows per CTA
constexpr int Q4_MAX_TENSORS = 384;  // pointer table travels as a kernel parameter (3 KB)

struct Q4Ptrs {
  const void* p[Q4_MAX_TENSORS];
};

struct Q4Layout {
  size_t tensor_stride, scale_off, zero_off;
};

__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

// ---- producer: quantise ----
template <int LANES>   // lanes per group = G / 8
__global__ void __launch_bounds__(Q4_THREADS) int4_quantize_kernel(const Q4Ptrs src, long long token_stride, int T, int width,
                                                                   uint8_t* __restrict__ out, Q4Layout lay) {
  const int ipr = width >> 3;                       // 8-element items per row
  const int row0 = blockIdx.x * Q4_ROWS;
  const int rows = min(Q4_ROWS, T - row0);
  const int n_items = rows * ipr;
  const __nv_bfloat16* x = (const __nv_bfloat16*)src.p[blockIdx.y];
  uint8_t* base = out + (size_t)blockIdx.y * lay.tensor_stride;
  uint32_t* qout = (uint32_t*)base;
  __nv_bfloat16* sout = (__nv_bfloat16*)(base + lay.scale_off);
  __nv_bfloat16* zout = (__nv_bfloat16*)(base + lay.zero_off);
  const int gpr = ipr / LANES;                      // groups per row
  const int lane = threadIdx.x & 31;
  for (int w0 = threadIdx.x - lane; w0 < n_items; w0 += Q4_THREADS * 4) {    // warp-uniform trip count (shuffles below)
    const int it0 = w0 + lane;
    uint4 v[4];
    int row[4], c8[4];
    bool ok[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int item = it0 + u * Q4_THREADS;
      ok[u] = item < n_items;
      row[u] = ok[u] ? item / ipr : 0;
      c8[u] = ok[u] ? item - row[u] * ipr : 0;
      v[u] = make_uint4(0u, 0u, 0u, 0u);
      if (ok[u]) v[u] = __ldcs(reinterpret_cast<const uint4*>(x + (size_t)(row0 + row[u]) * token_stride + c8[u] * 8));
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (w0 + u * Q4_THREADS >= n_items) break;                               // whole warp past the end
      const uint32_t w[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
      float f[8];
#pragma unroll
      for (int i = 0; i < 4; ++i) { f[2 * i] = bf16_lo(w[i]); f[2 * i + 1] = bf16_hi(w[i]); }
      float lo = f[0], hi = f[0];
#pragma unroll
      for (int i = 1; i < 8; ++i) { lo = fminf(lo, f[i]); hi = fmaxf(hi, f[i]); }
#pragma unroll
      for (int o = 1; o < LANES; o <<= 1) {
        lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, o));
      }
      float s = __bfloat162float(__float2bfloat16_rn(__fdiv_rn(__fsub_rn(hi, lo), 15.0f)));
      if (s == 0.0f) s = 1.0f;
      uint32_t packed = 0;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const float t = __fdiv_rn(__fsub_rn(f[i], lo), s);
        int q = __float2int_rn(t);
        q = q < 0 ? 0 : (q > 15 ? 15 : q);
        packed |= (uint32_t)q << (4 * i);
      }
      if (ok[u]) {
        const size_t r = (size_t)(row0 + row[u]);
        __stcs(qout + r * ipr + c8[u], packed);
        if ((c8[u] % LANES) == 0) {
          sout[r * gpr + c8[u] / LANES] = __float2bfloat16_rn(s);
          zout[r * gpr + c8[u] / LANES] = __float2bfloat16_rn(lo);
        }
      }
    }
  }
}

// ---- consumer: dequantise into the paged pool ----
template <int LANES>
__global__ void __launch_bounds__(Q4_THREADS) int4_dequantize_paged_kernel(const uint8_t* __restrict__ in, Q4Layout lay, const Q4Ptrs pools,
                                                                           BatchDev batch, int width) {
  __shared__ long long slots[Q4_ROWS];
  const int T = batch.total_tokens;
  const int ipr = width >> 3;
  const int row0 = blockIdx.x * Q4_ROWS;
  const int rows = min(Q4_ROWS, T - row0);
  if (threadIdx.x < Q4_ROWS) {
    long long slot = -1;
    int pos;
    if ((int)threadIdx.x < rows) row_to_pos_slot(batch, row0 + threadIdx.x, pos, slot);
    slots[threadIdx.x] = slot;
  }
  __syncthreads();
  const int n_items = rows * ipr;
  const uint8_t* base = in + (size_t)blockIdx.y * lay.tensor_stride;
  const uint32_t* qin = (const uint32_t*)base;
  const __nv_bfloat16* sin = (const __nv_bfloat16*)(base + lay.scale_off);
  const __nv_bfloat16* zin = (const __nv_bfloat16*)(base + lay.zero_off);
  __nv_bfloat16* pool = (__nv_bfloat16*)pools.p[blockIdx.y];
  const int gpr = ipr / LANES;
  for (int it0 = threadIdx.x; it0 < n_items; it0 += Q4_THREADS * 4) {
    uint32_t pk[4];
    float s[4], z[4];
    int row[4], c8[4];
    bool ok[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int item = it0 + u * Q4_THREADS;
      ok[u] = item < n_items;
      row[u] = ok[u] ? item / ipr : 0;
      c8[u] = ok[u] ? item - row[u] * ipr : 0;
      pk[u] = 0; s[u] = 0.f; z[u] = 0.f;
      if (ok[u]) {
        const size_t r = (size_t)(row0 + row[u]);
        pk[u] = __ldcs(qin + r * ipr + c8[u]);
        s[u] = __bfloat162float(__ldg(sin + r * gpr + c8[u] / LANES));
        z[u] = __bfloat162float(__ldg(zin + r * gpr + c8[u] / LANES));
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (!ok[u]) continue;
      const long long slot = slots[row[u]];
      if (slot < 0) continue;                        // page id outside the pool: the row is not written
      uint32_t o[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float a = fmaf((float)((pk[u] >> (8 * i)) & 15u), s[u], z[u]);
        const float b = fmaf((float)((pk[u] >> (8 * i + 4)) & 15u), s[u], z[u]);
        __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
        o[i] = *reinterpret_cast<uint32_t*>(&h);
      }
      ptx::stg128_cs((unsigned long long)(pool + (size_t)slot * width + c8[u] * 8), make_uint4(o[0], o[1], o[2], o[3]));
    }
  }
}

scd_status_t check_desc(const scd_int4_desc_t* d) {
  if (!d) return fail(SCD_E_ARG, "int4: null descriptor");
  if (d->n_kv_heads < 1 || d->head_dim < 1 || d->block_size < 1) return fail(SCD_E_ARG, "int4: bad geometry");
  if (d->group != 32 && d->group != 64 && d->group != 128) return fail(SCD_E_UNSUPPORTED, "int4: group %d not in {32, 64, 128}", d->group);
  if (d->head_dim % d->group) return fail(SCD_E_SHAPE, "int4: group %d does not divide head_dim %d", d->group, d->head_dim);
  return SCD_OK;
}

Q4Layout make_layout(const scd_int4_desc_t* d, int T) {
  const size_t W = (size_t)d->n_kv_heads * d->head_dim;
  Q4Layout l;
  const size_t qb = align_up((size_t)T * (W / 2), 128);
  const size_t mb = align_up((size_t)T * (W / d->group) * 2, 128);
  l.scale_off = qb;
  l.zero_off = qb + mb;
  l.tensor_stride = qb + 2 * mb;
  return l;
}

}  // namespace
}  // namespace scd

using namespace scd;

extern "C" scd_status_t scd_int4_layout(const scd_int4_desc_t* d, int32_t total_tokens, int32_t n_tensors, size_t* tensor_stride,
                                        size_t* scale_offset, size_t* zero_offset, size_t* total_bytes, size_t* payload_bytes) {
  scd_status_t st = check_desc(d);
  if (st != SCD_OK) return st;
  if (total_tokens < 0 || n_tensors < 0) return fail(SCD_E_ARG, "int4: negative size");
  const Q4Layout l = make_layout(d, total_tokens);
  if (tensor_stride) *tensor_stride = l.tensor_stride;
  if (scale_offset) *scale_offset = l.scale_off;
  if (zero_offset) *zero_offset = l.zero_off;
  if (total_bytes) *total_bytes = l.tensor_stride * (size_t)n_tensors;
  const size_t W = (size_t)d->n_kv_heads * d->head_dim;
  if (payload_bytes) *payload_bytes = (size_t)n_tensors * total_tokens * (W / 2 + 4 * (W / d->group));
  return SCD_OK;
}

extern "C" scd_status_t scd_int4_quantize(const scd_int4_desc_t* d, int32_t total_tokens, int32_t n_tensors, const void* const* src,
                                          int64_t token_stride, void* packed, void* stream) {
  reset_launch_count();
  scd_status_t st = check_desc(d);
  if (st != SCD_OK) return st;
  if (total_tokens < 0 || n_tensors < 0) return fail(SCD_E_ARG, "int4: negative size");
  if (total_tokens == 0 || n_tensors == 0) return SCD_OK;
  if (!src || !packed) return fail(SCD_E_ARG, "int4: null buffer");
  const int W = d->n_kv_heads * d->head_dim;
  if (token_stride < W || (token_stride % 8)) return fail(SCD_E_ALIGN, "int4: token stride %lld (needs >= %d, multiple of 8)", (long long)token_stride, W);
  if (((uintptr_t)packed) % 128) return fail(SCD_E_ALIGN, "int4: packed buffer not 128-byte aligned");
  const Q4Layout l = make_layout(d, total_tokens);
  cudaStream_t s = (cudaStream_t)stream;
  reset_launch_count();
  for (int t0 = 0; t0 < n_tensors; t0 += Q4_MAX_TENSORS) {
    const int nt = std::min(Q4_MAX_TENSORS, n_tensors - t0);
    Q4Ptrs P;
    for (int i = 0; i < nt; ++i) {
      if (!src[t0 + i] || ((uintptr_t)src[t0 + i] % 16)) return fail(SCD_E_ALIGN, "int4: source %d null or not 16-byte aligned", t0 + i);
      P.p[i] = src[t0 + i];
    }
    dim3 grid((total_tokens + Q4_ROWS - 1) / Q4_ROWS, nt);
    uint8_t* out = (uint8_t*)packed + (size_t)t0 * l.tensor_stride;
    prof_begin(s);
    if (d->group == 32) int4_quantize_kernel<4><<<grid, Q4_THREADS, 0, s>>>(P, token_stride, total_tokens, W, out, l);
    else if (d->group == 64) int4_quantize_kernel<8><<<grid, Q4_THREADS, 0, s>>>(P, token_stride, total_tokens, W, out, l);
    else int4_quantize_kernel<16><<<grid, Q4_THREADS, 0, s>>>(P, token_stride, total_tokens, W, out, l);
    prof_end(s, SCD_PROF_INT4_QUANT);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SCD_E_CUDA, "int4_quantize_kernel launch: %s", cudaGetErrorString(e));
    count_launch();
  }
  return SCD_OK;
}

extern "C" scd_status_t scd_int4_dequantize_paged(const scd_int4_desc_t* d, const scd_batch_t* b, int32_t n_tensors, const void* packed,
                                                  void* const* pools, int32_t n_blocks, void* stream) {
  reset_launch_count();
  scd_status_t st = check_desc(d);
  if (st != SCD_OK) return st;
  if (!b || n_tensors < 0 || b->total_tokens < 0) return fail(SCD_E_ARG, "int4: bad batch");
  if (b->total_tokens == 0 || b->n_seqs == 0 || n_tensors == 0) return SCD_OK;
  if (!packed || !pools || !b->cu_seqlens || !b->page_table) return fail(SCD_E_ARG, "int4: null buffer");
  if (n_blocks < 1) return fail(SCD_E_ARG, "int4: n_blocks %d", n_blocks);
  if (((uintptr_t)packed) % 128) return fail(SCD_E_ALIGN, "int4: packed buffer not 128-byte aligned");
  const int W = d->n_kv_heads * d->head_dim;
  const Q4Layout l = make_layout(d, b->total_tokens);
  BatchDev bd;
  bd.cu_seqlens = b->cu_seqlens;
  bd.page_table = b->page_table;
  bd.pos_offset = nullptr;
  bd.n_seqs = b->n_seqs;
  bd.total_tokens = b->total_tokens;
  bd.max_pages_per_seq = b->max_pages_per_seq;
  bd.block_size = d->block_size;
  bd.n_blocks = n_blocks;
  cudaStream_t s = (cudaStream_t)stream;
  reset_launch_count();
  for (int t0 = 0; t0 < n_tensors; t0 += Q4_MAX_TENSORS) {
    const int nt = std::min(Q4_MAX_TENSORS, n_tensors - t0);
    Q4Ptrs P;
    for (int i = 0; i < nt; ++i) {
      if (!pools[t0 + i] || ((uintptr_t)pools[t0 + i] % 16)) return fail(SCD_E_ALIGN, "int4: pool %d null or not 16-byte aligned", t0 + i);
      P.p[i] = pools[t0 + i];
    }
    dim3 grid((b->total_tokens + Q4_ROWS - 1) / Q4_ROWS, nt);
    const uint8_t* in = (const uint8_t*)packed + (size_t)t0 * l.tensor_stride;
    prof_begin(s);
    if (d->group == 32) int4_dequantize_paged_kernel<4><<<grid, Q4_THREADS, 0, s>>>(in, l, P, bd, W);
    else if (d->group == 64) int4_dequantize_paged_kernel<8><<<grid, Q4_THREADS, 0, s>>>(in, l, P, bd, W);
    else int4_dequantize_paged_kernel<16><<<grid, Q4_THREADS, 0, s>>>(in, l, P, bd, W);
    prof_end(s, SCD_PROF_INT4_DEQUANT);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SCD_E_CUDA, "int4_dequantize_paged_kernel launch: %s", cudaGetErrorString(e));
    count_launch();
  }
  return SCD_OK;
}
