// Group-wise INT4 KV codec: the paper's fastest transport baseline ("Quantized KV: transmits 4-bit quantized KV
// caches (group-wise INT4) and dequantizes on the consumer"; Table 4 :352-359) built as the same-box
// comparison codec of SURVEY 8(f) NEXT-3.  Definition: DESIGN.md section 2, U19 (oracle/int4_oracle.py restates it):
//
//   group = G consecutive channels of one token row (G in {32, 64, 128}, G | head_dim)
//   lo = min x, hi = max x;  s = bf16_rne((hi - lo) / 15) (1 if that is 0);  q = clamp(rint((x - lo) * (1 / s)), 0, 15)
//   byte j = q[2j] | q[2j + 1] << 4;  metadata = {bf16 s, bf16 lo} per group;  x^ = bf16_rne(q * s + lo)
//
// Every decision is IEEE fp32 (div.rn once per group, mul.rn, cvt.rni), so codes and dequantised values are bit-exact
// against the oracle.
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
  size_t tensor_stride, meta_off;
};

__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

// Work split of a CTA (256 threads, Q4_ROWS token rows of one tensor): `tpr` = 2^shift threads walk a row's 8-element
// items (item c8 = 8 channels = one 16-byte access of the bf16 side), 256 / tpr rows at a time; no integer division.
// ---- producer: quantise ----
template <int LANES>   // lanes per group = G / 8
__global__ void __launch_bounds__(Q4_THREADS) int4_quantize_kernel(const Q4Ptrs src, long long token_stride, int T, int width, int shift,
                                                                   uint8_t* __restrict__ out, Q4Layout lay) {
  const int ipr = width >> 3;                       // 8-element items per row
  const int row0 = blockIdx.x * Q4_ROWS;
  const int rows = min(Q4_ROWS, T - row0);
  const __nv_bfloat16* x = (const __nv_bfloat16*)src.p[blockIdx.y];
  uint8_t* base = out + (size_t)blockIdx.y * lay.tensor_stride;
  uint32_t* qout = (uint32_t*)base;
  uint32_t* mout = (uint32_t*)(base + lay.meta_off);      // {bf16 scale, bf16 zero} per group
  const int gpr = ipr / LANES;                      // groups per row
  const int tpr = 1 << shift, rpp = Q4_THREADS >> shift;
  const int c_first = threadIdx.x & (tpr - 1), r_first = threadIdx.x >> shift;
  for (int c0 = 0; c0 < ipr; c0 += tpr) {           // warp-uniform trip count (shuffles below)
    const int c8 = c0 + c_first;
    const bool c_ok = c8 < ipr;                     // ipr and tpr are multiples of LANES: a group never splits
    for (int r0 = r_first; r0 < Q4_ROWS; r0 += 4 * rpp) {
      uint4 v[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int r = r0 + u * rpp;
        v[u] = make_uint4(0u, 0u, 0u, 0u);
        if (r < rows && c_ok) v[u] = __ldcs(reinterpret_cast<const uint4*>(x + (size_t)(row0 + r) * token_stride + c8 * 8));
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int r = r0 + u * rpp;
        const uint32_t w[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
        float f[8];
#pragma unroll
        for (int i = 0; i < 4; ++i) { f[2 * i] = bf16_lo(w[i]); f[2 * i + 1] = bf16_hi(w[i]); }
        float lo = f[0], hi = f[0];
#pragma unroll
        for (int i = 1; i < 8; ++i) { lo = fminf(lo, f[i]); hi = fmaxf(hi, f[i]); }
#pragma unroll
        for (int o = 1; o < LANES; o <<= 1) {       // the LANES lanes of a group are adjacent lanes of one row
          lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, o));
          hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        const __nv_bfloat16 sb = __float2bfloat16_rn(__fdiv_rn(__fsub_rn(hi, lo), 15.0f));
        float s = __bfloat162float(sb);
        uint32_t meta = (uint32_t)__bfloat16_as_ushort(sb);
        if (s == 0.0f) { s = 1.0f; meta = 0x3f80u; }
        meta |= (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(lo)) << 16;
        const float inv = __fdiv_rn(1.0f, s);
        // 0 <= t = (x - lo) * (1 / s) <= 15 (1 + 2^-8)(1 + 2^-23)^2 < 15.5 because s = bf16((hi - lo) / 15) is within 2^-9 of
        // the quotient: the rounded code is in [0, 15] by construction and the oracle's clamp never acts.  rint(t) without the
        // quarter-rate F2I: t + 1.5 * 2^23 rounds to nearest-even at unit spacing, so the code is the sum's low mantissa bits,
        // bits(t + M) = 0x4B400000 + q; the eight nibbles are gathered by integer multiply-adds, the constant taken off once
        uint32_t packed = 0u - 0x4B400000u * 0x11111111u;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const uint32_t b = __float_as_uint(__fadd_rn(__fmul_rn(__fsub_rn(f[i], lo), inv), 12582912.0f));
          packed += b << (4 * i);
        }
        if (r < rows && c_ok) {
          const size_t rr = (size_t)(row0 + r);
          __stcs(qout + rr * ipr + c8, packed);
          if ((c8 & (LANES - 1)) == 0) __stcs(mout + rr * gpr + c8 / LANES, meta);
        }
      }
    }
  }
}

// ---- consumer: dequantise into the paged pool ----
template <int LANES>
__global__ void __launch_bounds__(Q4_THREADS) int4_dequantize_paged_kernel(const uint8_t* __restrict__ in, Q4Layout lay, const Q4Ptrs pools,
                                                                           BatchDev batch, int width, int shift) {
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
  const uint8_t* base = in + (size_t)blockIdx.y * lay.tensor_stride;
  const uint32_t* qin = (const uint32_t*)base;
  const uint32_t* min_ = (const uint32_t*)(base + lay.meta_off);
  __nv_bfloat16* pool = (__nv_bfloat16*)pools.p[blockIdx.y];
  const int gpr = ipr / LANES;
  const int tpr = 1 << shift, rpp = Q4_THREADS >> shift;
  const int c_first = threadIdx.x & (tpr - 1), r_first = threadIdx.x >> shift;
  for (int c8 = c_first; c8 < ipr; c8 += tpr) {
    for (int r0 = r_first; r0 < Q4_ROWS; r0 += 4 * rpp) {
      uint32_t pk[4], meta[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int r = r0 + u * rpp;
        pk[u] = 0; meta[u] = 0;
        if (r < rows) {
          const size_t rr = (size_t)(row0 + r);
          pk[u] = __ldcs(qin + rr * ipr + c8);
          meta[u] = __ldg(min_ + rr * gpr + c8 / LANES);
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int r = r0 + u * rpp;
        if (r >= rows) continue;
        const long long slot = slots[r];
        if (slot < 0) continue;                        // page id outside the pool: the row is not written
        const float s = bf16_lo(meta[u]), z = bf16_hi(meta[u]);
        uint32_t o[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const float a = fmaf((float)((pk[u] >> (8 * i)) & 15u), s, z);
          const float b = fmaf((float)((pk[u] >> (8 * i + 4)) & 15u), s, z);
          __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
          o[i] = *reinterpret_cast<uint32_t*>(&h);
        }
        ptx::stg128_cs((unsigned long long)(pool + (size_t)slot * width + c8 * 8), make_uint4(o[0], o[1], o[2], o[3]));
      }
    }
  }
}

// threads per row: the largest power of two <= min(256, items per row) that is a multiple of the group's lanes
int q4_shift(int ipr, int lanes) {
  int sh = 0;
  while ((2 << sh) <= ipr && (2 << sh) <= Q4_THREADS) ++sh;
  while ((1 << sh) < lanes) ++sh;
  return sh;
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
  const size_t mb = align_up((size_t)T * (W / d->group) * 4, 128);
  l.meta_off = qb;
  l.tensor_stride = qb + mb;
  return l;
}

}  // namespace
}  // namespace scd

using namespace scd;

extern "C" scd_status_t scd_int4_layout(const scd_int4_desc_t* d, int32_t total_tokens, int32_t n_tensors, size_t* tensor_stride,
                                        size_t* meta_offset, size_t* total_bytes, size_t* payload_bytes) {
  scd_status_t st = check_desc(d);
  if (st != SCD_OK) return st;
  if (total_tokens < 0 || n_tensors < 0) return fail(SCD_E_ARG, "int4: negative size");
  const Q4Layout l = make_layout(d, total_tokens);
  if (tensor_stride) *tensor_stride = l.tensor_stride;
  if (meta_offset) *meta_offset = l.meta_off;
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
    if (d->group == 32) int4_quantize_kernel<4><<<grid, Q4_THREADS, 0, s>>>(P, token_stride, total_tokens, W, q4_shift(W / 8, 4), out, l);
    else if (d->group == 64) int4_quantize_kernel<8><<<grid, Q4_THREADS, 0, s>>>(P, token_stride, total_tokens, W, q4_shift(W / 8, 8), out, l);
    else int4_quantize_kernel<16><<<grid, Q4_THREADS, 0, s>>>(P, token_stride, total_tokens, W, q4_shift(W / 8, 16), out, l);
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
    if (d->group == 32) int4_dequantize_paged_kernel<4><<<grid, Q4_THREADS, 0, s>>>(in, l, P, bd, W, q4_shift(W / 8, 4));
    else if (d->group == 64) int4_dequantize_paged_kernel<8><<<grid, Q4_THREADS, 0, s>>>(in, l, P, bd, W, q4_shift(W / 8, 8));
    else int4_dequantize_paged_kernel<16><<<grid, Q4_THREADS, 0, s>>>(in, l, P, bd, W, q4_shift(W / 8, 16));
    prof_end(s, SCD_PROF_INT4_DEQUANT);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SCD_E_CUDA, "int4_dequantize_paged_kernel launch: %s", cudaGetErrorString(e));
    count_launch();
  }
  return SCD_OK;
}
