// Small device helpers shared by the SIMT and tcgen05 kernels: element conversion,
// code (un)packing, RoPE pairing, packed-row -> (position, slot) lookup.
#pragma once

#include <cuda_bf16.h>
#include <cuda_fp8.h>
#include <stdint.h>

#include "scd_internal.h"

namespace scd {

__device__ __forceinline__ float to_float(float v) { return v; }
__device__ __forceinline__ float to_float(__nv_bfloat16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_float(float v);
template <> __device__ __forceinline__ float from_float<float>(float v) { return v; }
template <> __device__ __forceinline__ __nv_bfloat16 from_float<__nv_bfloat16>(float v) {
  return __float2bfloat16_rn(v);
}

// OCP e4m3fn, round-to-nearest-even, saturating to +-448.
__device__ __forceinline__ uint8_t float_to_e4m3_sat(float v) {
  return (uint8_t)__nv_cvt_float_to_fp8(v, __NV_SATFINITE, __NV_E4M3);
}
// two values at once: one cvt.rn.satfinite.e4m3x2.f32 (low byte = a)
__device__ __forceinline__ uint32_t float2_to_e4m3x2_sat(float a, float b) {
  return (uint32_t)__nv_cvt_float2_to_fp8x2(make_float2(a, b), __NV_SATFINITE, __NV_E4M3);
}
__device__ __forceinline__ float e4m3_to_float(uint8_t b) {
  __half_raw h = __nv_cvt_fp8_to_halfraw((__nv_fp8_storage_t)b, __NV_E4M3);
  return __half2float(__half(h));
}

__device__ __forceinline__ float load_code(const void* base, size_t idx, int code_dtype) {
  if (code_dtype == SCD_F32) return ((const float*)base)[idx];
  if (code_dtype == SCD_BF16) return __bfloat162float(((const __nv_bfloat16*)base)[idx]);
  return e4m3_to_float(((const uint8_t*)base)[idx]);
}
// f32 / bf16 only; e4m3 needs the row amax first and is written by the caller.
__device__ __forceinline__ void store_code(void* base, size_t idx, float v, int code_dtype) {
  if (code_dtype == SCD_F32) ((float*)base)[idx] = v;
  else ((__nv_bfloat16*)base)[idx] = __float2bfloat16_rn(v);
}

// RoPE pairing of channel j of a head: frequency index fi, partner channel jp, and
// whether j is the first ("a") element of its pair.
__device__ __forceinline__ void rope_partner(int style, int j, int half, int& fi, int& jp, bool& first) {
  if (style == SCD_ROPE_HALF) {
    first = j < half;
    fi = first ? j : j - half;
    jp = first ? j + half : j - half;
  } else {
    first = (j & 1) == 0;
    fi = j >> 1;
    jp = j ^ 1;
  }
}

// Packed row n -> request b (largest b with cu_seqlens[b] <= n), t = n - cu_seqlens[b];
// position id = pos_offset[b] + t; slot = page_table[b][t / bs] * bs + t % bs.
__device__ __forceinline__ void row_to_pos_slot(const BatchDev& batch, int row, int& pos, long long& slot) {
  int lo = 0, hi = batch.n_seqs;           // invariant: cu[lo] <= row < cu[hi]
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (__ldg(batch.cu_seqlens + mid) <= row) lo = mid; else hi = mid;
  }
  int t = row - __ldg(batch.cu_seqlens + lo);
  pos = (batch.pos_offset ? __ldg(batch.pos_offset + lo) : 0) + t;
  slot = -1;
  if (batch.page_table) {
    int page = __ldg(batch.page_table + (size_t)lo * batch.max_pages_per_seq + t / batch.block_size);
    // page tables live on the device, so the host cannot validate them: a page id outside the pool (the -1 of an
    // unused entry reached through an inconsistent cu_seqlens, or a stale id) leaves slot = -1 and the row unwritten
    if (page >= 0 && (batch.n_blocks <= 0 || page < batch.n_blocks))
      slot = (long long)page * batch.block_size + t % batch.block_size;
  }
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

}  // namespace scd
