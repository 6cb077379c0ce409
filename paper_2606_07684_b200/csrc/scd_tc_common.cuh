// Shared between the tcgen05 kernels (scd_tc.cu: generic GEMM + epilogues; scd_tc_kv.cu: the
// paged-KV specialisation): kernel parameters, tile constants, small device helpers.
#pragma once

#include <cuda_fp16.h>

#include <utility>

#include "ptx.cuh"
#include "scd_device.cuh"
#include "scd_tc.h"

namespace scd {

// ---------------------------------------------------------------------------------
// kernel parameters
// ---------------------------------------------------------------------------------
struct TcSeg {
  const float* col_vec;      // EPI_CODES: c[n] (subtracted); else mean / bias [N] (added)
  const float* a_scale;      // row scales of e4m3 codes used as A (null otherwise)
  void* out0;
  void* out1;
  float* aux;
  float* scale0;             // fp8 pools: per-(slot, head) scales of out0 / out1
  float* scale1;
  const float* rowscale_in;  // NORM_RMS: sum-of-squares partials [n_partials][M]
  int32_t a_map, a_z, b_map, rope_cols;
};

struct TcParams {
  CUtensorMap a_maps[TC_MAX_AMAPS];
  TcSeg segs[TC_MAX_SEGS];
  uint32_t rope_g[64];                // theta^(-2j/d_h) / (2 pi) as a Q0.32 fraction of a turn
  const CUtensorMap* b_maps;          // plan-owned, global memory
  BatchDev batch;
  int32_t n_segs, M, N, K;
  int32_t m_tiles, n_tiles, num_kb, block_n, stages;
  int32_t kv_compact;                 // generic kernel, EPI_KV: compact epilogue (4 KB staging, bias through L1)
  int32_t sub_n;                      // generic kernel: columns per epilogue staging sub-tile
  int32_t stg_warp_bytes;             // generic kernel: per-warp epilogue staging bytes
  int32_t a_prefetch;                 // generic kernel: k-blocks of A pulled into L2 ahead of their TMA load (0 = off)
  int32_t msb;                        // generic kernel: m-tiles per L2 super-block (tile_decode)
  int32_t a_kb_per_head;              // >0: A is [T, H, d_h] head-strided, k-blocks per head
  int32_t split, pool_width, head_dim, rope_style, act, code_dtype;
  int32_t n_partials, rms_dim;
  float rms_eps;
  int32_t* sched;                     // paged-KV kernel: {next chunk, CTAs done}
  int32_t chunk_tiles, n_chunks;      // paged-KV kernel: consecutive tiles per dynamically claimed unit
  int32_t head_rank;                  // paged-KV kernel, per-head REUSE: codes per head (A/B are block-diagonal), else 0
  int32_t prof_id;                    // host only: id under which scd_profile_* reports the launch
  int32_t static_tiles, dyn_begin;    // paged-KV kernel: per-CTA static share, first dynamically claimed tile
  int32_t a_is_codes;                 // paged-KV kernel: A is a code segment (e4m3 codes are widened in shared memory)
  int32_t pool_e4m3;                  // paged-KV kernel: pools are e4m3 bytes + per-(slot, head) fp32 scales
  int32_t pair;                       // generic kernel, host only: launch as CTA pairs (cta_group::2), B maps have 128-row boxes
  int32_t a_gather;                   // generic kernel: A rows are gathered through P.batch.page_table (paged producer cache)
  int32_t dep_wait_late;              // both kernels: this launch reads nothing its stream predecessor writes (see tc_encode)
  int32_t b_res;                      // generic kernel, PATCH GEMM-1: the B tile stays resident across a CTA's consecutive m-tiles
  long long pool_slots;               // paged epilogues: n_blocks * block_size (slot numbers are kept as int32)
};

constexpr int KV_SCHED_SETS = 64;
constexpr int BLOCK_M = 128, BLOCK_K = 64, MAX_STAGES = 8, TMEM_COLS = 512;
constexpr int EPI_WARPS = 8;                                // two per TMEM lane quadrant, splitting the columns
constexpr int A_STAGE_BYTES = BLOCK_M * BLOCK_K * 2;        // 16 KB
constexpr int SUB_N = 128;                                  // epilogue sub-tile width (columns)
constexpr int STG_WARP_BYTES = 32 * SUB_N * 2;              // per-warp staging: 32 rows x 256 B
constexpr int VEC_WARP_BYTES = 256 * 4;                     // per-warp copy of the tile's mean / bias slice


__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

// (cos, sin) of position * theta^(-2j/d_h).  The angle is tracked as a 32-bit fraction of a
// turn: pos * g wraps modulo 2^32 exactly, so the reduced angle in [-pi, pi) has an absolute
// error <= pos * 2 pi * 2^-33 + 2^-24 turn (2.4e-5 rad at 32k positions) before the MUFU
// approximations (2^-21 abs).  No table, no memory traffic.
__device__ __forceinline__ float2 rope_cs(int pos, uint32_t g) {
  const float x = (float)(int32_t)((uint32_t)pos * g) * 1.4629180792671596e-9f;   // 2 pi / 2^32
  return make_float2(__cosf(x), __sinf(x));
}

// two e4m3 codes, each in the high byte of a 16-bit half -> two bf16 (exact): s.eeee.mmm -> s.0000eeee.mmm0000 is the
// same number times 2^-120, normals and subnormals alike; one exact bf16 multiply by 2^120 finishes the conversion
__device__ __forceinline__ uint32_t e4m3x2_to_bf16x2(uint32_t x) {
  const uint32_t y = (x & 0x80008000u) | ((x >> 4) & 0x07f007f0u);
  uint32_t r;
  asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(y), "r"(0x7b807b80u));   // x 2^120
  return r;
}

// packed fp32 pairs (FFMA2 / FMUL2 on sm_100a): half the FMA-pipe instructions of the epilogue
__device__ __forceinline__ unsigned long long f2_pack(float lo, float hi) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void f2_unpack(unsigned long long v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long f2_fma(unsigned long long a, unsigned long long b, unsigned long long c) {
  unsigned long long r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
// ptxas folds this into the consuming FFMA2's operand negation
__device__ __forceinline__ unsigned long long f2_neg(unsigned long long a) {
  float lo, hi;
  f2_unpack(a, lo, hi);
  return f2_pack(-lo, -hi);
}
__device__ __forceinline__ unsigned long long f2_add(unsigned long long a, unsigned long long b) {
  unsigned long long r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ unsigned long long f2_mul(unsigned long long a, unsigned long long b) {
  unsigned long long r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}

// Launch with programmatic stream serialisation: barrier init / TMEM allocation / descriptor fetch of this
// kernel overlap the tail of the previous one; the kernels call grid_dep_wait() before touching global memory.
// `cluster` > 1: thread-block clusters of that many CTAs along x (CTA pairs for cta_group::2 kernels).
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t s, int cluster, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)block);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  if (cluster > 1) {
    at[1].id = cudaLaunchAttributeClusterDimension;
    at[1].val.clusterDim.x = (unsigned)cluster;
    at[1].val.clusterDim.y = 1;
    at[1].val.clusterDim.z = 1;
    cfg.numAttrs = 2;
  }
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}
// how many clusters of `cluster` CTAs of this kernel can be resident at once (persistent kernels size their grid by it)
template <typename... KArgs>
inline int max_active_clusters(void (*kernel)(KArgs...), int block, size_t smem, int cluster) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)cluster);
  cfg.blockDim = dim3((unsigned)block);
  cfg.dynamicSmemBytes = smem;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = (unsigned)cluster;
  at[0].val.clusterDim.y = 1;
  at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  int n = 0;
  if (cudaOccupancyMaxActiveClusters(&n, kernel, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
  return n;
}

__device__ __forceinline__ float4 ldg_f4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

// scd_tc_kv.cu: can the specialised paged-KV kernel take this launch?  (head_dim 128, HALF RoPE,
// 256-column tiles, whole tiles only.)  P.M/N/K/block_n/split/rope fields must be filled.
bool tc_kv_eligible(const scd_plan_t* p, const TcParams& P);
scd_status_t launch_tc_kv(const scd_plan_t* p, TcParams& P, cudaStream_t s);


}  // namespace scd
