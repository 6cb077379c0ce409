// tcgen05 / TMEM / TMA path (bf16 states): host entry points used by scd_host.cu.
#pragma once

#include "scd_internal.h"

namespace scd {

constexpr int TC_MAX_SEGS = 64;    // segments per launch (kernel-parameter budget)
constexpr int TC_MAX_AMAPS = 64;   // per-call A tensor maps per launch

// Is this (model, layers) combination implemented on the tensor-core path?
scd_status_t tc_supported(const scd_plan_t* p, const scd_layer_desc_t* layers);
// Builds plan-owned TMA descriptors (B operands) and the fp16 RoPE tables.
scd_status_t tc_plan_init(scd_plan_t* p, cudaStream_t s);

scd_status_t tc_encode(const scd_plan_t* p, const scd_batch_t* batch, const scd_src_t* src, void* codes,
                       const size_t* off, const size_t* soff, cudaStream_t s);
scd_status_t tc_reuse_decode(const scd_plan_t* p, const scd_batch_t* batch, const void* codes,
                             const scd_paged_kv_t* kv, const size_t* off, const size_t* soff, cudaStream_t s);
scd_status_t tc_patch(const scd_plan_t* p, const scd_batch_t* batch, const void* codes, const scd_paged_kv_t* kv,
                      void* ws_act, void* ws_u, float* ws_ss, int group, size_t act_stride, size_t u_stride, size_t ss_stride,
                      const size_t* off, const size_t* soff, cudaStream_t s);

// TMA descriptor of a bf16 matrix [rows][cols] (K-major operand of the tcgen05 kernels): box {64, box_rows}, 128-B swizzle
scd_status_t tc_make_map_2d_bf16(CUtensorMap* m, const void* base, uint64_t cols, uint64_t rows, uint64_t row_pitch_bytes,
                                 uint32_t box_rows);

}  // namespace scd
