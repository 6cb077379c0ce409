// Tensor-core path of the SCD codec for bf16 states on sm_100a.
//
// Every step of the path is one GEMM shape, C[M,N] = A[M,K] Bt[N,K]^T with both operands
// K-major, plus an A-side transform and a fused epilogue (scd_internal.h: EpiKind, AMode).
// One persistent, warp-specialised kernel template serves all of them:
//
//   warp 0      TMA producer: A tile [128 x 64] and Bt tile [BLOCK_N x 64] per k-block into a
//               4-deep shared-memory ring (128-byte swizzle), mbarrier expect_tx / complete_tx
//   warp 1      MMA issuer: one elected thread issues tcgen05.mma (128 x BLOCK_N x 16, bf16 ->
//               fp32) into one of two TMEM accumulator buffers; tcgen05.commit releases the
//               smem stage and finally signals the epilogue
//   warp 2      TMEM allocator (512 columns = 2 accumulator buffers of <= 256 columns)
//   warps 4-7   epilogue: tcgen05.ld (one token row per thread), fused mean / row-scale /
//               RoPE / activation / quantisation, 16-byte stores (codes, workspace, or the
//               token's slot of the paged KV pool); overlaps the next tile's MMAs
//   warps 8-11  (A_DEROPE only) rotate the freshly landed K tile in shared memory by
//               -position (Eq. 5) before the MMA may read it
//
// A launch covers many (layer, branch) segments of equal shape: tile -> (segment, n-tile,
// m-tile) with m fastest, tiles dealt round-robin to one CTA per SM.
#include <cuda_fp16.h>

#include <algorithm>
#include <cstring>

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
  const float* rowscale_in;  // NORM_RMS: sum-of-squares partials [n_partials][M]
  int32_t a_map, a_z, b_map, rope_cols;
};

struct TcParams {
  CUtensorMap a_maps[TC_MAX_AMAPS];
  TcSeg segs[TC_MAX_SEGS];
  const CUtensorMap* b_maps;          // plan-owned, global memory
  BatchDev batch;
  const __half2* rope_h;              // [max_position][head_dim/2] (cos, sin) fp16
  int32_t n_segs, M, N, K;
  int32_t m_tiles, n_tiles, num_kb, block_n;
  int32_t a_kb_per_head;              // >0: A is [T, H, d_h] head-strided, k-blocks per head
  int32_t split, pool_width, head_dim, rope_style, act, code_dtype;
  int32_t n_partials, rms_dim;
  float rms_eps;
};

constexpr int BLOCK_M = 128, BLOCK_K = 64, STAGES = 4, TMEM_COLS = 512;
constexpr int A_STAGE_BYTES = BLOCK_M * BLOCK_K * 2;        // 16 KB

struct __align__(8) TcBarriers {
  uint64_t full[STAGES], empty[STAGES], ready[STAGES];
  uint64_t tmem_full[2], tmem_empty[2];
  uint32_t tmem_base;
};

static size_t tc_smem_bytes(int block_n) {
  return 1024 /*align slack*/ + (size_t)STAGES * (A_STAGE_BYTES + (size_t)block_n * BLOCK_K * 2) + sizeof(TcBarriers);
}

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

// ---------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------
template <int EPI, int AMODE>
__global__ void __launch_bounds__(AMODE == A_DEROPE ? 384 : 256, 1)
tc_gemm_kernel(const __grid_constant__ TcParams P) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const int block_n = P.block_n;
  const uint32_t b_stage_bytes = (uint32_t)block_n * BLOCK_K * 2;
  uint8_t* smem_a = smem;
  uint8_t* smem_b = smem + STAGES * A_STAGE_BYTES;
  TcBarriers* bars = (TcBarriers*)(smem_b + STAGES * b_stage_bytes);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int total_tiles = P.n_segs * P.n_tiles * P.m_tiles;

  if (warp == 0 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) {
      ptx::mbar_init(&bars->full[s], 1);
      ptx::mbar_init(&bars->empty[s], 1);
      ptx::mbar_init(&bars->ready[s], 128);
    }
    for (int a = 0; a < 2; ++a) {
      ptx::mbar_init(&bars->tmem_full[a], 1);
      ptx::mbar_init(&bars->tmem_empty[a], 4);
    }
    ptx::fence_barrier_init();
  }
  if (warp == 2) {
    ptx::tmem_alloc<TMEM_COLS>(&bars->tmem_base);
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = bars->tmem_base;

  if (warp == 0) {
    // ============================== TMA producer ==============================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        const int m_tile = tile % P.m_tiles;
        const int n_tile = (tile / P.m_tiles) % P.n_tiles;
        const TcSeg& sg = P.segs[tile / (P.m_tiles * P.n_tiles)];
        const CUtensorMap* am = &P.a_maps[sg.a_map];
        const CUtensorMap* bm = P.b_maps + sg.b_map;
        for (int kb = 0; kb < P.num_kb; ++kb) {
          ptx::mbar_wait(&bars->empty[stage], phase ^ 1);
          ptx::mbar_expect_tx(&bars->full[stage], A_STAGE_BYTES + b_stage_bytes);
          if (P.a_kb_per_head > 0)
            ptx::tma_load_3d(smem_a + stage * A_STAGE_BYTES, am, &bars->full[stage],
                             (kb % P.a_kb_per_head) * BLOCK_K, kb / P.a_kb_per_head, m_tile * BLOCK_M);
          else
            ptx::tma_load_3d(smem_a + stage * A_STAGE_BYTES, am, &bars->full[stage], kb * BLOCK_K,
                             m_tile * BLOCK_M, sg.a_z);
          ptx::tma_load_2d(smem_b + stage * b_stage_bytes, bm, &bars->full[stage], kb * BLOCK_K, n_tile * block_n);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ============================== MMA issuer ==============================
    if (lane == 0) {
      const uint32_t idesc = ptx::umma_idesc_bf16(BLOCK_M, block_n);
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x, ++it) {
        const int acc = it & 1;
        const uint32_t acc_phase = (it >> 1) & 1;
        ptx::mbar_wait(&bars->tmem_empty[acc], acc_phase ^ 1);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(acc * block_n);
        for (int kb = 0; kb < P.num_kb; ++kb) {
          ptx::mbar_wait(AMODE == A_DEROPE ? &bars->ready[stage] : &bars->full[stage], phase);
          ptx::tc_fence_after();
          const uint64_t da = ptx::umma_desc_sw128(ptx::smem_u32(smem_a + stage * A_STAGE_BYTES));
          const uint64_t db = ptx::umma_desc_sw128(ptx::smem_u32(smem_b + stage * b_stage_bytes));
#pragma unroll
          for (int k = 0; k < BLOCK_K / 16; ++k)
            ptx::mma_bf16(d_tmem, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, (kb | k) != 0);
          ptx::mma_commit(&bars->empty[stage]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        ptx::mma_commit(&bars->tmem_full[acc]);
      }
    }
  } else if (warp >= 4 && warp < 8) {
    // ============================== epilogue ==============================
    const int ew = warp - 4;
    const int half = P.head_dim / 2;
    int it = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x, ++it) {
      const int m_tile = tile % P.m_tiles;
      const int n_tile = (tile / P.m_tiles) % P.n_tiles;
      const TcSeg& sg = P.segs[tile / (P.m_tiles * P.n_tiles)];
      const int acc = it & 1;
      const uint32_t acc_phase = (it >> 1) & 1;
      const int row = m_tile * BLOCK_M + ew * 32 + lane;
      const bool valid = row < P.M;
      const int n0 = n_tile * block_n;
      const int n_end = min(block_n, P.N - n0);              // valid columns in this tile

      // per-row quantities (global loads issued before waiting for the accumulator)
      int pos = 0;
      long long slot = 0;
      float rs = 1.0f;
      if (valid) {
        if (EPI == EPI_KV) row_to_pos_slot(P.batch, row, pos, slot);
        if ((EPI == EPI_KV || EPI == EPI_ACT) && sg.a_scale) rs = __ldg(sg.a_scale + row);
        if (EPI == EPI_KV && sg.rowscale_in) {
          float ss = 0.0f;
          for (int p = 0; p < P.n_partials; ++p) ss += __ldg(sg.rowscale_in + (size_t)p * P.M + row);
          rs *= rsqrtf(ss / (float)P.rms_dim + P.rms_eps);
        }
      }

      ptx::mbar_wait(&bars->tmem_full[acc], acc_phase);
      ptx::tc_fence_after();
      const uint32_t t_row = tmem_base + (uint32_t)(acc * block_n) + ((uint32_t)(ew * 32) << 16);

      if (EPI == EPI_KV) {
        const bool to1 = n0 >= P.split;
        __nv_bfloat16* out = (__nv_bfloat16*)(to1 ? sg.out1 : sg.out0) + (size_t)slot * P.pool_width +
                             (to1 ? n0 - P.split : n0);
        int c = 0;
        while (c < n_end) {
          const int col = n0 + c;
          if (col < sg.rope_cols && P.rope_style == SCD_ROPE_HALF) {
            // one head: pairs (j, j + half), 16 pairs at a time
            for (int j0 = 0; j0 < half; j0 += 16) {
              uint32_t ra[16], rb[16];
              ptx::tmem_ld16(t_row + c + j0, ra);
              ptx::tmem_ld16(t_row + c + half + j0, rb);
              ptx::tmem_ld_wait();
              if (valid) {
                const uint4* tp = reinterpret_cast<const uint4*>(P.rope_h + (size_t)pos * half + j0);
                uint32_t oa[8], ob[8];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                  const uint4 cs4 = __ldg(tp + q);
                  const uint32_t csw[4] = {cs4.x, cs4.y, cs4.z, cs4.w};
                  float va[4], vb[4];
#pragma unroll
                  for (int e = 0; e < 4; ++e) {
                    const int i = q * 4 + e;
                    const float2 cs = __half22float2(*reinterpret_cast<const __half2*>(&csw[e]));
                    float a = __uint_as_float(ra[i]) * rs, b = __uint_as_float(rb[i]) * rs;
                    if (sg.col_vec) {
                      a += __ldg(sg.col_vec + col + j0 + i);
                      b += __ldg(sg.col_vec + col + half + j0 + i);
                    }
                    va[e] = a * cs.x - b * cs.y;
                    vb[e] = b * cs.x + a * cs.y;
                  }
                  oa[q * 2] = pack_bf16x2(va[0], va[1]); oa[q * 2 + 1] = pack_bf16x2(va[2], va[3]);
                  ob[q * 2] = pack_bf16x2(vb[0], vb[1]); ob[q * 2 + 1] = pack_bf16x2(vb[2], vb[3]);
                }
                uint4* da = reinterpret_cast<uint4*>(out + c + j0);
                uint4* db = reinterpret_cast<uint4*>(out + c + half + j0);
                da[0] = make_uint4(oa[0], oa[1], oa[2], oa[3]); da[1] = make_uint4(oa[4], oa[5], oa[6], oa[7]);
                db[0] = make_uint4(ob[0], ob[1], ob[2], ob[3]); db[1] = make_uint4(ob[4], ob[5], ob[6], ob[7]);
              }
            }
            c += P.head_dim;
          } else {
            // 32 columns: plain, or INTERLEAVED RoPE (pairs (2i, 2i+1) are adjacent)
            uint32_t r[32];
            ptx::tmem_ld32(t_row + c, r);
            ptx::tmem_ld_wait();
            if (valid) {
              float v[32];
#pragma unroll
              for (int i = 0; i < 32; ++i) {
                v[i] = __uint_as_float(r[i]) * rs;
                if (sg.col_vec) v[i] += __ldg(sg.col_vec + col + i);
              }
              if (col < sg.rope_cols) {
                const __half2* tp = P.rope_h + (size_t)pos * half + (col % P.head_dim) / 2;
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                  const float2 cs = __half22float2(__ldg(tp + i));
                  const float a = v[2 * i], b = v[2 * i + 1];
                  v[2 * i] = a * cs.x - b * cs.y;
                  v[2 * i + 1] = b * cs.x + a * cs.y;
                }
              }
              uint4* dst = reinterpret_cast<uint4*>(out + c);
#pragma unroll
              for (int q = 0; q < 4; ++q)
                dst[q] = make_uint4(pack_bf16x2(v[q * 8], v[q * 8 + 1]), pack_bf16x2(v[q * 8 + 2], v[q * 8 + 3]),
                                    pack_bf16x2(v[q * 8 + 4], v[q * 8 + 5]), pack_bf16x2(v[q * 8 + 6], v[q * 8 + 7]));
            }
            c += 32;
          }
        }
      } else if (EPI == EPI_CODES) {
        // z = acc - c[n]; bf16 codes, or e4m3 with a per-row fp32 scale (tile spans all of N)
        float amax = 0.0f;
        if (P.code_dtype == SCD_E4M3_ROWSCALE) {
          for (int c = 0; c < n_end; c += 32) {
            uint32_t r[32];
            ptx::tmem_ld32(t_row + c, r);
            ptx::tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i)
              if (c + i < n_end) amax = fmaxf(amax, fabsf(__uint_as_float(r[i]) - __ldg(sg.col_vec + n0 + c + i)));
          }
        }
        const float sc = amax > 0.0f ? amax / 448.0f : 1.0f;
        if (P.code_dtype == SCD_E4M3_ROWSCALE && valid) sg.aux[row] = sc;
        for (int c = 0; c < n_end; c += 32) {
          uint32_t r[32];
          ptx::tmem_ld32(t_row + c, r);
          ptx::tmem_ld_wait();
          if (valid) {
            float v[32];
#pragma unroll
            for (int i = 0; i < 32; ++i)
              v[i] = (c + i < n_end) ? __uint_as_float(r[i]) - __ldg(sg.col_vec + n0 + c + i) : 0.0f;
            if (P.code_dtype == SCD_E4M3_ROWSCALE) {
              uint8_t* dst = (uint8_t*)sg.out0 + (size_t)row * P.N + n0 + c;
#pragma unroll
              for (int q = 0; q < 2; ++q) {
                if (c + q * 16 >= n_end) break;
                uint32_t w[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                  uint32_t b = 0;
#pragma unroll
                  for (int y = 0; y < 4; ++y)
                    b |= (uint32_t)float_to_e4m3_sat(__fdiv_rn(v[q * 16 + e * 4 + y], sc)) << (8 * y);
                  w[e] = b;
                }
                reinterpret_cast<uint4*>(dst)[q] = make_uint4(w[0], w[1], w[2], w[3]);
              }
            } else {
              __nv_bfloat16* dst = (__nv_bfloat16*)sg.out0 + (size_t)row * P.N + n0 + c;
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                if (c + q * 8 >= n_end) break;
                reinterpret_cast<uint4*>(dst)[q] =
                    make_uint4(pack_bf16x2(v[q * 8], v[q * 8 + 1]), pack_bf16x2(v[q * 8 + 2], v[q * 8 + 3]),
                               pack_bf16x2(v[q * 8 + 4], v[q * 8 + 5]), pack_bf16x2(v[q * 8 + 6], v[q * 8 + 7]));
              }
            }
          }
        }
      } else {
        // EPI_ACT: act(acc * rs + b1) ; EPI_U: acc + b2 and the row's partial sum of squares
        float ss = 0.0f;
        __nv_bfloat16* dst_row = (__nv_bfloat16*)sg.out0 + (size_t)row * P.N + n0;
        for (int c = 0; c < n_end; c += 32) {
          uint32_t r[32];
          ptx::tmem_ld32(t_row + c, r);
          ptx::tmem_ld_wait();
          if (valid) {
            float v[32];
#pragma unroll
            for (int i = 0; i < 32; ++i) {
              float x = 0.0f;
              if (c + i < n_end) {
                x = __uint_as_float(r[i]) * rs;
                if (sg.col_vec) x += __ldg(sg.col_vec + n0 + c + i);
                if (EPI == EPI_ACT && P.act == SCD_ACT_SILU) x = x / (1.0f + __expf(-x));
                if (EPI == EPI_U) ss += x * x;
              }
              v[i] = x;
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              if (c + q * 8 >= n_end) break;
              reinterpret_cast<uint4*>(dst_row + c)[q] =
                  make_uint4(pack_bf16x2(v[q * 8], v[q * 8 + 1]), pack_bf16x2(v[q * 8 + 2], v[q * 8 + 3]),
                             pack_bf16x2(v[q * 8 + 4], v[q * 8 + 5]), pack_bf16x2(v[q * 8 + 6], v[q * 8 + 7]));
            }
          }
        }
        if (EPI == EPI_U && valid && sg.aux) sg.aux[(size_t)n_tile * P.M + row] = ss;
      }

      // hand the accumulator buffer back to the MMA warp
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(&bars->tmem_empty[acc]);
    }
  } else if (AMODE == A_DEROPE && warp >= 8) {
    // ============================== A transform: deRoPE in shared memory ==============================
    // One token row per thread.  A k-block row is 128 B = 8 chunks of 16 B, chunk c stored at
    // position c ^ (row & 7) (128-byte swizzle).  Channel pairs (j, j + d_h/2) of a head:
    //   d_h = 128: same chunk / element of two consecutive k-blocks (stages s, s+1)
    //   d_h =  64: chunks c and c + 4 of one k-block;  d_h = 32: chunks c and c + 2 (two heads per block)
    const int tr = threadIdx.x - 256;                 // 0..127 = row in tile
    const int half = P.head_dim / 2;
    int stage = 0;
    uint32_t phase = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
      const int m_tile = tile % P.m_tiles;
      const int row = m_tile * BLOCK_M + tr;
      int pos = 0;
      long long slot;
      if (row < P.M) row_to_pos_slot(P.batch, row, pos, slot);
      const __half2* trow = P.rope_h + (size_t)pos * half;
      const uint32_t row_off = (uint32_t)(tr >> 3) * 1024 + (uint32_t)(tr & 7) * 128;
      const int step = P.head_dim == 128 ? 2 : 1;     // k-blocks consumed per iteration
      for (int kb = 0; kb < P.num_kb; kb += step) {
        const int s0 = stage, s1 = (stage + 1) % STAGES;
        ptx::mbar_wait(&bars->full[s0], phase);
        if (step == 2) ptx::mbar_wait(&bars->full[s1], (s1 == 0) ? (phase ^ 1) : phase);
        uint8_t* ra = smem_a + s0 * A_STAGE_BYTES + row_off;
        uint8_t* rb = step == 2 ? smem_a + s1 * A_STAGE_BYTES + row_off : ra;
        const int pair_chunks = P.head_dim == 128 ? 8 : half / 8;      // chunks in the "a" half
        const int groups = P.head_dim == 128 ? 1 : BLOCK_K / P.head_dim; // heads per k-block
        for (int gidx = 0; gidx < groups; ++gidx)
          for (int cc = 0; cc < pair_chunks; ++cc) {
            const int ca = P.head_dim == 128 ? cc : gidx * (P.head_dim / 8) + cc;
            const int cb = P.head_dim == 128 ? cc : ca + pair_chunks;
            uint4* pa = reinterpret_cast<uint4*>(ra + ((ca ^ (tr & 7)) << 4));
            uint4* pb = reinterpret_cast<uint4*>(rb + ((cb ^ (tr & 7)) << 4));
            uint4 xa = *pa, xb = *pb;
            const uint4 cs4a = __ldg(reinterpret_cast<const uint4*>(trow + cc * 8));
            const uint4 cs4b = __ldg(reinterpret_cast<const uint4*>(trow + cc * 8 + 4));
            const uint32_t csw[8] = {cs4a.x, cs4a.y, cs4a.z, cs4a.w, cs4b.x, cs4b.y, cs4b.z, cs4b.w};
            uint32_t* wa = reinterpret_cast<uint32_t*>(&xa);
            uint32_t* wb = reinterpret_cast<uint32_t*>(&xb);
#pragma unroll
            for (int w = 0; w < 4; ++w) {
              const float2 a2 = __bfloat1622float2(*reinterpret_cast<__nv_bfloat162*>(&wa[w]));
              const float2 b2 = __bfloat1622float2(*reinterpret_cast<__nv_bfloat162*>(&wb[w]));
              const float2 c0 = __half22float2(*reinterpret_cast<const __half2*>(&csw[2 * w]));
              const float2 c1 = __half22float2(*reinterpret_cast<const __half2*>(&csw[2 * w + 1]));
              // rotation by -phi:  a' = a cos + b sin ; b' = b cos - a sin
              wa[w] = pack_bf16x2(a2.x * c0.x + b2.x * c0.y, a2.y * c1.x + b2.y * c1.y);
              wb[w] = pack_bf16x2(b2.x * c0.x - a2.x * c0.y, b2.y * c1.x - a2.y * c1.y);
            }
            *pa = xa;
            *pb = xb;
          }
        ptx::fence_proxy_async_smem();
        ptx::mbar_arrive(&bars->ready[s0]);
        if (step == 2) ptx::mbar_arrive(&bars->ready[s1]);
        for (int q = 0; q < step; ++q)
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
    }
  }

  // ============================== teardown ==============================
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc<TMEM_COLS>(tmem_base);
}

// ---------------------------------------------------------------------------------
// host side: tensor maps
// ---------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

// bf16 tensor [d2][d1][d0] (d0 contiguous), strides in bytes for d1, d2; box {64, box1, 1}, 128-B swizzle
static scd_status_t make_map(CUtensorMap* m, const void* base, uint64_t d0, uint64_t d1, uint64_t d2, uint64_t s1,
                             uint64_t s2, uint32_t box1_or_0, uint32_t box2_rows) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return fail(SCD_E_CUDA, "cuTensorMapEncodeTiled entry point not found");
  cuuint64_t dims[3] = {d0, d1, d2};
  cuuint64_t strides[2] = {s1, s2};
  cuuint32_t box[3] = {BLOCK_K, box1_or_0, box2_rows};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS)
    return fail(SCD_E_CUDA, "cuTensorMapEncodeTiled failed (%d): dims %llu,%llu,%llu strides %llu,%llu box %u,%u,%u", (int)r,
                (unsigned long long)d0, (unsigned long long)d1, (unsigned long long)d2, (unsigned long long)s1,
                (unsigned long long)s2, box[0], box[1], box[2]);
  return SCD_OK;
}

// Bt [N, K] K-major, 2-D
static scd_status_t make_b_map(CUtensorMap* m, const void* base, int N, int K, int block_n) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return fail(SCD_E_CUDA, "cuTensorMapEncodeTiled entry point not found");
  cuuint64_t dims[2] = {(cuuint64_t)K, (cuuint64_t)N};
  cuuint64_t strides[1] = {(cuuint64_t)K * 2};
  cuuint32_t box[2] = {BLOCK_K, (cuuint32_t)block_n};
  cuuint32_t es[2] = {1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, es,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(SCD_E_CUDA, "cuTensorMapEncodeTiled (B %dx%d box %d) failed (%d)", N, K, block_n, (int)r);
  return SCD_OK;
}

static int pick_block_n_div(int n) {            // largest tile width that divides n (paged / split epilogues)
  for (int b : {256, 128, 64, 32})
    if (n % b == 0) return b;
  return 0;
}
static int pick_block_n_cover(int n) {          // smallest multiple of 16 covering n, capped at 256
  int b = (n + 15) / 16 * 16;
  return b > 256 ? 256 : b;
}

// fp16 (cos, sin) tables, built from the plan's fp32 tables
__global__ void rope_to_half_kernel(const float2* __restrict__ src, __half2* __restrict__ dst, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    dst[i] = __floats2half2_rn(src[i].x, src[i].y);
}

scd_status_t tc_supported(const scd_plan_t* p, const scd_layer_desc_t* layers) {
  const scd_model_desc_t& m = p->model;
  if (p->D % 32) return fail(SCD_E_UNSUPPORTED, "D = %d not a multiple of 32", p->D);
  if (m.d_model % 8) return fail(SCD_E_UNSUPPORTED, "d_model %d not a multiple of 8", m.d_model);
  for (int l = 0; l < m.n_layers; ++l) {
    if (layers[l].kind == SCD_PATCH && layers[l].d_aligner % 8)
      return fail(SCD_E_UNSUPPORTED, "layer %d: d_aligner not a multiple of 8", l);
    if (m.code_dtype == SCD_E4M3_ROWSCALE) {
      int r[3] = {layers[l].kind == SCD_REUSE ? layers[l].r_k : 0, layers[l].kind == SCD_REUSE ? layers[l].r_v : 0,
                  layers[l].kind == SCD_PATCH ? layers[l].r_h : 0};
      for (int x : r)
        if (x > 256) return fail(SCD_E_UNSUPPORTED, "layer %d: e4m3 codes need rank <= 256 (row amax in one tile)", l);
    }
  }
  return SCD_OK;
}

scd_status_t tc_plan_init(scd_plan_t* p, cudaStream_t s) {
  const scd_model_desc_t& m = p->model;
  const int nseg = (int)p->segs.size(), np = (int)p->patches.size();
  std::vector<CUtensorMap> maps((size_t)2 * nseg + 3 * np);
  memset(maps.data(), 0, maps.size() * sizeof(CUtensorMap));
  scd_status_t st;
  for (int i = 0; i < nseg; ++i) {
    const SegPlan& sp = p->segs[i];
    if ((st = make_b_map(&maps[i], sp.enc_t, sp.rank, sp.width, pick_block_n_cover(sp.rank))) != SCD_OK) return st;
    if (sp.dec_t)
      if ((st = make_b_map(&maps[nseg + i], sp.dec_t, p->D, sp.rank, pick_block_n_div(p->D))) != SCD_OK) return st;
  }
  for (int j = 0; j < np; ++j) {
    const PatchPlan& pp = p->patches[j];
    if ((st = make_b_map(&maps[2 * nseg + 3 * j], pp.w1_t, pp.d_a, pp.r_h, pick_block_n_cover(pp.d_a))) != SCD_OK) return st;
    if ((st = make_b_map(&maps[2 * nseg + 3 * j + 1], pp.w2_t, m.d_model, pp.d_a, pick_block_n_cover(m.d_model))) != SCD_OK) return st;
    if ((st = make_b_map(&maps[2 * nseg + 3 * j + 2], pp.wkv, 2 * p->D, m.d_model, pick_block_n_div(p->D))) != SCD_OK) return st;
  }
  void* d = nullptr;
  if (cudaMalloc(&d, maps.size() * sizeof(CUtensorMap) + 64) != cudaSuccess) return fail(SCD_E_NOMEM, "cudaMalloc(tensor maps)");
  p->allocs.push_back(d);
  if (cudaMemcpy(d, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice) != cudaSuccess)
    return fail(SCD_E_CUDA, "cudaMemcpy(tensor maps)");
  p->tc_bmaps = d;

  const size_t n = (size_t)m.max_position * (m.head_dim / 2);
  void* hc = nullptr;
  if (cudaMalloc(&hc, n * sizeof(__half2)) != cudaSuccess) return fail(SCD_E_NOMEM, "cudaMalloc(rope fp16)");
  p->allocs.push_back(hc);
  rope_to_half_kernel<<<1024, 256, 0, s>>>(p->rope_cons, (__half2*)hc, n);
  p->rope_cons_h = hc;
  if (p->rope_prod == p->rope_cons) {
    p->rope_prod_h = hc;
  } else {
    void* hp = nullptr;
    if (cudaMalloc(&hp, n * sizeof(__half2)) != cudaSuccess) return fail(SCD_E_NOMEM, "cudaMalloc(rope fp16)");
    p->allocs.push_back(hp);
    rope_to_half_kernel<<<1024, 256, 0, s>>>(p->rope_prod, (__half2*)hp, n);
    p->rope_prod_h = hp;
  }
  if (cudaGetLastError() != cudaSuccess) return fail(SCD_E_CUDA, "rope_to_half_kernel launch failed");
  return SCD_OK;
}

// ---------------------------------------------------------------------------------
// launch helper
// ---------------------------------------------------------------------------------
template <int EPI, int AMODE>
static scd_status_t launch_tc(const scd_plan_t* p, TcParams& P, cudaStream_t s) {
  P.m_tiles = (P.M + BLOCK_M - 1) / BLOCK_M;
  P.n_tiles = (P.N + P.block_n - 1) / P.block_n;
  P.num_kb = (P.K + BLOCK_K - 1) / BLOCK_K;
  const int total = P.n_segs * P.m_tiles * P.n_tiles;
  if (total <= 0) return SCD_OK;
  const size_t smem = tc_smem_bytes(P.block_n);
  static thread_local size_t configured = 0;   // per instantiation
  if (configured < smem) {
    cudaError_t e = cudaFuncSetAttribute(tc_gemm_kernel<EPI, AMODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return fail(SCD_E_CUDA, "cudaFuncSetAttribute(smem %zu): %s", smem, cudaGetErrorString(e));
    configured = smem;
  }
  const int grid = std::min(total, p->sm_count);
  prof_begin(s);
  tc_gemm_kernel<EPI, AMODE><<<grid, AMODE == A_DEROPE ? 384 : 256, smem, s>>>(P);
  prof_end(s, 100 + 10 * EPI + AMODE);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(SCD_E_CUDA, "tc_gemm_kernel launch: %s", cudaGetErrorString(e));
  count_launch();
  return SCD_OK;
}

static void fill_common(const scd_plan_t* p, const scd_batch_t* b, bool pages, bool producer, TcParams& P) {
  memset(&P, 0, sizeof(P));
  P.b_maps = (const CUtensorMap*)p->tc_bmaps;
  P.batch.cu_seqlens = b->cu_seqlens;
  P.batch.page_table = pages ? b->page_table : nullptr;
  P.batch.pos_offset = b->pos_offset;
  P.batch.n_seqs = b->n_seqs;
  P.batch.total_tokens = b->total_tokens;
  P.batch.max_pages_per_seq = b->max_pages_per_seq;
  P.batch.block_size = p->model.block_size;
  P.rope_h = (const __half2*)(producer ? p->rope_prod_h : p->rope_cons_h);
  P.head_dim = p->model.head_dim;
  P.rope_style = p->model.rope_style;
  P.act = p->model.patch_act;
  P.code_dtype = p->model.code_dtype;
  P.M = b->total_tokens;
}

// ---------------------------------------------------------------------------------
// scd_encode on tensor cores: one launch per (branch kind, chunk of <= 64 segments)
// ---------------------------------------------------------------------------------
scd_status_t tc_encode(const scd_plan_t* p, const scd_batch_t* batch, const scd_src_t* src, void* codes,
                       const size_t* off, const size_t* soff, cudaStream_t s) {
  const scd_model_desc_t& m = p->model;
  const int T = batch->total_tokens;
  const bool e4 = m.code_dtype == SCD_E4M3_ROWSCALE;
  scd_status_t st;
  if ((src->kv_token_stride % 8) || (src->kv_head_stride % 8) || (src->h_token_stride % 8))
    return fail(SCD_E_ALIGN, "source strides must be multiples of 8 elements on the bf16 path");
  const bool dense_kv = src->kv_head_stride == m.head_dim;
  if (!dense_kv && (m.head_dim % BLOCK_K))
    return fail(SCD_E_UNSUPPORTED, "head-strided K/V needs head_dim %% 64 == 0");

  size_t i = 0;
  const size_t nseg = p->segs.size();
  while (i < nseg) {
    // a launch = run of segments with the same branch, rank and width
    size_t j = i;
    while (j < nseg && j - i < (size_t)TC_MAX_SEGS && p->segs[j].branch == p->segs[i].branch &&
           p->segs[j].rank == p->segs[i].rank)
      ++j;
    const SegPlan& s0 = p->segs[i];
    static thread_local TcParams P;
    fill_common(p, batch, false, true, P);
    P.n_segs = (int)(j - i);
    P.N = s0.rank;
    P.K = s0.width;
    P.block_n = pick_block_n_cover(s0.rank);
    P.a_kb_per_head = (s0.branch != SCD_BRANCH_H && !dense_kv) ? m.head_dim / BLOCK_K : 0;
    for (size_t q = i; q < j; ++q) {
      const SegPlan& sp = p->segs[q];
      const int key = sp.layer * 3 + sp.branch;
      TcSeg& sg = P.segs[q - i];
      sg.col_vec = sp.enc_c;
      sg.out0 = (char*)codes + off[key];
      sg.aux = e4 ? (float*)((char*)codes + soff[key]) : nullptr;
      sg.a_map = (int)(q - i);
      sg.a_z = 0;
      sg.b_map = sp.seg_index;
      CUtensorMap* am = &P.a_maps[q - i];
      if (sp.branch == SCD_BRANCH_H)
        st = make_map(am, src->h[sp.layer], m.d_model, T, 1, (uint64_t)src->h_token_stride * 2,
                      (uint64_t)src->h_token_stride * 2 * T, BLOCK_M, 1);
      else {
        const void* a = sp.branch == SCD_BRANCH_K ? src->k[sp.layer] : src->v[sp.layer];
        if (dense_kv)
          st = make_map(am, a, p->D, T, 1, (uint64_t)src->kv_token_stride * 2, (uint64_t)src->kv_token_stride * 2 * T,
                        BLOCK_M, 1);
        else
          st = make_map(am, a, m.head_dim, m.n_kv_heads, T, (uint64_t)src->kv_head_stride * 2,
                        (uint64_t)src->kv_token_stride * 2, 1, BLOCK_M);
      }
      if (st != SCD_OK) return st;
    }
    if (s0.branch == SCD_BRANCH_K && m.k_is_roped) {
      if (m.rope_style != SCD_ROPE_HALF)
        return fail(SCD_E_UNSUPPORTED, "deRoPE-on-load implements the HALF pairing only on the bf16 path");
      st = launch_tc<EPI_CODES, A_DEROPE>(p, P, s);
    } else {
      st = launch_tc<EPI_CODES, A_PLAIN>(p, P, s);
    }
    if (st != SCD_OK) return st;
    i = j;
  }
  return SCD_OK;
}

// ---------------------------------------------------------------------------------
// scd_reuse_decode on tensor cores
// ---------------------------------------------------------------------------------
scd_status_t tc_reuse_decode(const scd_plan_t* p, const scd_batch_t* batch, const void* codes,
                             const scd_paged_kv_t* kv, const size_t* off, const size_t* soff, cudaStream_t s) {
  const scd_model_desc_t& m = p->model;
  const int T = batch->total_tokens;
  if (m.code_dtype == SCD_E4M3_ROWSCALE) return fail(SCD_E_UNSUPPORTED, "e4m3 decode on tensor cores: not yet");
  scd_status_t st;
  const int nseg_all = (int)p->segs.size();
  size_t i = 0;
  std::vector<int> reuse;
  for (int q = 0; q < nseg_all; ++q)
    if (p->segs[q].branch != SCD_BRANCH_H) reuse.push_back(q);
  while (i < reuse.size()) {
    size_t j = i;
    while (j < reuse.size() && j - i < (size_t)TC_MAX_SEGS && p->segs[reuse[j]].rank == p->segs[reuse[i]].rank) ++j;
    const SegPlan& s0 = p->segs[reuse[i]];
    static thread_local TcParams P;
    fill_common(p, batch, true, false, P);
    P.n_segs = (int)(j - i);
    P.N = p->D;
    P.K = s0.rank;
    P.block_n = pick_block_n_div(p->D);
    P.split = P.N;
    P.pool_width = p->D;
    // segments of a run are consecutive in the code buffer with a uniform stride: one 3-D map
    const size_t seg_stride = align_up((size_t)T * s0.rank * 2, 128);
    const int key0 = s0.layer * 3 + s0.branch;
    bool uniform = true;
    for (size_t q = i; q < j; ++q) {
      const SegPlan& sp = p->segs[reuse[q]];
      if (off[sp.layer * 3 + sp.branch] != off[key0] + (q - i) * seg_stride) uniform = false;
    }
    if (uniform) {
      if ((st = make_map(&P.a_maps[0], (const char*)codes + off[key0], s0.rank, T, j - i, (uint64_t)s0.rank * 2,
                         seg_stride, BLOCK_M, 1)) != SCD_OK)
        return st;
    }
    for (size_t q = i; q < j; ++q) {
      const SegPlan& sp = p->segs[reuse[q]];
      const int key = sp.layer * 3 + sp.branch;
      TcSeg& sg = P.segs[q - i];
      sg.col_vec = sp.mean_dst;
      sg.out0 = sp.branch == SCD_BRANCH_K ? kv->k_pool[sp.layer] : kv->v_pool[sp.layer];
      sg.rope_cols = (sp.branch == SCD_BRANCH_K && m.rope_on_reuse_k) ? p->D : 0;
      sg.b_map = nseg_all + sp.seg_index;
      if (uniform) {
        sg.a_map = 0;
        sg.a_z = (int)(q - i);
      } else {
        sg.a_map = (int)(q - i);
        sg.a_z = 0;
        if ((st = make_map(&P.a_maps[q - i], (const char*)codes + off[key], sp.rank, T, 1, (uint64_t)sp.rank * 2,
                           seg_stride, BLOCK_M, 1)) != SCD_OK)
          return st;
      }
    }
    if ((st = launch_tc<EPI_KV, A_PLAIN>(p, P, s)) != SCD_OK) return st;
    i = j;
  }
  (void)soff;
  return SCD_OK;
}

// ---------------------------------------------------------------------------------
// scd_patch on tensor cores: per PATCH layer  GEMM-1 (aligner in) -> GEMM-2 (aligner out,
// row sum of squares) -> GEMM-3 ([gamma.W_k | gamma.W_v], row scale, RoPE, paged write)
// ---------------------------------------------------------------------------------
scd_status_t tc_patch(const scd_plan_t* p, const scd_batch_t* batch, const void* codes, const scd_paged_kv_t* kv,
                      void* ws_act, void* ws_u, float* ws_ss, const size_t* off, const size_t* soff, cudaStream_t s) {
  const scd_model_desc_t& m = p->model;
  const int T = batch->total_tokens, d = m.d_model, D = p->D;
  if (m.code_dtype == SCD_E4M3_ROWSCALE) return fail(SCD_E_UNSUPPORTED, "e4m3 patch on tensor cores: not yet");
  const bool rms = m.patch_norm == SCD_NORM_RMS;
  const int nseg = (int)p->segs.size();
  scd_status_t st;
  for (size_t j = 0; j < p->patches.size(); ++j) {
    const PatchPlan& pp = p->patches[j];
    const int key = pp.layer * 3 + SCD_BRANCH_H;
    static thread_local TcParams P;
    // GEMM-1: [T, r_h] x [r_h, d_a]
    fill_common(p, batch, true, false, P);
    P.n_segs = 1; P.N = pp.d_a; P.K = pp.r_h; P.block_n = pick_block_n_cover(pp.d_a);
    if ((st = make_map(&P.a_maps[0], (const char*)codes + off[key], pp.r_h, T, 1, (uint64_t)pp.r_h * 2,
                       align_up((size_t)T * pp.r_h * 2, 128), BLOCK_M, 1)) != SCD_OK) return st;
    P.segs[0].col_vec = pp.b1; P.segs[0].out0 = ws_act; P.segs[0].b_map = 2 * nseg + 3 * (int)j;
    if ((st = launch_tc<EPI_ACT, A_PLAIN>(p, P, s)) != SCD_OK) return st;
    // GEMM-2: [T, d_a] x [d_a, d]
    fill_common(p, batch, true, false, P);
    P.n_segs = 1; P.N = d; P.K = pp.d_a; P.block_n = pick_block_n_cover(d);
    if ((st = make_map(&P.a_maps[0], ws_act, pp.d_a, T, 1, (uint64_t)pp.d_a * 2, (uint64_t)pp.d_a * 2 * T, BLOCK_M, 1)) != SCD_OK) return st;
    P.segs[0].col_vec = pp.b2; P.segs[0].out0 = ws_u; P.segs[0].aux = rms ? ws_ss : nullptr;
    P.segs[0].b_map = 2 * nseg + 3 * (int)j + 1;
    const int n_partials = (d + P.block_n - 1) / P.block_n;
    if ((st = launch_tc<EPI_U, A_PLAIN>(p, P, s)) != SCD_OK) return st;
    // GEMM-3: [T, d] x [d, 2D]
    fill_common(p, batch, true, false, P);
    P.n_segs = 1; P.N = 2 * D; P.K = d; P.block_n = pick_block_n_div(D);
    P.split = D; P.pool_width = D; P.n_partials = n_partials; P.rms_dim = d; P.rms_eps = m.rms_eps;
    if ((st = make_map(&P.a_maps[0], ws_u, d, T, 1, (uint64_t)d * 2, (uint64_t)d * 2 * T, BLOCK_M, 1)) != SCD_OK) return st;
    P.segs[0].col_vec = pp.bkv; P.segs[0].out0 = kv->k_pool[pp.layer]; P.segs[0].out1 = kv->v_pool[pp.layer];
    P.segs[0].rowscale_in = rms ? ws_ss : nullptr; P.segs[0].rope_cols = D;
    P.segs[0].b_map = 2 * nseg + 3 * (int)j + 2;
    if ((st = launch_tc<EPI_KV, A_PLAIN>(p, P, s)) != SCD_OK) return st;
  }
  (void)soff;
  return SCD_OK;
}

}  // namespace scd
