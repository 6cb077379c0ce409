// SIMT (CUDA-core) kernels: the fp32 path of the codec (Tiny config, 1e-5 tolerance --
// tensor cores would give TF32 ~1e-3) and a debug path for bf16 states.  One launch per
// GEMM segment; C[M,N] = A[M,K] Bt[N,K]^T with fp32 FFMA accumulation, A-side transforms
// (deRoPE of Eq. 5, code unpacking, exact mean subtraction) applied on load and the
// encode / paged-KV / aligner epilogues fused after the k-loop.
#include "scd_device.cuh"
#include "scd_internal.h"

namespace scd {
namespace {

constexpr int BM = 32, BN = 128, BK = 32, NT = 256;

template <typename TS, int EPI>
__global__ void __launch_bounds__(NT)
simt_gemm_kernel(GemmSeg g, int a_mode, int code_dtype, BatchDev batch, RopeDev rope, int nt_per_block) {
  extern __shared__ float panel[];                  // EPI_CODES + e4m3 only: [BM][N] codes before quantisation
  __shared__ float As[BM][BK + 1];
  __shared__ float Bs[BN][BK + 1];
  __shared__ float Cs[BM][BN + 1];
  __shared__ int s_pos[BM];
  __shared__ long long s_slot[BM];
  __shared__ float s_rowscale[BM];

  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  const int m0 = blockIdx.x * BM;
  const int half = rope.head_dim / 2;

  if (tid < BM) {
    int row = m0 + tid;
    int pos = 0;
    long long slot = -1;
    float rs = 1.0f;
    if (row < g.M) {
      row_to_pos_slot(batch, row, pos, slot);
      if (g.a_scale) rs = g.a_scale[row];
      if (EPI == EPI_KV && g.rowscale_in) {
        float ss = 0.0f;
        for (int p = 0; p < g.n_partials; ++p) ss += g.rowscale_in[(size_t)p * g.M + row];
        rs *= 1.0f / sqrtf(ss / (float)g.rms_dim + g.rms_eps);
      }
    }
    s_pos[tid] = pos;
    s_slot[tid] = slot;
    s_rowscale[tid] = rs;
  }
  __syncthreads();

  const int n_tiles = (g.N + BN - 1) / BN;
  const int nt_begin = blockIdx.y * nt_per_block;
  const int nt_end = min(n_tiles, nt_begin + nt_per_block);
  const bool use_panel = (EPI == EPI_CODES) && code_dtype == SCD_E4M3_ROWSCALE;

  for (int nt = nt_begin; nt < nt_end; ++nt) {
    const int n0 = nt * BN;
    float acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) acc[i][j] = 0.0f;

    for (int k0 = 0; k0 < g.K; k0 += BK) {
      // ---- A tile: 32 x 32, transforms on load ----
#pragma unroll
      for (int i = 0; i < (BM * BK) / NT; ++i) {
        int e = tid + i * NT;
        int r = e / BK, kk = e % BK;
        int row = m0 + r, k = k0 + kk;
        float v = 0.0f;
        if (row < g.M && k < g.K) {
          if (a_mode == A_CODES) {
            v = load_code(g.a, (size_t)row * g.lda + k, code_dtype);
          } else {
            const TS* a = (const TS*)g.a;
            size_t base = (size_t)row * g.lda;
            auto at = [&](int kc) -> float {
              size_t off = g.a_head_stride ? (size_t)(kc / rope.head_dim) * g.a_head_stride + kc % rope.head_dim
                                           : (size_t)kc;
              return to_float(a[base + off]);
            };
            v = at(k);
            if (a_mode == A_DEROPE) {
              int j = k % rope.head_dim;
              int fi, kp;
              bool first;
              rope_partner(rope.style, j, half, fi, kp, first);
              float2 cs = rope.table[(size_t)s_pos[r] * half + fi];
              float w = at(k - j + kp);
              // deRoPE = rotation by -phi:  a' = a cos + b sin ; b' = b cos - a sin
              v = first ? (v * cs.x + w * cs.y) : (v * cs.x - w * cs.y);
            }
          }
          if (g.a_sub) v -= g.a_sub[k];
        }
        As[r][kk] = v;
      }
      // ---- Bt tile: 128 x 32 ----
#pragma unroll
      for (int i = 0; i < (BN * BK) / NT; ++i) {
        int e = tid + i * NT;
        int n = e / BK, kk = e % BK;
        int col = n0 + n, k = k0 + kk;
        Bs[n][kk] = (col < g.N && k < g.K) ? to_float(((const TS*)g.bt)[(size_t)col * g.K + k]) : 0.0f;
      }
      __syncthreads();
#pragma unroll
      for (int kk = 0; kk < BK; ++kk) {
        float a[4], b[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) a[i] = As[ty * 4 + i][kk];
#pragma unroll
        for (int j = 0; j < 4; ++j) b[j] = Bs[tx + 32 * j][kk];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
      }
      __syncthreads();
    }

    // ---- stage the fp32 tile so that RoPE partners / row reductions can see it ----
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) Cs[ty * 4 + i][tx + 32 * j] = acc[i][j];
    __syncthreads();

    // value of element (r, c) after the linear part of the epilogue
    auto lin = [&](int r, int c) -> float {
      int col = n0 + c;
      float v = Cs[r][c] * s_rowscale[r];
      if (g.col_vec) v = (EPI == EPI_CODES) ? v - g.col_vec[col] : v + g.col_vec[col];
      return v;
    };

    if (EPI == EPI_U) {
      // each warp owns 4 rows: store + per-row sum of squares over this n-tile
      for (int i = 0; i < 4; ++i) {
        int r = ty * 4 + i, row = m0 + r;
        float ss = 0.0f;
        for (int c = tx; c < BN; c += 32) {
          int col = n0 + c;
          if (row < g.M && col < g.N) {
            float v = lin(r, c);
            ss += v * v;
            ((TS*)g.out0)[(size_t)row * g.N + col] = from_float<TS>(v);
          }
        }
        ss = warp_sum(ss);
        if (tx == 0 && row < g.M && g.aux) g.aux[(size_t)nt * g.M + row] = ss;
      }
    } else {
      for (int e = tid; e < BM * BN; e += NT) {
        int r = e / BN, c = e % BN;
        int row = m0 + r, col = n0 + c;
        if (row >= g.M || col >= g.N) continue;
        float v = lin(r, c);
        if (EPI == EPI_CODES) {
          if (use_panel) panel[(size_t)r * g.N + col] = v;
          else store_code(g.out0, (size_t)row * g.N + col, v, code_dtype);
        } else if (EPI == EPI_ACT) {
          if (g.act == SCD_ACT_SILU) v = v / (1.0f + expf(-v));
          ((TS*)g.out0)[(size_t)row * g.N + col] = from_float<TS>(v);
        } else {   // EPI_KV
          if (col < g.rope_cols) {
            int j = col % rope.head_dim;
            int fi, jp;
            bool first;
            rope_partner(rope.style, j, half, fi, jp, first);
            float w = lin(r, c - j + jp);
            float2 cs = rope.table[(size_t)s_pos[r] * half + fi];
            // RoPE = rotation by +phi:  a' = a cos - b sin ; b' = b cos + a sin
            v = first ? (v * cs.x - w * cs.y) : (v * cs.x + w * cs.y);
          }
          TS* pool = (TS*)(col < g.split ? g.out0 : g.out1);
          int pc = col < g.split ? col : col - g.split;
          if (s_slot[r] >= 0) pool[(size_t)s_slot[r] * g.pool_width + pc] = from_float<TS>(v);   // -1: page id outside the pool
        }
      }
    }
    __syncthreads();
  }

  if (use_panel) {
    // e4m3 + per-row fp32 scale: s = amax/448 (1 for an all-zero row), q = sat-RNE(z / s)
    for (int i = 0; i < 4; ++i) {
      int r = ty * 4 + i, row = m0 + r;
      if (row >= g.M) continue;
      float amax = 0.0f;
      for (int c = tx; c < g.N; c += 32) amax = fmaxf(amax, fabsf(panel[(size_t)r * g.N + c]));
      amax = warp_max(amax);
      float s = amax > 0.0f ? amax / 448.0f : 1.0f;
      if (tx == 0) g.aux[row] = s;
      for (int c = tx; c < g.N; c += 32)
        ((uint8_t*)g.out0)[(size_t)row * g.N + c] = float_to_e4m3_sat(panel[(size_t)r * g.N + c] / s);
    }
  }
}

template <typename TS>
cudaError_t launch(const GemmSeg& g, int epi, int a_mode, int code_dtype, const BatchDev& batch,
                   const RopeDev& rope, cudaStream_t s) {
  if (g.M <= 0 || g.N <= 0) return cudaSuccess;
  int n_tiles = (g.N + BN - 1) / BN;
  bool panel = epi == EPI_CODES && code_dtype == SCD_E4M3_ROWSCALE;
  dim3 grid((g.M + BM - 1) / BM, panel ? 1 : n_tiles);
  int ntpb = panel ? n_tiles : 1;
  size_t smem = panel ? (size_t)BM * g.N * sizeof(float) : 0;
#define SCD_SIMT_CASE(E)                                                                                      \
  case E: {                                                                                                   \
    if (smem > 0) {                                                                                           \
      cudaError_t e = cudaFuncSetAttribute(simt_gemm_kernel<TS, E>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                           (int)smem);                                                        \
      if (e != cudaSuccess) return e;                                                                         \
    }                                                                                                         \
    prof_begin(s);                                                                                            \
    simt_gemm_kernel<TS, E><<<grid, NT, smem, s>>>(g, a_mode, code_dtype, batch, rope, ntpb);                 \
    prof_end(s, 10 * E + a_mode);                                                                             \
    break;                                                                                                    \
  }
  switch (epi) {
    SCD_SIMT_CASE(EPI_CODES)
    SCD_SIMT_CASE(EPI_KV)
    SCD_SIMT_CASE(EPI_ACT)
    SCD_SIMT_CASE(EPI_U)
    default: return cudaErrorInvalidValue;
  }
#undef SCD_SIMT_CASE
  count_launch();
  return cudaGetLastError();
}

}  // namespace

cudaError_t simt_gemm(const GemmSeg& seg, int epi, int a_mode, int state_dtype, int code_dtype,
                      const BatchDev& batch, const RopeDev& rope, cudaStream_t s) {
  if (state_dtype == SCD_F32) return launch<float>(seg, epi, a_mode, code_dtype, batch, rope, s);
  return launch<__nv_bfloat16>(seg, epi, a_mode, code_dtype, batch, rope, s);
}

}  // namespace scd
