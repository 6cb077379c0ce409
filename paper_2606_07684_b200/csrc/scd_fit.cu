// Offline REUSE calibration fit on the GPU: stack-SVD of X = [A B] and the ridge encoder,
// PAPER.md:129-139 (section 4.3.1, Eq. 6-7), App. F.1 :583-586; Table 6 :602 gives the paper's cost (905.5 s).
// Readings U4 / U2: Z = X V_r, W_dec = V_r^T split in halves, lam = lam_rel tr(A^T A) / W,
// optional centring.  oracle/fit_oracle.py restates the definition with library SVD / solve.
//
// Everything the fit needs is a function of the Gram matrix G = X^T X (2W x 2W), so the N-row sample is read once:
//
//   1. fit_transpose_kernel   X = [A B] (bf16, [N, W] each) -> Xt [2W, N] K-major, zero-padded; fit_colsum_kernel: fp64
//                             column sums (means)
//   2. fit_gram_kernel        G = Xt Xt^T on tcgen05: bf16 x bf16 products are exact in fp32; a TMEM accumulator takes
//                             at most GRAM_CHUNK_KB k-blocks (4096 samples) and is then added into the fp64 matrix by the
//                             CTA that owns the output tile (deterministic, no atomics), so rounding does not grow with N
//   3. fit_center_kernel      G <- (G + G^T) / 2 - N mu mu^T   (fp64)
//   4. jacobi_step_kernel     one-sided (Hestenes) Jacobi on G in fp64, round-robin pair schedule, n/2 CTAs per step,
//                             n - 1 steps per sweep: at convergence row i = lambda_i v_i
//   5. rank / extract         eigenvalues sorted, V_r = top-r eigenvectors, sigma = sqrt(lambda)
//   6. ridge                  (G_AA + lam I)^-1 G_A: V_r through the same Jacobi solver on G_AA (Q Lambda Q^T) and three
//                             small fp64 GEMMs
#include <algorithm>
#include <cmath>
#include <cstring>

#include "scd_tc_common.cuh"

namespace scd {
namespace {

// ---------------------------------------------------------------------------------
// 1. transpose + column sums
// ---------------------------------------------------------------------------------
// Xt[c][n] = X[n][c] for c in [0, 2W): c < W from A, else from B.  32 x 32 tiles through shared memory; columns
// n in [N, Np) are written as zeros (the Gram kernel's k-blocks run to Np).
__global__ void __launch_bounds__(256) fit_transpose_kernel(const __nv_bfloat16* __restrict__ a, const __nv_bfloat16* __restrict__ b,
                                                            long long row_stride, long long N, long long Np, int W,
                                                            __nv_bfloat16* __restrict__ xt) {
  __shared__ __nv_bfloat16 tile[32][33];
  const long long n0 = (long long)blockIdx.x * 32;
  const int c0 = blockIdx.y * 32;                    // column of X = row of Xt
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8
  for (int i = ty; i < 32; i += 8) {
    const long long n = n0 + i;
    const int c = c0 + tx;
    __nv_bfloat16 v = __float2bfloat16_rn(0.0f);
    if (n < N && c < 2 * W) v = c < W ? a[n * row_stride + c] : b[n * row_stride + (c - W)];
    tile[i][tx] = v;
  }
  __syncthreads();
  for (int i = ty; i < 32; i += 8) {
    const int c = c0 + i;
    const long long n = n0 + tx;
    if (c < 2 * W && n < Np) xt[(long long)c * Np + n] = tile[tx][i];
  }
}

__device__ __forceinline__ double block_sum(double v, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[w] = v;
  __syncthreads();
  double s = 0.0;
  for (int i = 0; i < nw; ++i) s += red[i];
  return s;
}

// colsum[c] = sum_n Xt[c][n]  (fp64; one CTA per row of Xt)
__global__ void __launch_bounds__(256) fit_colsum_kernel(const __nv_bfloat16* __restrict__ xt, long long Np, double* __restrict__ colsum) {
  __shared__ double red[8];
  const __nv_bfloat16* row = xt + (long long)blockIdx.x * Np;
  double s = 0.0;
  for (long long n = threadIdx.x; n < Np; n += 256) s += (double)__bfloat162float(row[n]);
  s = block_sum(s, red);
  if (threadIdx.x == 0) colsum[blockIdx.x] = s;
}

// ---------------------------------------------------------------------------------
// 3. symmetrise + centre:  Gc[i][j] = U[min(i,j)][max(i,j)] - colsum_i colsum_j / N   (centre != 0), U = the two partials' sum
// ---------------------------------------------------------------------------------
__global__ void fit_center_kernel(const double* __restrict__ g, const double* __restrict__ colsum, double inv_n, int center, int n,
                                  double* __restrict__ gc) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
  if (j >= n) return;
  // the Gram kernel fills the tiles that touch the upper triangle, as two split-K partials: entry (min, max) of their sum
  const size_t at = i <= j ? (size_t)i * n + j : (size_t)j * n + i;
  double v = g[at] + g[(size_t)n * n + at];
  if (center) v -= colsum[i] * colsum[j] * inv_n;
  gc[(size_t)i * n + j] = v;
}

// dst [m x m] = src[:m, :m] of an [n x n] matrix
__global__ void fit_copy_block_kernel(const double* __restrict__ src, int n, int m, double* __restrict__ dst) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
  if (j < m) dst[(size_t)i * m + j] = src[(size_t)i * n + j];
}

// ---------------------------------------------------------------------------------
// 4. one-sided Jacobi, one rotation per CTA
// ---------------------------------------------------------------------------------
constexpr int JAC_THREADS = 256;
constexpr int JAC_PER_THREAD = 8;            // n <= 2048

// Round-robin (circle) schedule over n players (n even): in step s player n-1 meets s, and (s + i) mod (n - 1) meets
// (s - i) mod (n - 1) for i = 1 .. n/2 - 1: every pair meets exactly once per sweep of n - 1 steps.
__device__ __forceinline__ void jacobi_pair(int n, int step, int i, int& p, int& q) {
  const int m = n - 1;
  if (i == 0) { p = m; q = step % m; }
  else { p = (step + i) % m; q = (step - i + m) % m; }
  if (p > q) { const int t = p; p = q; q = t; }
}

// u: [n][n] fp64, "column" k of the matrix being orthogonalised is the contiguous row u[k][:].  rotated: incremented
// when a rotation was applied (the host stops when a sweep applied none).
__global__ void __launch_bounds__(JAC_THREADS) jacobi_step_kernel(double* __restrict__ u, int n, int step, double tol, int* __restrict__ rotated) {
  __shared__ double red[3][JAC_THREADS / 32];
  int p, q;
  jacobi_pair(n, step, blockIdx.x, p, q);
  double* up = u + (size_t)p * n;
  double* uq = u + (size_t)q * n;
  double xp[JAC_PER_THREAD], xq[JAC_PER_THREAD];
  double a = 0.0, b = 0.0, c = 0.0;
#pragma unroll
  for (int k = 0; k < JAC_PER_THREAD; ++k) {
    const int j = threadIdx.x + k * JAC_THREADS;
    xp[k] = j < n ? up[j] : 0.0;
    xq[k] = j < n ? uq[j] : 0.0;
    a = fma(xp[k], xp[k], a);
    b = fma(xq[k], xq[k], b);
    c = fma(xp[k], xq[k], c);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
    c += __shfl_xor_sync(0xffffffffu, c, o);
  }
  if ((threadIdx.x & 31) == 0) {
    red[0][threadIdx.x >> 5] = a;
    red[1][threadIdx.x >> 5] = b;
    red[2][threadIdx.x >> 5] = c;
  }
  __syncthreads();
  a = b = c = 0.0;
#pragma unroll
  for (int w = 0; w < JAC_THREADS / 32; ++w) { a += red[0][w]; b += red[1][w]; c += red[2][w]; }
  if (c == 0.0 || fabs(c) <= tol * sqrt(a * b)) return;          // already orthogonal (same decision in every thread)
  // rotation that zeroes <u_p', u_q'>:  zeta = (b - a) / 2c,  t = sign(zeta) / (|zeta| + sqrt(1 + zeta^2))
  const double zeta = (b - a) / (2.0 * c);
  const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
  const double cs = 1.0 / sqrt(1.0 + t * t), sn = cs * t;
#pragma unroll
  for (int k = 0; k < JAC_PER_THREAD; ++k) {
    const int j = threadIdx.x + k * JAC_THREADS;
    if (j < n) {
      up[j] = cs * xp[k] - sn * xq[k];
      uq[j] = sn * xp[k] + cs * xq[k];
    }
  }
  if (threadIdx.x == 0) atomicAdd(rotated, 1);
}

// ---------------------------------------------------------------------------------
// 5. eigenvalues (row norms), descending rank, normalised eigenvectors
// ---------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) fit_row_norm_kernel(const double* __restrict__ u, int n, double* __restrict__ lam) {
  __shared__ double red[8];
  const double* row = u + (size_t)blockIdx.x * n;
  double s = 0.0;
  for (int j = threadIdx.x; j < n; j += 256) s = fma(row[j], row[j], s);
  s = block_sum(s, red);
  if (threadIdx.x == 0) lam[blockIdx.x] = sqrt(s);
}
// order[k] = index of the k-th largest eigenvalue (ties: lower index first)
__global__ void fit_rank_kernel(const double* __restrict__ lam, int n, int* __restrict__ order) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double li = lam[i];
  int rank = 0;
  for (int j = 0; j < n; ++j) {
    const double lj = lam[j];
    rank += (lj > li || (lj == li && j < i)) ? 1 : 0;
  }
  order[rank] = i;
}
// v[k][:] = u[order[k]][:] / lam[order[k]] for k < r;  lam_sorted[k] = lam[order[k]]  (k < n_sorted)
__global__ void fit_extract_kernel(const double* __restrict__ u, const double* __restrict__ lam, const int* __restrict__ order, int n,
                                   double* __restrict__ v, double* __restrict__ lam_sorted) {
  const int k = blockIdx.y, src = order[k];
  const double l = lam[src];
  const double inv = l > 0.0 ? 1.0 / l : 0.0;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j < n) v[(size_t)k * n + j] = u[(size_t)src * n + j] * inv;
  if (j == 0) lam_sorted[k] = l;
}

// ---------------------------------------------------------------------------------
// 6. small fp64 GEMM with general strides:  C[i][k] = rowscale_i * sum_j A[i sa_i + j sa_j] B[j sb_j + k sb_k]
//    rowscale_i = 1 / (shift_vec[i] + *shift) when shift_vec != null
// ---------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) fit_dgemm_kernel(const double* __restrict__ A, long long sa_i, long long sa_j, const double* __restrict__ B,
                                                        long long sb_j, long long sb_k, double* __restrict__ C, int M, int N, int K,
                                                        const double* __restrict__ shift_vec, const double* __restrict__ shift) {
  __shared__ double As[16][17], Bs[16][17];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int i = blockIdx.y * 16 + ty, k = blockIdx.x * 16 + tx;
  double acc = 0.0;
  for (int j0 = 0; j0 < K; j0 += 16) {
    As[ty][tx] = (i < M && j0 + tx < K) ? A[i * sa_i + (long long)(j0 + tx) * sa_j] : 0.0;
    Bs[ty][tx] = (j0 + ty < K && k < N) ? B[(long long)(j0 + ty) * sb_j + k * sb_k] : 0.0;
    __syncthreads();
#pragma unroll
    for (int j = 0; j < 16; ++j) acc = fma(As[ty][j], Bs[j][tx], acc);
    __syncthreads();
  }
  if (i < M && k < N) {
    if (shift_vec) acc /= (shift_vec[i] + *shift);
    C[(size_t)i * N + k] = acc;
  }
}

// lam_ridge = lam_rel * trace(G_AA) / W
__global__ void fit_ridge_lambda_kernel(const double* __restrict__ gc, int n, int W, double lam_rel, double* __restrict__ out) {
  __shared__ double red[8];
  double s = 0.0;
  for (int i = threadIdx.x; i < W; i += blockDim.x) s += gc[(size_t)i * n + i];
  s = block_sum(s, red);
  if (threadIdx.x == 0) *out = lam_rel * s / (double)W;
}

// fp64 [rows][cols] (row pitch ld, column offset c0) -> out dtype, dense [rows][cols]
__global__ void fit_store_kernel(const double* __restrict__ src, int ld, int c0, int rows, int cols, void* __restrict__ dst, int out_dtype,
                                 int take_sqrt, double scale) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
  if (j >= cols) return;
  double v = src[(size_t)i * ld + c0 + j] * scale;
  if (take_sqrt) v = sqrt(v > 0.0 ? v : 0.0);
  if (out_dtype == SCD_F32) ((float*)dst)[(size_t)i * cols + j] = (float)v;
  else ((__nv_bfloat16*)dst)[(size_t)i * cols + j] = __double2bfloat16(v);
}

}  // namespace
}  // namespace scd

// ---------------------------------------------------------------------------------
// 2. Gram matrix on tcgen05:  G[2W, 2W] (fp64) = Xa Xb^T,  Xa, Xb: [2W, Np] bf16 K-major (the same matrix for bf16 states)
// ---------------------------------------------------------------------------------
namespace scd {
namespace {

constexpr int GRAM_BLOCK_N = 256;
constexpr int GRAM_STAGES = 4;
constexpr int GRAM_B_STAGE_BYTES = GRAM_BLOCK_N * BLOCK_K * 2;        // 32 KB
constexpr int GRAM_CHUNK_KB = 64;                                      // k-blocks per TMEM accumulation (4096 samples)
constexpr int GRAM_EPI_WARPS = 8;                                      // two per TMEM lane quadrant (column halves)
constexpr int GRAM_THREADS = (2 + GRAM_EPI_WARPS) * 32;                // TMA, MMA, epilogue
constexpr int GRAM_MAX_TILES = 80;                                     // tiles touching the upper triangle at n = 2048: 72
constexpr int GRAM_SPLIT = 2;                                          // split-K partials (each its own fp64 matrix)

struct GramParams {
  CUtensorMap map_a, map_b;
  double* g;             // GRAM_SPLIT matrices [n][n]
  int n;                 // 2W
  int num_kb;            // Np / 64
  int n_tiles_kept;      // tiles (m, n) with m <= 2 n + 1: G is symmetric, the rest is mirrored afterwards
  uint8_t tile_m[GRAM_MAX_TILES], tile_n[GRAM_MAX_TILES];
};

struct __align__(8) GramBarriers {
  uint64_t full[GRAM_STAGES], empty[GRAM_STAGES];
  uint64_t tmem_full[2], tmem_empty[2];
  uint32_t tmem_base;
};

constexpr size_t GRAM_SMEM = 1024 + (size_t)GRAM_STAGES * (A_STAGE_BYTES + GRAM_B_STAGE_BYTES) + sizeof(GramBarriers);

__global__ void __launch_bounds__(GRAM_THREADS, 1) fit_gram_kernel(const __grid_constant__ GramParams P) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t* smem_a = smem;
  uint8_t* smem_b = smem + GRAM_STAGES * A_STAGE_BYTES;
  GramBarriers* bars = (GramBarriers*)(smem_b + GRAM_STAGES * GRAM_B_STAGE_BYTES);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // work item = (kept tile, split-K half): item -> tile item / 2, k-blocks [kb_lo, kb_hi) of half item % 2
  const int total_items = P.n_tiles_kept * GRAM_SPLIT;
  const int kb_half = (P.num_kb + GRAM_SPLIT - 1) / GRAM_SPLIT;

  if (warp == 1 && lane == 0) {
    for (int s = 0; s < GRAM_STAGES; ++s) {
      ptx::mbar_init(&bars->full[s], 1);
      ptx::mbar_init(&bars->empty[s], 1);
    }
    for (int a = 0; a < 2; ++a) {
      ptx::mbar_init(&bars->tmem_full[a], 1);
      ptx::mbar_init(&bars->tmem_empty[a], GRAM_EPI_WARPS);
    }
    ptx::fence_barrier_init();
  }
  if (warp == 0) {
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
      for (int item = blockIdx.x; item < total_items; item += gridDim.x) {
        const int t = item / GRAM_SPLIT, half = item - t * GRAM_SPLIT;
        const int m0 = P.tile_m[t] * BLOCK_M, n0 = P.tile_n[t] * GRAM_BLOCK_N;
        const int kb_lo = half * kb_half, kb_hi = min(P.num_kb, kb_lo + kb_half);
        for (int kb = kb_lo; kb < kb_hi; ++kb) {
          ptx::mbar_wait_suspend(&bars->empty[stage], phase ^ 1);
          ptx::mbar_expect_tx(&bars->full[stage], A_STAGE_BYTES + GRAM_B_STAGE_BYTES);
          ptx::tma_load_3d(smem_a + stage * A_STAGE_BYTES, &P.map_a, &bars->full[stage], kb * BLOCK_K, m0, 0);
          ptx::tma_load_3d(smem_b + stage * GRAM_B_STAGE_BYTES, &P.map_b, &bars->full[stage], kb * BLOCK_K, n0, 0);
          ptx::tma_load_3d(smem_b + stage * GRAM_B_STAGE_BYTES + A_STAGE_BYTES, &P.map_b, &bars->full[stage], kb * BLOCK_K, n0 + 128, 0);
          if (++stage == GRAM_STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ============================== MMA issuer ==============================
    if (lane == 0) {
      const uint32_t idesc = ptx::umma_idesc_bf16(BLOCK_M, GRAM_BLOCK_N);
      int stage = 0, it = 0;
      uint32_t phase = 0;
      for (int item = blockIdx.x; item < total_items; item += gridDim.x) {
        const int half = item % GRAM_SPLIT;
        const int kb_lo = half * kb_half, kb_hi = min(P.num_kb, kb_lo + kb_half);
        for (int c0 = kb_lo; c0 < kb_hi; c0 += GRAM_CHUNK_KB, ++it) {
          const int acc = it & 1;
          ptx::mbar_wait_suspend(&bars->tmem_empty[acc], ((it >> 1) & 1) ^ 1);
          ptx::tc_fence_after();
          const uint32_t d_tmem = tmem_base + (uint32_t)(acc * GRAM_BLOCK_N);
          const int c1 = min(kb_hi, c0 + GRAM_CHUNK_KB);
          for (int kb = c0; kb < c1; ++kb) {
            ptx::mbar_wait_suspend(&bars->full[stage], phase);
            ptx::tc_fence_after();
            const uint64_t da = ptx::umma_desc_sw128(ptx::smem_u32(smem_a + stage * A_STAGE_BYTES));
            const uint64_t db = ptx::umma_desc_sw128(ptx::smem_u32(smem_b + stage * GRAM_B_STAGE_BYTES));
#pragma unroll
            for (int k = 0; k < BLOCK_K / 16; ++k)
              ptx::mma_bf16(d_tmem, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, (kb > c0) || k != 0);
            ptx::mma_commit(&bars->empty[stage]);
            if (++stage == GRAM_STAGES) { stage = 0; phase ^= 1; }
          }
          ptx::mma_commit(&bars->tmem_full[acc]);
        }
      }
    }
  } else {
    // ============================== epilogue: partial G tile (+)= chunk accumulator, fp64 ==============================
    const int q = warp & 3;                           // TMEM lane quadrant this warp may read
    const int ch = (warp - 2) >> 2;                   // column half of the tile
    int it = 0;
    for (int item = blockIdx.x; item < total_items; item += gridDim.x) {
      const int t = item / GRAM_SPLIT, half = item - t * GRAM_SPLIT;
      const int m0 = P.tile_m[t] * BLOCK_M, n0 = P.tile_n[t] * GRAM_BLOCK_N;
      const int kb_lo = half * kb_half, kb_hi = min(P.num_kb, kb_lo + kb_half);
      const int row = m0 + q * 32 + lane;
      double* grow = P.g + (size_t)half * P.n * P.n + (size_t)row * P.n + n0;
      if (kb_lo >= kb_hi) {                           // an empty half (fewer k-blocks than halves): its partial is zero
        if (row < P.n)
          for (int c = ch * 128; c < ch * 128 + 128 && n0 + c < P.n; ++c) grow[c] = 0.0;
        continue;
      }
      for (int c0 = kb_lo; c0 < kb_hi; c0 += GRAM_CHUNK_KB, ++it) {
        const int acc = it & 1;
        ptx::mbar_wait_suspend(&bars->tmem_full[acc], (it >> 1) & 1);
        ptx::tc_fence_after();
        const uint32_t t_row = tmem_base + (uint32_t)(acc * GRAM_BLOCK_N) + ((uint32_t)(q * 32) << 16);
        for (int c = ch * 128; c < ch * 128 + 128 && n0 + c < P.n; c += 32) {
          uint32_t r[32];
          ptx::tmem_ld32(t_row + c, r);
          ptx::tmem_ld_wait();
          if (row < P.n) {
#pragma unroll
            for (int j = 0; j < 32; j += 2) {
              if (n0 + c + j < P.n) {               // n is even: columns j, j + 1 are valid together
                double2 v = c0 > kb_lo ? *reinterpret_cast<double2*>(grow + c + j) : make_double2(0.0, 0.0);
                v.x += (double)__uint_as_float(r[j]);
                v.y += (double)__uint_as_float(r[j + 1]);
                *reinterpret_cast<double2*>(grow + c + j) = v;
              }
            }
          }
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&bars->tmem_empty[acc]);
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 0) ptx::tmem_dealloc<TMEM_COLS>(tmem_base);
}

}  // namespace
}  // namespace scd

// ---------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------
namespace scd {
namespace {

constexpr int FIT_MAX_SWEEPS = 60;
constexpr double FIT_JACOBI_TOL = 1e-13;

struct FitLayout {
  long long Np;
  size_t xt, g, u, ga, colsum, lam, lam_sorted, order, v, lam_a, lam_a_sorted, order_a, q, r1, r2, wenc, scal, flag, total;
};

FitLayout fit_layout(int W, int r, long long N) {
  FitLayout L;
  const size_t n = 2 * (size_t)W;
  L.Np = (N + BLOCK_K - 1) / BLOCK_K * BLOCK_K;
  size_t at = 0;
  auto take = [&](size_t bytes) { size_t o = at; at = align_up(at + bytes, 256); return o; };
  L.xt = take(n * (size_t)L.Np * 2);
  L.g = take(n * n * 8 * GRAM_SPLIT);    // split-K partials of the Gram kernel; the first is reused for the centred matrix
  L.u = take(n * n * 8);                 // centred Gram matrix, then the Jacobi iterate
  L.ga = take((size_t)W * W * 8);
  L.colsum = take(n * 8);
  L.lam = take(n * 8);
  L.lam_sorted = take(n * 8);
  L.order = take(n * 4);
  L.v = take((size_t)r * n * 8);         // V_r^T: top-r eigenvectors as rows
  L.lam_a = take((size_t)W * 8);
  L.lam_a_sorted = take((size_t)W * 8);
  L.order_a = take((size_t)W * 4);
  L.q = take((size_t)W * W * 8);         // eigenvectors of G_AA as rows
  L.r1 = take((size_t)W * r * 8);
  L.r2 = take((size_t)W * r * 8);
  L.wenc = take((size_t)W * r * 8);
  L.scal = take(64);
  L.flag = take(64);
  L.total = at;
  return L;
}

scd_status_t check_fit(const scd_fit_desc_t* d, long long N) {
  if (!d) return fail(SCD_E_ARG, "fit: null descriptor");
  if (d->width < 8 || (d->width % 8)) return fail(SCD_E_SHAPE, "fit: width %d must be a positive multiple of 8", d->width);
  if (2 * d->width > JAC_THREADS * JAC_PER_THREAD) return fail(SCD_E_UNSUPPORTED, "fit: width %d > %d", d->width, JAC_THREADS * JAC_PER_THREAD / 2);
  if (d->rank < 1 || d->rank > 2 * d->width) return fail(SCD_E_SHAPE, "fit: rank %d outside [1, 2 * width]", d->rank);
  if (d->state_dtype != SCD_BF16) return fail(SCD_E_UNSUPPORTED, "fit: bf16 states only");
  if (d->out_dtype != SCD_BF16 && d->out_dtype != SCD_F32) return fail(SCD_E_ARG, "fit: out_dtype must be F32 or BF16");
  if (!(d->lam_rel >= 0.0f)) return fail(SCD_E_ARG, "fit: lam_rel must be >= 0");
  if (N < 1) return fail(SCD_E_ARG, "fit: n_rows %lld", N);
  return SCD_OK;
}

#define FIT_LAUNCH_CHECK(what)                                                                  \
  do {                                                                                          \
    cudaError_t _e = cudaGetLastError();                                                        \
    if (_e != cudaSuccess) return fail(SCD_E_CUDA, "%s: %s", what, cudaGetErrorString(_e));     \
    count_launch();                                                                             \
  } while (0)

// one-sided Jacobi to convergence on u [n x n]; returns the number of sweeps (synchronises the stream once per sweep)
scd_status_t jacobi_solve(double* u, int n, int* flag, cudaStream_t s, int* sweeps_out) {
  int sweeps = 0;
  for (; sweeps < FIT_MAX_SWEEPS; ++sweeps) {
    if (cudaMemsetAsync(flag, 0, sizeof(int), s) != cudaSuccess) return fail(SCD_E_CUDA, "fit: memset(flag)");
    for (int step = 0; step < n - 1; ++step) jacobi_step_kernel<<<n / 2, JAC_THREADS, 0, s>>>(u, n, step, FIT_JACOBI_TOL, flag);
    FIT_LAUNCH_CHECK("jacobi_step_kernel");
    int h = 0;
    if (cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess)
      return fail(SCD_E_CUDA, "fit: reading the Jacobi convergence flag: %s", cudaGetErrorString(cudaGetLastError()));
    if (h == 0) { ++sweeps; break; }
  }
  if (sweeps_out) *sweeps_out = sweeps;
  return SCD_OK;
}

}  // namespace
}  // namespace scd

using namespace scd;

extern "C" scd_status_t scd_fit_query(const scd_fit_desc_t* d, int64_t n_rows, size_t* workspace_bytes) {
  scd_status_t st = check_fit(d, n_rows);
  if (st != SCD_OK) return st;
  if (workspace_bytes) *workspace_bytes = fit_layout(d->width, d->rank, n_rows).total;
  return SCD_OK;
}

extern "C" scd_status_t scd_fit_reuse(const scd_fit_desc_t* d, const void* a, const void* b, int64_t n_rows, int64_t row_stride,
                                      void* w_enc, void* w_dec_a, void* w_dec_b, float* mu_a, float* mu_b, float* sigma,
                                      void* workspace, size_t workspace_bytes, int32_t* sweeps, void* stream) {
  reset_launch_count();
  scd_status_t st = check_fit(d, n_rows);
  if (st != SCD_OK) return st;
  if (!a || !b || !w_enc || !w_dec_b || !workspace) return fail(SCD_E_ARG, "fit: null buffer");
  const int W = d->width, r = d->rank, n = 2 * W;
  if (row_stride < W) return fail(SCD_E_ALIGN, "fit: row stride %lld < width %d", (long long)row_stride, W);
  if (d->center && (!mu_a || !mu_b)) return fail(SCD_E_ARG, "fit: centring needs mu_a and mu_b");
  const FitLayout L = fit_layout(W, r, n_rows);
  if (workspace_bytes < L.total) return fail(SCD_E_WORKSPACE, "fit: workspace %zu < %zu bytes", workspace_bytes, L.total);
  if (((uintptr_t)workspace) % 256) return fail(SCD_E_ALIGN, "fit: workspace not 256-byte aligned");
  cudaStream_t s = (cudaStream_t)stream;
  char* ws = (char*)workspace;
  __nv_bfloat16* xt = (__nv_bfloat16*)(ws + L.xt);
  double *g = (double*)(ws + L.g), *u = (double*)(ws + L.u), *ga = (double*)(ws + L.ga), *colsum = (double*)(ws + L.colsum);
  double *lam = (double*)(ws + L.lam), *lam_sorted = (double*)(ws + L.lam_sorted), *v = (double*)(ws + L.v);
  double *lam_a = (double*)(ws + L.lam_a), *lam_a_sorted = (double*)(ws + L.lam_a_sorted), *q = (double*)(ws + L.q);
  double *r1 = (double*)(ws + L.r1), *r2 = (double*)(ws + L.r2), *wenc = (double*)(ws + L.wenc), *scal = (double*)(ws + L.scal);
  int *order = (int*)(ws + L.order), *order_a = (int*)(ws + L.order_a), *flag = (int*)(ws + L.flag);
  if (sweeps) sweeps[0] = sweeps[1] = 0;

  // 1. K-major copy of X = [A B] and its column sums
  {
    dim3 grid((unsigned)((L.Np + 31) / 32), (unsigned)((n + 31) / 32));
    fit_transpose_kernel<<<grid, 256, 0, s>>>((const __nv_bfloat16*)a, (const __nv_bfloat16*)b, row_stride, n_rows, L.Np, W, xt);
    FIT_LAUNCH_CHECK("fit_transpose_kernel");
    fit_colsum_kernel<<<n, 256, 0, s>>>(xt, L.Np, colsum);
    FIT_LAUNCH_CHECK("fit_colsum_kernel");
  }
  // 2. Gram matrix on the tensor cores
  {
    static thread_local GramParams P;
    memset(&P, 0, sizeof(P));
    if ((st = tc_make_map_2d_bf16(&P.map_a, xt, (uint64_t)L.Np, (uint64_t)n, (uint64_t)L.Np * 2, BLOCK_M)) != SCD_OK) return st;
    P.map_b = P.map_a;
    P.g = g;
    P.n = n;
    P.num_kb = (int)(L.Np / BLOCK_K);
    const int mt = (n + BLOCK_M - 1) / BLOCK_M, nt = (n + GRAM_BLOCK_N - 1) / GRAM_BLOCK_N;
    P.n_tiles_kept = 0;
    for (int tn = 0; tn < nt; ++tn)
      for (int tm = 0; tm < mt && tm <= 2 * tn + 1; ++tm) {
        if (P.n_tiles_kept >= GRAM_MAX_TILES) return fail(SCD_E_UNSUPPORTED, "fit: too many Gram tiles");
        P.tile_m[P.n_tiles_kept] = (uint8_t)tm;
        P.tile_n[P.n_tiles_kept] = (uint8_t)tn;
        ++P.n_tiles_kept;
      }
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    static std::atomic<int> configured[SCD_MAX_DEVICES];
    if (dev >= 0 && dev < SCD_MAX_DEVICES && !configured[dev].load()) {
      cudaError_t e = cudaFuncSetAttribute(fit_gram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GRAM_SMEM);
      if (e != cudaSuccess) return fail(SCD_E_CUDA, "cudaFuncSetAttribute(gram smem): %s", cudaGetErrorString(e));
      configured[dev].store(1);
    }
    const int items = P.n_tiles_kept * GRAM_SPLIT;
    prof_begin(s);
    fit_gram_kernel<<<std::min(items, std::max(sms, 1)), GRAM_THREADS, GRAM_SMEM, s>>>(P);
    prof_end(s, SCD_PROF_FIT_GRAM);
    FIT_LAUNCH_CHECK("fit_gram_kernel");
  }
  // 3. symmetrise, centre
  {
    dim3 grid((n + 255) / 256, n);
    fit_center_kernel<<<grid, 256, 0, s>>>(g, colsum, 1.0 / (double)n_rows, d->center ? 1 : 0, n, u);
    FIT_LAUNCH_CHECK("fit_center_kernel");
    // keep the centred matrix in g: the ridge step needs G_A: after u has been rotated away
    if (cudaMemcpyAsync(g, u, (size_t)n * n * 8, cudaMemcpyDeviceToDevice, s) != cudaSuccess) return fail(SCD_E_CUDA, "fit: copy of the centred Gram matrix");
    dim3 grid_a((W + 255) / 256, W);
    fit_copy_block_kernel<<<grid_a, 256, 0, s>>>(g, n, W, ga);
    FIT_LAUNCH_CHECK("fit_copy_block_kernel");
  }
  // 4-5. eigen-decomposition of the joint Gram matrix: V_r, sigma
  if ((st = jacobi_solve(u, n, flag, s, sweeps)) != SCD_OK) return st;
  fit_row_norm_kernel<<<n, 256, 0, s>>>(u, n, lam);
  FIT_LAUNCH_CHECK("fit_row_norm_kernel");
  fit_rank_kernel<<<(n + 255) / 256, 256, 0, s>>>(lam, n, order);
  FIT_LAUNCH_CHECK("fit_rank_kernel");
  {
    dim3 grid((n + 255) / 256, r);
    fit_extract_kernel<<<grid, 256, 0, s>>>(u, lam, order, n, v, lam_sorted);
    FIT_LAUNCH_CHECK("fit_extract_kernel");
  }
  // 6. ridge encoder: G_AA = Q Lam Q^T;  W_enc = Q (Lam + lam I)^-1 Q^T (G_A: V_r)
  if ((st = jacobi_solve(ga, W, flag, s, sweeps ? sweeps + 1 : nullptr)) != SCD_OK) return st;
  fit_row_norm_kernel<<<W, 256, 0, s>>>(ga, W, lam_a);
  FIT_LAUNCH_CHECK("fit_row_norm_kernel");
  fit_rank_kernel<<<(W + 255) / 256, 256, 0, s>>>(lam_a, W, order_a);
  FIT_LAUNCH_CHECK("fit_rank_kernel");
  {
    dim3 grid((W + 255) / 256, W);
    fit_extract_kernel<<<grid, 256, 0, s>>>(ga, lam_a, order_a, W, q, lam_a_sorted);
    FIT_LAUNCH_CHECK("fit_extract_kernel");
    fit_ridge_lambda_kernel<<<1, 256, 0, s>>>(g, n, W, (double)d->lam_rel, scal);
    FIT_LAUNCH_CHECK("fit_ridge_lambda_kernel");
    dim3 gg((r + 15) / 16, (W + 15) / 16);
    // R1[i][k] = sum_j Gc[i][j] V[k][j]          (W x r, K = 2W)
    fit_dgemm_kernel<<<gg, 256, 0, s>>>(g, n, 1, v, 1, n, r1, W, r, n, nullptr, nullptr);
    FIT_LAUNCH_CHECK("fit_dgemm_kernel");
    // R2[m][k] = (sum_i Q[m][i] R1[i][k]) / (Lam_m + lam)
    fit_dgemm_kernel<<<gg, 256, 0, s>>>(q, W, 1, r1, r, 1, r2, W, r, W, lam_a_sorted, scal);
    FIT_LAUNCH_CHECK("fit_dgemm_kernel");
    // W_enc[i][k] = sum_m Q[m][i] R2[m][k]
    fit_dgemm_kernel<<<gg, 256, 0, s>>>(q, 1, W, r2, r, 1, wenc, W, r, W, nullptr, nullptr);
    FIT_LAUNCH_CHECK("fit_dgemm_kernel");
  }
  // outputs
  {
    dim3 g_enc((r + 127) / 128, W), g_dec((W + 127) / 128, r);
    fit_store_kernel<<<g_enc, 128, 0, s>>>(wenc, r, 0, W, r, w_enc, d->out_dtype, 0, 1.0);
    if (w_dec_a) fit_store_kernel<<<g_dec, 128, 0, s>>>(v, n, 0, r, W, w_dec_a, d->out_dtype, 0, 1.0);
    fit_store_kernel<<<g_dec, 128, 0, s>>>(v, n, W, r, W, w_dec_b, d->out_dtype, 0, 1.0);
    if (sigma) fit_store_kernel<<<dim3((r + 127) / 128, 1), 128, 0, s>>>(lam_sorted, r, 0, 1, r, sigma, SCD_F32, 1, 1.0);
    if (d->center) {
      fit_store_kernel<<<dim3((W + 127) / 128, 1), 128, 0, s>>>(colsum, n, 0, 1, W, mu_a, SCD_F32, 0, 1.0 / (double)n_rows);
      fit_store_kernel<<<dim3((W + 127) / 128, 1), 128, 0, s>>>(colsum, n, W, 1, W, mu_b, SCD_F32, 0, 1.0 / (double)n_rows);
    }
    FIT_LAUNCH_CHECK("fit_store_kernel");
  }
  return SCD_OK;
}
