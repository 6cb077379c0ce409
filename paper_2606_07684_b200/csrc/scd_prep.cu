// Plan-time repack kernels: run once per scd_plan (the offline "load artifacts" step,
// PAPER.md:102), never on the hot path.  They bring every B operand of the path's GEMMs
// into K-major [N, K] form, fold the RMSNorm weight into W_k|W_v, project the source
// mean through the encoder in fp64 and tabulate RoPE angles in fp64.
#include <algorithm>

#include "scd_internal.h"

namespace scd {
namespace {

template <typename T> __device__ __forceinline__ float ldf(const T* p, size_t i);
template <> __device__ __forceinline__ float ldf<float>(const float* p, size_t i) { return p[i]; }
template <> __device__ __forceinline__ float ldf<__nv_bfloat16>(const __nv_bfloat16* p, size_t i) {
  return __bfloat162float(p[i]);
}
template <typename T> __device__ __forceinline__ T cvt(float v);
template <> __device__ __forceinline__ float cvt<float>(float v) { return v; }
template <> __device__ __forceinline__ __nv_bfloat16 cvt<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

// dst[c, r] = src[r, c]; 32x32 smem tile, coalesced both ways.
template <typename T>
__global__ void transpose_kernel(const T* __restrict__ src, T* __restrict__ dst, int rows, int cols) {
  __shared__ T tile[32][33];
  int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
  for (int i = threadIdx.y; i < 32; i += blockDim.y) {
    int r = r0 + i, c = c0 + threadIdx.x;
    if (r < rows && c < cols) tile[i][threadIdx.x] = src[(size_t)r * cols + c];
  }
  __syncthreads();
  for (int i = threadIdx.y; i < 32; i += blockDim.y) {
    int c = c0 + i, r = r0 + threadIdx.x;
    if (r < rows && c < cols) dst[(size_t)c * rows + r] = tile[threadIdx.x][i];
  }
}

template <typename T>
__global__ void fold_gamma_kernel(const T* __restrict__ w, const T* __restrict__ gamma, T* __restrict__ dst,
                                  int rows, int cols) {
  size_t n = (size_t)rows * cols;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    float g = gamma ? ldf<T>(gamma, i % cols) : 1.0f;
    dst[i] = cvt<T>(ldf<T>(w, i) * g);
  }
}

// One thread per output n; fp64 accumulation over the width.
template <typename T>
__global__ void mean_proj_kernel(const float* __restrict__ mu, const T* __restrict__ w_enc, float* __restrict__ c,
                                 int width, int rank) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= rank) return;
  double acc = 0.0;
  if (mu)
    for (int k = 0; k < width; ++k) acc += (double)mu[k] * (double)ldf<T>(w_enc, (size_t)k * rank + n);
  c[n] = (float)acc;
}

template <typename T>
__global__ void to_f32_kernel(const T* __restrict__ src, float* __restrict__ dst, int n) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = src ? ldf<T>(src, i) : 0.0f;
}

__global__ void rope_table_kernel(float2* __restrict__ table, int max_position, int head_dim, double theta) {
  int half = head_dim / 2;
  size_t n = (size_t)max_position * half;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    int p = (int)(i / half), j = (int)(i % half);
    double inv_freq = pow(theta, -2.0 * (double)j / (double)head_dim);
    double phi = (double)p * inv_freq;
    table[i] = make_float2((float)cos(phi), (float)sin(phi));
  }
}

}  // namespace

cudaError_t prep_transpose(const void* src, void* dst, int rows, int cols, int state_dtype, cudaStream_t s) {
  dim3 grid((cols + 31) / 32, (rows + 31) / 32), block(32, 8);
  if (state_dtype == SCD_F32)
    transpose_kernel<float><<<grid, block, 0, s>>>((const float*)src, (float*)dst, rows, cols);
  else
    transpose_kernel<__nv_bfloat16><<<grid, block, 0, s>>>((const __nv_bfloat16*)src, (__nv_bfloat16*)dst, rows, cols);
  return cudaGetLastError();
}

cudaError_t prep_fold_gamma(const void* w, const void* gamma, void* dst, int rows, int cols, int state_dtype,
                            cudaStream_t s) {
  int grid = (int)((((size_t)rows * cols + 255) / 256) < 4096 ? (((size_t)rows * cols + 255) / 256) : 4096);
  if (grid < 1) grid = 1;
  if (state_dtype == SCD_F32)
    fold_gamma_kernel<float><<<grid, 256, 0, s>>>((const float*)w, (const float*)gamma, (float*)dst, rows, cols);
  else
    fold_gamma_kernel<__nv_bfloat16><<<grid, 256, 0, s>>>((const __nv_bfloat16*)w, (const __nv_bfloat16*)gamma,
                                                         (__nv_bfloat16*)dst, rows, cols);
  return cudaGetLastError();
}

cudaError_t prep_mean_proj(const float* mu, const void* w_enc, float* c, int width, int rank, int state_dtype,
                           cudaStream_t s) {
  int grid = (rank + 63) / 64;
  if (state_dtype == SCD_F32)
    mean_proj_kernel<float><<<grid, 64, 0, s>>>(mu, (const float*)w_enc, c, width, rank);
  else
    mean_proj_kernel<__nv_bfloat16><<<grid, 64, 0, s>>>(mu, (const __nv_bfloat16*)w_enc, c, width, rank);
  return cudaGetLastError();
}

cudaError_t prep_to_f32(const void* src, float* dst, int n, int state_dtype, cudaStream_t s) {
  int grid = (n + 255) / 256;
  if (state_dtype == SCD_F32)
    to_f32_kernel<float><<<grid, 256, 0, s>>>((const float*)src, dst, n);
  else
    to_f32_kernel<__nv_bfloat16><<<grid, 256, 0, s>>>((const __nv_bfloat16*)src, dst, n);
  return cudaGetLastError();
}

cudaError_t prep_copy_f32(const float* src, float* dst, int n, cudaStream_t s) {
  to_f32_kernel<float><<<(n + 255) / 256, 256, 0, s>>>(src, dst, n);
  return cudaGetLastError();
}

cudaError_t prep_rope_table(float2* table, int max_position, int head_dim, double theta, cudaStream_t s) {
  size_t n = (size_t)max_position * (head_dim / 2);
  int grid = (int)((n + 255) / 256 < 2048 ? (n + 255) / 256 : 2048);
  if (grid < 1) grid = 1;
  rope_table_kernel<<<grid, 256, 0, s>>>(table, max_position, head_dim, theta);
  return cudaGetLastError();
}

template <typename T>
__global__ void block_diag_kernel(const T* src, T* dst, int rows, int cols, int heads) {
  const long long n = (long long)heads * rows * heads * cols;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int c = (int)(i % ((long long)heads * cols)), r = (int)(i / ((long long)heads * cols));
    const bool on = (r / rows) == (c / cols);
    dst[i] = on ? src[(size_t)(r % rows) * cols + (c % cols)] : T(0.0f);
  }
}
cudaError_t prep_block_diag(const void* src, void* dst, int rows, int cols, int heads, int state_dtype, cudaStream_t s) {
  const long long n = (long long)heads * rows * heads * cols;
  const int grid = (int)std::min<long long>((n + 255) / 256, 4096);
  if (state_dtype == SCD_F32) block_diag_kernel<float><<<grid, 256, 0, s>>>((const float*)src, (float*)dst, rows, cols, heads);
  else block_diag_kernel<__nv_bfloat16><<<grid, 256, 0, s>>>((const __nv_bfloat16*)src, (__nv_bfloat16*)dst, rows, cols, heads);
  return cudaGetLastError();
}
__global__ void tile_f32_kernel(const float* src, float* dst, int n, int heads) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n * heads; i += gridDim.x * blockDim.x) dst[i] = src[i % n];
}
cudaError_t prep_tile_f32(const float* src, float* dst, int n, int heads, cudaStream_t s) {
  tile_f32_kernel<<<(n * heads + 255) / 256, 256, 0, s>>>(src, dst, n, heads);
  return cudaGetLastError();
}

}  // namespace scd
