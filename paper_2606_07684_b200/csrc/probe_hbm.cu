// Stand-alone HBM probe (not part of libscd.so): write-only, read-only, copy and 8:1 write:read streams over 1 GiB with
// plain 16-byte stores, 32-byte stores, TMA bulk stores and cudaMemset, from 148 CTAs up to 65536.  It answers one
// question for the REUSE decode (89 % writes): is write-only bandwidth on this part lower than the copy figure in
// MEASURED_PEAKS.json?  (No: profiles/r01_hbm_probe.md.)
//   nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a paper_2606_07684_b200/csrc/probe_hbm.cu -o /tmp/probe_hbm
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("ERR %s line %d\n", cudaGetErrorString(e), __LINE__); return 1; } } while (0)

__global__ void w_v4(uint4* p, size_t n) {  // grid-stride
  size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x, st = (size_t)gridDim.x * blockDim.x;
  uint4 v = make_uint4(1, 2, 3, 4);
  for (; i < n; i += st) p[i] = v;
}
__global__ void w_v4_cs(uint4* p, size_t n) {
  size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x, st = (size_t)gridDim.x * blockDim.x;
  for (; i < n; i += st) asm volatile("st.global.cs.v4.u32 [%0], {%1,%1,%1,%1};" ::"l"(p + i), "r"(7) : "memory");
}
__global__ void w_v8(uint4* p, size_t n) {  // 256-bit stores
  size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x, st = (size_t)gridDim.x * blockDim.x;
  for (; 2 * i + 1 < n; i += st)
    asm volatile("st.global.v8.u32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"l"(p + 2 * i), "r"(7) : "memory");
}
// contiguous chunk per CTA (each CTA owns n/grid contiguous uint4s), block-strided inside
__global__ void w_v4_chunk(uint4* p, size_t n) {
  size_t per = n / gridDim.x;
  uint4* q = p + per * blockIdx.x;
  uint4 v = make_uint4(1, 2, 3, 4);
  for (size_t i = threadIdx.x; i < per; i += blockDim.x) q[i] = v;
}
// rows of 2 KB at pseudo-random slots: each warp writes 512 B segments (like the decode epilogue)
__global__ void w_rows(uint4* p, size_t n_rows) {  // row = 128 uint4
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  uint4 v = make_uint4(1, 2, 3, 4);
  for (size_t r = (size_t)blockIdx.x * nw + warp; r < n_rows * 4; r += (size_t)gridDim.x * nw) {
    p[r * 32 + lane] = v;
  }
}
// TMA bulk store: smem -> global, CHUNK bytes each, one thread issues
template <int CHUNK>
__global__ void w_bulk(uint8_t* p, size_t bytes) {
  extern __shared__ __align__(128) uint8_t sm[];
  for (int i = threadIdx.x; i < CHUNK / 4; i += blockDim.x) ((uint32_t*)sm)[i] = i;
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t s = (uint32_t)__cvta_generic_to_shared(sm);
    size_t nchunks = bytes / CHUNK;
    for (size_t c = blockIdx.x; c < nchunks; c += gridDim.x) {
      asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(p + c * CHUNK), "r"(s), "r"(CHUNK) : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      asm volatile("cp.async.bulk.wait_group.read 8;" ::: "memory");
    }
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  }
}
__global__ void r_v4(const uint4* p, size_t n, uint32_t* out) {
  size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x, st = (size_t)gridDim.x * blockDim.x;
  uint32_t acc = 0;
  for (; i < n; i += st) { uint4 v = p[i]; acc ^= v.x ^ v.y ^ v.z ^ v.w; }
  if (acc == 0x12345) *out = acc;
}
__global__ void copy_v4(const uint4* a, uint4* b, size_t n) {
  size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x, st = (size_t)gridDim.x * blockDim.x;
  for (; i < n; i += st) b[i] = a[i];
}
// 8:1 write:read mix like decode
__global__ void mix_v4(const uint4* a, uint4* b, size_t n) {
  size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x, st = (size_t)gridDim.x * blockDim.x;
  for (; i < n / 8; i += st) { uint4 v = a[i];
#pragma unroll
    for (int k = 0; k < 8; ++k) b[i + k * (n / 8)] = v; }
}

int main() {
  const size_t bytes = 1ull << 30;
  uint8_t *a, *b; uint32_t* out;
  CK(cudaMalloc(&a, bytes)); CK(cudaMalloc(&b, bytes)); CK(cudaMalloc(&out, 4));
  CK(cudaMemset(a, 1, bytes)); CK(cudaMemset(b, 1, bytes));
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const size_t n = bytes / 16;
  auto run = [&](const char* name, auto launch, double moved) {
    float best = 1e9, sum = 0;
    for (int it = 0; it < 12; ++it) {
      cudaMemsetAsync(a, it, 256 << 20);  // flush-ish
      cudaEventRecord(e0); launch(); cudaEventRecord(e1); cudaEventSynchronize(e1);
      float ms; cudaEventElapsedTime(&ms, e0, e1);
      if (it >= 2) { best = ms < best ? ms : best; sum += ms; }
    }
    cudaError_t e = cudaGetLastError();
    printf("%-40s best %.3f ms %.0f GB/s  avg %.0f GB/s %s\n", name, best, moved / best * 1e-6, moved / (sum / 10) * 1e-6,
           e == cudaSuccess ? "" : cudaGetErrorString(e));
  };
  for (int g : {148, 296, 592, 1184, 4736, 65536}) {
    char nm[64]; snprintf(nm, 64, "w_v4 grid %d x 1024", g);
    run(nm, [&] { w_v4<<<g, 1024>>>((uint4*)b, n); }, (double)bytes);
  }
  run("w_v4 grid 148*8 x 256", [&] { w_v4<<<148 * 8, 256>>>((uint4*)b, n); }, (double)bytes);
  run("w_v4_cs grid 1184 x 1024", [&] { w_v4_cs<<<1184, 1024>>>((uint4*)b, n); }, (double)bytes);
  run("w_v8 grid 1184 x 1024", [&] { w_v8<<<1184, 1024>>>((uint4*)b, n); }, (double)bytes);
  run("w_v4_chunk grid 148 x 1024", [&] { w_v4_chunk<<<148, 1024>>>((uint4*)b, n); }, (double)(n / 148 * 148 * 16));
  run("w_v4_chunk grid 1184 x 512", [&] { w_v4_chunk<<<1184, 512>>>((uint4*)b, n); }, (double)(n / 1184 * 1184 * 16));
  run("w_rows 148 x 512", [&] { w_rows<<<148, 512>>>((uint4*)b, bytes / 2048); }, (double)bytes);
  run("w_rows 592 x 512", [&] { w_rows<<<592, 512>>>((uint4*)b, bytes / 2048); }, (double)bytes);
  run("cudaMemsetAsync", [&] { cudaMemsetAsync(b, 3, bytes); }, (double)bytes);
  run("w_bulk<2048> 148", [&] { w_bulk<2048><<<148, 128, 2048>>>(b, bytes); }, (double)bytes);
  run("w_bulk<8192> 148", [&] { w_bulk<8192><<<148, 128, 8192>>>(b, bytes); }, (double)bytes);
  run("w_bulk<32768> 148", [&] { w_bulk<32768><<<148, 128, 32768>>>(b, bytes); }, (double)bytes);
  run("w_bulk<8192> 592", [&] { w_bulk<8192><<<592, 128, 8192>>>(b, bytes); }, (double)bytes);
  run("w_bulk<512> 592", [&] { w_bulk<512><<<592, 128, 512>>>(b, bytes); }, (double)bytes);
  run("r_v4 grid 1184 x 1024", [&] { r_v4<<<1184, 1024>>>((const uint4*)b, n, out); }, (double)bytes);
  run("r_v4 grid 4736 x 512", [&] { r_v4<<<4736, 512>>>((const uint4*)b, n, out); }, (double)bytes);
  run("copy_v4 grid 1184 x 1024", [&] { copy_v4<<<1184, 1024>>>((const uint4*)a, (uint4*)b, n); }, 2.0 * bytes);
  run("mix 8w:1r grid 1184 x 1024", [&] { mix_v4<<<1184, 1024>>>((const uint4*)a, (uint4*)b, n); }, 1.125 * bytes);
  return 0;
}
