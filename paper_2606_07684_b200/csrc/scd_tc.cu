// Tensor-core path of the SCD codec for bf16 states on sm_100a.
//
// Every step of the path is one GEMM shape, C[M,N] = A[M,K] Bt[N,K]^T with both operands
// K-major, plus an A-side transform and a fused epilogue (scd_internal.h: EpiKind, AMode).
// One persistent, warp-specialised kernel template serves all of them:
//
//   warp 0        TMA producer: A tile [128 x 64] and Bt tile [BLOCK_N x 64] per k-block into a shared-memory
//                 ring (128-byte swizzle, 3-6 stages: as many as the launch's epilogue leaves room for),
//                 mbarrier expect_tx / complete_tx; the encode's A stream is pulled into L2 a few k-blocks ahead
//   warp 1        MMA issuer: one elected thread issues tcgen05.mma (128 x BLOCK_N x 16, bf16 -> fp32) into one
//                 of two TMEM accumulator buffers; tcgen05.commit releases the smem stage and finally signals
//                 the epilogue
//   warp 2        TMEM allocator (512 columns = 2 accumulator buffers of 256 columns)
//   warps 4-11    epilogue: tcgen05.ld (one token row per thread; the two warps of a lane quadrant split the
//                 columns or, for two-head K tiles, the RoPE frequencies), fused mean / row-scale / RoPE /
//                 activation / quantisation, swizzled per-warp staging, coalesced 16-byte stores (codes,
//                 workspace, or the token's slot of the paged KV pool); overlaps the next tile's MMAs
//   warps 12-27   (A_DEROPE / A_CODES only) transform the freshly landed A tile in shared memory, 4 threads per
//                 token row, before the MMA may read it: rotate K by -position (Eq. 5) / widen e4m3 codes to bf16
//
// A launch covers many (layer, branch) segments of equal shape: tile -> (segment, L2 super-block, n-tile,
// m-tile) with m fastest, tiles dealt round-robin to one CTA per SM.  Launched with programmatic stream
// serialisation: everything above the first global access overlaps the previous kernel's tail.
#include <algorithm>
#include <cmath>
#include <cstring>

#include "scd_tc_common.cuh"

namespace scd {

// A_DEROPE / A_CODES: 16 extra warps transform the landed A tile in shared memory, 4 threads per token row
// (rotate the K tile by -position; expand e4m3 codes to the bf16 operand the MMA takes)
constexpr int DEROPE_WARPS = 16;
constexpr int DEROPE_NTHREADS = (4 + EPI_WARPS + DEROPE_WARPS) * 32;   // 896

struct __align__(8) TcBarriers {
  uint64_t full[MAX_STAGES], empty[MAX_STAGES], ready[MAX_STAGES];
  uint64_t tmem_full[2], tmem_empty[2];
  uint64_t b_full[4], b_empty[4];              // B-resident mode (PATCH GEMM-1): the resident B tile's k-block slots
  uint64_t sched_full[4], sched_empty[4];      // dynamic tile claiming (plain encodes): ring of claimed tile ids
  int32_t sched_tile[4];                       // -1 = no more tiles
  uint32_t tmem_base;
};

// per-warp staging the epilogue needs: 32 rows x the widest sub-tile row, in whole 128-B swizzle spans.  The encode
// epilogue (narrow code tiles) needs half of STG_WARP_BYTES; the shared memory it leaves buys a pipeline stage.
// Shared memory is what buys pipeline stages, and three 48 KB stages (128 x 256 tiles) do not cover the TMA latency of the
// PATCH GEMM-2 (K = d_a).  Its epilogue is off the critical path, so it stages 64 columns at a time (4 KB per warp) and reads
// the bias straight from L1/L2 instead of a per-warp shared copy: that is the room for a fourth stage.
static int tc_sub_n(int epi, bool compact) { return (epi == EPI_U || epi == EPI_ACT || compact) ? 64 : SUB_N; }
// epilogue warps of an instantiation: PATCH GEMM-1 (two k-blocks per tile, SiLU on the MUFU pipe) is paced by its epilogue,
// so its plain-A kernel runs sixteen (four per TMEM lane quadrant, 64 columns each) -- one warp's MUFU phase overlaps the
// others' TMEM reads and copy-out; every other kernel eight (two per quadrant)
__host__ __device__ constexpr int tc_epi_warps(int epi, int amode, bool pair) {
  return (epi == EPI_ACT && amode == A_PLAIN && !pair) ? 16 : EPI_WARPS;
}
static int tc_vec_warp_bytes(int epi, bool compact) { return (epi == EPI_U || epi == EPI_CODES || compact) ? 0 : VEC_WARP_BYTES; }
static int tc_stg_warp_bytes(int epi, int block_n, bool compact, int out_eb) {
  if (compact) return 32 * 128;
  if (epi == EPI_KV) return STG_WARP_BYTES;
  const int cols = (block_n % 64) == 0 ? block_n / 2 : block_n;      // the warp pair splits the columns (gran = 32)
  const int sub = cols < tc_sub_n(epi, false) ? cols : tc_sub_n(epi, false);
  return 32 * ((sub * out_eb + 127) & ~127);       // out_eb: 1 for e4m3 codes, else 2
}
// b_rows: rows of the B tile a CTA holds per stage (block_n, or half of it when a CTA pair shares the tile)
static size_t tc_smem_bytes(int b_rows, int stages, int stg_warp_bytes, int vec_warp_bytes, int epi_warps) {
  return 1024 /*align slack*/ + (size_t)stages * (A_STAGE_BYTES + (size_t)b_rows * BLOCK_K * 2) +
         epi_warps * (stg_warp_bytes + vec_warp_bytes) + sizeof(TcBarriers);
}
// B-resident mode: num_kb slots for the B tile + a ring of A stages
static size_t tc_smem_bytes_bres(int b_rows, int num_kb, int stages, int stg_warp_bytes, int vec_warp_bytes, int epi_warps) {
  return 1024 + (size_t)stages * A_STAGE_BYTES + (size_t)num_kb * b_rows * BLOCK_K * 2 + epi_warps * (stg_warp_bytes + vec_warp_bytes) +
         sizeof(TcBarriers);
}
static int tc_pick_stages_bres(int b_rows, int num_kb, int stg_warp_bytes, int vec_warp_bytes, int epi_warps) {
  const long long budget = 232448 - 1024 - epi_warps * (stg_warp_bytes + vec_warp_bytes) - (long long)sizeof(TcBarriers) -
                           (long long)num_kb * b_rows * BLOCK_K * 2;
  const int st = (int)(budget / A_STAGE_BYTES);
  return st > MAX_STAGES ? MAX_STAGES : st;
}
static int tc_pick_stages(int b_rows, int num_kb, int stg_warp_bytes, int vec_warp_bytes, int epi_warps) {
  const size_t budget = 232448 - 1024 - epi_warps * (stg_warp_bytes + vec_warp_bytes) - sizeof(TcBarriers);
  int st = (int)(budget / (A_STAGE_BYTES + (size_t)b_rows * BLOCK_K * 2));
  st = st > MAX_STAGES ? MAX_STAGES : st;
  if (st > 2 * num_kb && num_kb >= 1) st = 2 * num_kb > 2 ? 2 * num_kb : 2;   // two tiles in flight is plenty (3, 4 measured: same)
  return st < 2 ? 2 : st;          // odd rings are fine for deRoPE: a k-block pair may straddle the wrap
}


// Tile order inside a segment: super-blocks of P.msb m-tiles; inside a super-block all its m-tiles for
// n-tile 0, then n-tile 1, ...  The A rows of a super-block (msb x 128 tokens) stay L2-resident while every
// B slice passes once per super-block, instead of A being re-streamed from HBM once per n-tile when
// T x K x 2 B outgrows the L2 (PATCH GEMM-2 at 32k tokens: 268-537 MB).  msb >= m_tiles: plain m-fastest order.
// `mt` = m-tiles of the walk: P.m_tiles, or the number of 256-row pair tiles when CTA pairs share an MMA (P.msb is then
// in pair tiles too).
__device__ __forceinline__ void tile_decode(const TcParams& P, int mt, int tile, int& m_tile, int& n_tile, int& seg) {
  const int per_seg = mt * P.n_tiles;
  seg = tile / per_seg;
  const int t = tile - seg * per_seg;
  if (P.msb >= mt) {
    n_tile = t / mt;
    m_tile = t - n_tile * mt;
    return;
  }
  const int per_sb = P.msb * P.n_tiles;
  const int sb = t / per_sb;
  const int rem = t - sb * per_sb;
  const int rows = min(P.msb, mt - sb * P.msb);     // the last super-block may be short
  n_tile = rem / rows;
  m_tile = sb * P.msb + (rem - n_tile * rows);
}

// per-warp staging tile (shared-space address `stg`): row pitch `pitch` bytes (>= 128), 16-byte
// chunks XOR-swizzled on the low 3 bits of the row so that row-per-thread writes and
// row-per-half-warp reads are both bank-conflict free
__device__ __forceinline__ uint32_t stg_addr(uint32_t stg, int pitch, int row, int chunk) {
  return stg + row * pitch + (((chunk & ~7) | ((chunk ^ row) & 7)) << 4);
}
__device__ __forceinline__ void stg_put(uint32_t stg, int pitch, int row, int chunk, uint4 v) {
  ptx::sts128(stg_addr(stg, pitch, row, chunk), v);
}

// Copy the warp's staged sub-tile (32 rows x row_bytes) to global: LPR lanes cover one row with
// one fully coalesced 16-B store each; row base pointers come from the owning lane by shuffle
// (null = row beyond M).  `valid_bytes` masks the N tail.
// `streaming`: pool rows and codes are written once and not read back by this call chain -> evict-first stores, so
// they do not push the operands out of L2; workspace tensors (read by the next GEMM) use plain stores.
template <int LPR>
__device__ __forceinline__ void stg_copy_out_t(uint32_t stg, int pitch, int valid_bytes, unsigned long long my_row_ptr,
                                               unsigned long long byte_off, int lane, bool streaming) {
  constexpr int rpi = 32 / LPR;
  const int chunk = lane % LPR;
#pragma unroll
  for (int it = 0; it < LPR; ++it) {
    const int r = it * rpi + lane / LPR;
    const unsigned long long base = __shfl_sync(0xffffffffu, my_row_ptr, r);
    const uint4 v = ptx::lds128(stg_addr(stg, pitch, r, chunk));
    if (base != 0ull && chunk * 16 < valid_bytes) {
      if (streaming) ptx::stg128_cs(base + byte_off + (unsigned long long)chunk * 16, v);
      else ptx::stg128(base + byte_off + (unsigned long long)chunk * 16, v);
    }
  }
}
__device__ __forceinline__ void stg_copy_out(uint32_t stg, int pitch, int row_bytes, int valid_bytes,
                                             unsigned long long my_row_ptr, unsigned long long byte_off, int lane, bool streaming) {
  int lpr = 1;
  while (lpr * 16 < row_bytes) lpr <<= 1;             // lanes per row: next power of two
  switch (lpr) {
    case 16: stg_copy_out_t<16>(stg, pitch, valid_bytes, my_row_ptr, byte_off, lane, streaming); break;
    case 8: stg_copy_out_t<8>(stg, pitch, valid_bytes, my_row_ptr, byte_off, lane, streaming); break;
    case 4: stg_copy_out_t<4>(stg, pitch, valid_bytes, my_row_ptr, byte_off, lane, streaming); break;
    case 2: stg_copy_out_t<2>(stg, pitch, valid_bytes, my_row_ptr, byte_off, lane, streaming); break;
    default: stg_copy_out_t<1>(stg, pitch, valid_bytes, my_row_ptr, byte_off, lane, streaming); break;
  }
}

// ---- PATCH GEMM-1 (aligner in) epilogue of a whole 256-column tile: 64 of this warp's columns of its 32 rows ----
// v = acc * scale + bias (packed fp32), SiLU(x) = h + h tanh(h) with h = x / 2 (the caller passes scale / 2 and the
// staged bias is already halved), bf16, staged row-per-thread in the warp's [32 x 128 B] swizzled buffer.
template <bool SILU>
__device__ __forceinline__ void act_stage64(uint32_t t_cols, uint32_t stg, uint32_t wvec, float scale, int lane) {
  const unsigned long long s2 = f2_pack(scale, scale);
#pragma unroll 1
  for (int c = 0; c < 64; c += 32) {
    uint32_t r[32];
    ptx::tmem_ld32(t_cols + c, r);
    ptx::tmem_ld_wait();
    uint32_t o[16];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const float4 m4 = ptx::lds_f4(wvec + (c + q * 4) * 4);
      float v0, v1, v2, v3;
      f2_unpack(f2_fma(f2_pack(__uint_as_float(r[q * 4]), __uint_as_float(r[q * 4 + 1])), s2, f2_pack(m4.x, m4.y)), v0, v1);
      f2_unpack(f2_fma(f2_pack(__uint_as_float(r[q * 4 + 2]), __uint_as_float(r[q * 4 + 3])), s2, f2_pack(m4.z, m4.w)), v2, v3);
      if (SILU) {
        float t0, t1, t2, t3;
        asm("tanh.approx.f32 %0, %1;" : "=f"(t0) : "f"(v0));
        asm("tanh.approx.f32 %0, %1;" : "=f"(t1) : "f"(v1));
        asm("tanh.approx.f32 %0, %1;" : "=f"(t2) : "f"(v2));
        asm("tanh.approx.f32 %0, %1;" : "=f"(t3) : "f"(v3));
        v0 = fmaf(v0, t0, v0); v1 = fmaf(v1, t1, v1); v2 = fmaf(v2, t2, v2); v3 = fmaf(v3, t3, v3);
      }
      o[q * 2] = pack_bf16x2(v0, v1);
      o[q * 2 + 1] = pack_bf16x2(v2, v3);
    }
#pragma unroll
    for (int q = 0; q < 4; ++q)
      ptx::sts128(stg_addr(stg, 128, lane, (c >> 3) + q), make_uint4(o[4 * q], o[4 * q + 1], o[4 * q + 2], o[4 * q + 3]));
  }
}
// The staged [32 x 128 B] buffer to a row-major tensor: rows are consecutive (row r at out + r * row_stride), eight lanes
// per row, one 16-B store per lane, no per-row pointers; rows >= rows_valid (the M tail) are skipped.
__device__ __forceinline__ void rowmajor_copy_out_128(uint32_t stg, unsigned long long out, unsigned long long row_stride,
                                                      int rows_valid, int lane) {
  const int chunk = lane & 7, rq = lane >> 3;
  unsigned long long p = out + (unsigned long long)rq * row_stride + (unsigned long long)chunk * 16ull;
#pragma unroll
  for (int it = 0; it < 8; ++it) {
    const int r = it * 4 + rq;
    const uint4 v = ptx::lds128(stg_addr(stg, 128, r, chunk));
    if (r < rows_valid) ptx::stg128(p, v);
    p += 4ull * row_stride;
  }
}

// RoPE epilogue of one K tile, specialised for HALF pairing, head_dim 128, 256-column tiles (two
// heads).  The warp pair of a lane quadrant splits the FREQUENCIES, not the columns: warp JG owns
// j in [32 JG, 32 JG + 32) of both heads, so every (cos, sin) is computed once and used twice.
// Staged row = 4 runs of 32 columns: (head 0, a) (head 0, b) (head 1, a) (head 1, b).
template <int JG>
__device__ __forceinline__ void rope_tile_h128(const TcParams& P, uint32_t t_row, uint32_t stg, uint32_t wvec, int pos,
                                               float rs, int lane) {
#pragma unroll
  for (int jj = 0; jj < 32; jj += 16) {
    // (cos, cos), (sin, sin), (-sin, -sin) packed over adjacent frequency pairs
    unsigned long long c2[8], s2[8], ns2[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const float2 x = rope_cs(pos, P.rope_g[JG * 32 + jj + 2 * i]), y = rope_cs(pos, P.rope_g[JG * 32 + jj + 2 * i + 1]);
      c2[i] = f2_pack(x.x, y.x);
      s2[i] = f2_pack(x.y, y.y);
      ns2[i] = f2_pack(-x.y, -y.y);
    }
    const unsigned long long rs2 = f2_pack(rs, rs);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      uint32_t ra[16], rb[16];
      const int ca = h * 128 + JG * 32 + jj;          // tile column of the "a" elements; "b" = +64
      ptx::tmem_ld16(t_row + ca, ra);
      ptx::tmem_ld16(t_row + ca + 64, rb);
      ptx::tmem_ld_wait();
      uint32_t oa[8], ob[8];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const float4 ma = ptx::lds_f4(wvec + (ca + q * 4) * 4), mb = ptx::lds_f4(wvec + (ca + 64 + q * 4) * 4);
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int i = q * 4 + e * 2;                 // elements i, i + 1
          const unsigned long long a = f2_fma(f2_pack(__uint_as_float(ra[i]), __uint_as_float(ra[i + 1])), rs2,
                                              e ? f2_pack(ma.z, ma.w) : f2_pack(ma.x, ma.y));
          const unsigned long long b = f2_fma(f2_pack(__uint_as_float(rb[i]), __uint_as_float(rb[i + 1])), rs2,
                                              e ? f2_pack(mb.z, mb.w) : f2_pack(mb.x, mb.y));
          float x0, x1, y0, y1;
          f2_unpack(f2_fma(b, ns2[i >> 1], f2_mul(a, c2[i >> 1])), x0, x1);   // a cos - b sin
          f2_unpack(f2_fma(a, s2[i >> 1], f2_mul(b, c2[i >> 1])), y0, y1);    // b cos + a sin
          oa[q * 2 + e] = pack_bf16x2(x0, x1);
          ob[q * 2 + e] = pack_bf16x2(y0, y1);
        }
      }
      const int k0 = h * 8 + (jj >> 3);               // chunk of run (h, a); run (h, b) = +4
      stg_put(stg, 256, lane, k0, make_uint4(oa[0], oa[1], oa[2], oa[3]));
      stg_put(stg, 256, lane, k0 + 1, make_uint4(oa[4], oa[5], oa[6], oa[7]));
      stg_put(stg, 256, lane, k0 + 4, make_uint4(ob[0], ob[1], ob[2], ob[3]));
      stg_put(stg, 256, lane, k0 + 5, make_uint4(ob[4], ob[5], ob[6], ob[7]));
    }
  }
}
// Compact variant for long-K tiles (PATCH GEMM-3), where the epilogue is off the critical path and shared memory is
// better spent on a fourth pipeline stage: one head at a time through a 4 KB per-warp staging tile (row = run a | run b,
// 64 B each), bias read through L1, (cos, sin) recomputed per head.  `bias` = col_vec + n0 or null.
template <int JG>
__device__ __forceinline__ void rope_tile_h128_compact(const TcParams& P, uint32_t t_row, uint32_t stg, const float* bias,
                                                       int pos, float rs, unsigned long long my_row_ptr, int lane) {
  const unsigned long long rs2 = f2_pack(rs, rs);
#pragma unroll 1
  for (int h = 0; h < 2; ++h) {
#pragma unroll
    for (int jj = 0; jj < 32; jj += 16) {
      unsigned long long c2[8], s2[8], ns2[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const float2 x = rope_cs(pos, P.rope_g[JG * 32 + jj + 2 * i]), y = rope_cs(pos, P.rope_g[JG * 32 + jj + 2 * i + 1]);
        c2[i] = f2_pack(x.x, y.x);
        s2[i] = f2_pack(x.y, y.y);
        ns2[i] = f2_pack(-x.y, -y.y);
      }
      uint32_t ra[16], rb[16];
      const int ca = h * 128 + JG * 32 + jj;          // tile column of the "a" elements; "b" = +64
      ptx::tmem_ld16(t_row + ca, ra);
      ptx::tmem_ld16(t_row + ca + 64, rb);
      ptx::tmem_ld_wait();
      uint32_t oa[8], ob[8];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
        const float4 ma = bias ? ldg_f4(bias + ca + q * 4) : z4, mb = bias ? ldg_f4(bias + ca + 64 + q * 4) : z4;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int i = q * 4 + e * 2;
          const unsigned long long a = f2_fma(f2_pack(__uint_as_float(ra[i]), __uint_as_float(ra[i + 1])), rs2,
                                              e ? f2_pack(ma.z, ma.w) : f2_pack(ma.x, ma.y));
          const unsigned long long b = f2_fma(f2_pack(__uint_as_float(rb[i]), __uint_as_float(rb[i + 1])), rs2,
                                              e ? f2_pack(mb.z, mb.w) : f2_pack(mb.x, mb.y));
          float x0, x1, y0, y1;
          f2_unpack(f2_fma(b, ns2[i >> 1], f2_mul(a, c2[i >> 1])), x0, x1);   // a cos - b sin
          f2_unpack(f2_fma(a, s2[i >> 1], f2_mul(b, c2[i >> 1])), y0, y1);    // b cos + a sin
          oa[q * 2 + e] = pack_bf16x2(x0, x1);
          ob[q * 2 + e] = pack_bf16x2(y0, y1);
        }
      }
      const int k0 = jj >> 3;                          // chunk of run a; run b = +4
      stg_put(stg, 128, lane, k0, make_uint4(oa[0], oa[1], oa[2], oa[3]));
      stg_put(stg, 128, lane, k0 + 1, make_uint4(oa[4], oa[5], oa[6], oa[7]));
      stg_put(stg, 128, lane, k0 + 4, make_uint4(ob[0], ob[1], ob[2], ob[3]));
      stg_put(stg, 128, lane, k0 + 5, make_uint4(ob[4], ob[5], ob[6], ob[7]));
    }
    __syncwarp();
    {
      const int l = lane & 7;                          // 8 lanes per row: run l / 4, chunk l % 4
      const unsigned long long off = (unsigned long long)((h * 128 + (l >> 2) * 64 + JG * 32 + (l & 3) * 8) * 2);
#pragma unroll
      for (int it = 0; it < 8; ++it) {
        const int r = it * 4 + (lane >> 3);
        const unsigned long long base = __shfl_sync(0xffffffffu, my_row_ptr, r);
        const uint4 v = ptx::lds128(stg_addr(stg, 128, r, l));
        if (base != 0ull) ptx::stg128_cs(base + off, v);
      }
    }
    __syncwarp();
  }
}
// copy-out of the 4-run layout above: lane l of a half-warp holds run l / 4, chunk l % 4
template <int JG>
__device__ __forceinline__ void rope_tile_h128_copy_out(uint32_t stg, unsigned long long my_row_ptr, int lane) {
  const int l = lane & 15;
  const unsigned long long off = (unsigned long long)(((l >> 3) * 128 + ((l >> 2) & 1) * 64 + JG * 32 + (l & 3) * 8) * 2);
#pragma unroll
  for (int it = 0; it < 16; ++it) {
    const int r = it * 2 + (lane >> 4);
    const unsigned long long base = __shfl_sync(0xffffffffu, my_row_ptr, r);
    const uint4 v = ptx::lds128(stg_addr(stg, 256, r, l));
    if (base != 0ull) ptx::stg128_cs(base + off, v);
  }
}

// ---------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------
// PAIR: two CTAs on the SMs of one TPC (cluster of 2) run ONE tcgen05.mma.cta_group::2 of M = 256: each CTA loads its own
// 128 rows of A and HALF of the B tile, so a B tile leaves L2 once per 256 output rows and a stage costs 32 KB instead of
// 48 KB (two more pipeline stages).  The even CTA ("leader") issues the MMAs; loads of both CTAs report to its `full`
// barriers, its commits are multicast to both CTAs' `empty` / `tmem_full` barriers, and the epilogue warps of both CTAs
// hand accumulators back on its `tmem_empty` barriers.  Tile = (segment, n-tile, pair of m-tiles).
template <int EPI, int AMODE, bool PAIR = false>
__global__ void __launch_bounds__(AMODE != A_PLAIN ? DEROPE_NTHREADS : (4 + tc_epi_warps(EPI, AMODE, PAIR)) * 32, 1)
tc_gemm_kernel(const __grid_constant__ TcParams P) {
  static_assert(!PAIR || AMODE == A_PLAIN, "CTA pairs: plain A operands only");
  constexpr int NEPI = tc_epi_warps(EPI, AMODE, PAIR);           // epilogue warps: 8, or 16 for PATCH GEMM-1
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  const int block_n = P.block_n;
  const uint32_t b_stage_bytes = (uint32_t)block_n * BLOCK_K * (PAIR ? 1 : 2);   // PAIR: this CTA's half of the B tile
  const uint32_t cta_rank = PAIR ? ptx::cluster_ctarank() : 0u;
  const int walk_mt = PAIR ? (P.m_tiles + 1) / 2 : P.m_tiles;
  const int walker = PAIR ? (int)(blockIdx.x >> 1) : (int)blockIdx.x;            // index of this CTA (pair) in the tile walk
  const int walk_stride = PAIR ? (int)(gridDim.x >> 1) : (int)gridDim.x;
  const int STAGES = P.stages;
  // B-resident mode (PATCH GEMM-1: K = r_h is one or two k-blocks, so the 64 KB B tile is two thirds of a tile's operand bytes):
  // each CTA walks a CONTIGUOUS share of the (segment, n-tile, m-tile) order, m fastest, keeps the B tile of its (segment,
  // n-tile) in slots of its own and streams only the A tiles through the ring
  constexpr bool BRES_OK = EPI == EPI_ACT && AMODE == A_PLAIN && !PAIR;
  const bool bres = BRES_OK && P.b_res;
  uint8_t* smem_a = smem;
  uint8_t* smem_b = smem + STAGES * A_STAGE_BYTES;
  uint8_t* smem_stg = smem_b + (bres ? P.num_kb : STAGES) * b_stage_bytes;
  uint8_t* smem_vec = smem_stg + NEPI * P.stg_warp_bytes;
  constexpr bool VEC_SMEM = (EPI == EPI_KV || EPI == EPI_ACT);   // else the mean / bias is read through L1 (tc_vec_warp_bytes)
  const bool vec_smem = VEC_SMEM && !(EPI == EPI_KV && P.kv_compact);
  TcBarriers* bars = (TcBarriers*)(smem_vec + (vec_smem ? NEPI * VEC_WARP_BYTES : 0));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int total_tiles = P.n_segs * P.n_tiles * walk_mt;
  // this CTA's tiles: t_begin, t_begin + t_step, ... < t_end
  const int t_begin = bres ? (int)((long long)blockIdx.x * total_tiles / gridDim.x) : walker;
  const int t_end = bres ? (int)((long long)(blockIdx.x + 1) * total_tiles / gridDim.x) : total_tiles;
  const int t_step = bres ? 1 : walk_stride;
  // Dynamic tile claiming (the encode's plain launches, P.sched set by the host): every CTA starts on tile blockIdx.x and then
  // claims tiles from a global counter (the producer thread, always one claim ahead of the tile it is loading) and hands
  // them to the MMA thread and the epilogue warps through a four-entry ring.  A launch that starts while its predecessor's
  // last wave is still running (dep_wait_late) then fills the hole that wave leaves: CTAs that start late claim fewer tiles.
  constexpr bool DYN_OK = EPI == EPI_CODES && AMODE == A_PLAIN && !PAIR;
  const bool dyn = DYN_OK && P.sched != nullptr;

  if (warp == 0 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) {
      ptx::mbar_init(&bars->full[s], 1);
      ptx::mbar_init(&bars->empty[s], 1);
      ptx::mbar_init(&bars->ready[s], DEROPE_WARPS * 32);
    }
    for (int k = 0; k < 4; ++k) {
      ptx::mbar_init(&bars->b_full[k], 1);
      ptx::mbar_init(&bars->b_empty[k], 1);
      ptx::mbar_init(&bars->sched_full[k], 1);
      ptx::mbar_init(&bars->sched_empty[k], 1 + NEPI);           // MMA thread + one lane per epilogue warp
    }
    for (int a = 0; a < 2; ++a) {
      ptx::mbar_init(&bars->tmem_full[a], 1);
      ptx::mbar_init(&bars->tmem_empty[a], PAIR ? 2 * EPI_WARPS : NEPI);
    }
    ptx::fence_barrier_init();
  }
  if (warp == 2) {
    if (PAIR) {
      ptx::tmem_alloc_cg2<TMEM_COLS>(&bars->tmem_base);
      ptx::tmem_relinquish_cg2();
    } else {
      ptx::tmem_alloc<TMEM_COLS>(&bars->tmem_base);
      ptx::tmem_relinquish();
    }
  }
  ptx::tc_fence_before();
  if (PAIR) ptx::cluster_sync();        // the peer's barriers exist before anything is sent to them
  else __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = bars->tmem_base;
  // The previous kernel of the stream has completed and flushed -- unless this launch is independent of it (P.dep_wait_late:
  // the 2nd, 3rd ... launch of one scd_encode call reads the caller's states and writes its own code segments), in which case
  // its CTAs start working as the predecessor's last wave frees SMs and wait for it at their END instead, so that this grid's
  // completion still implies the predecessor's (the next call's first kernel waits on the last launch only).
  if (!P.dep_wait_late) ptx::grid_dep_wait();
  ptx::grid_dep_launch_dependents();    // the next one may start its prologue as SMs free up

  // A_DEROPE / A_CODES: 896 threads x 72 registers, re-dealt per role: control warps 40 (at 24 the TMA producer's and
  // the MMA thread's loops were starved: encode K 0.134 -> 0.129 ms), epilogue warps 120, transform warps 56 (<= 64512)
  if (warp < 4) {
  if (AMODE != A_PLAIN) ptx::setmaxnreg_dec<40>();
  if (warp == 0) {
    // ============================== TMA producer ==============================
    if (P.a_gather) {
      // Paged producer cache: the tile's 128 token rows sit at the slots the producer's page table gives them.  Lane l
      // owns rows 4l .. 4l+3 and fetches them with one tile::gather4 per k-block (32 gathers = one A tile); lane 0
      // also arms the barrier and loads the B tile.  Rows beyond M (and page ids outside the pool) read slot 0.
      int stage = 0;
      uint32_t phase = 0;
      int cur_m = -1;
      int r4[4] = {0, 0, 0, 0};
      bool page_run = false;             // the 16 rows of this lane's group (4 lanes) sit in 16 consecutive slots: one tiled box
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        int m_tile, n_tile, seg_i;
        tile_decode(P, walk_mt, tile, m_tile, n_tile, seg_i);
        const TcSeg& sg = P.segs[seg_i];
        const CUtensorMap* am = &P.a_maps[sg.a_map];
        const CUtensorMap* bm = P.b_maps + sg.b_map;
        if (m_tile != cur_m) {
          cur_m = m_tile;
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int row = m_tile * BLOCK_M + lane * 4 + i;
            int pos;
            long long slot = -1;
            if (row < P.M) row_to_pos_slot(P.batch, row, pos, slot);
            r4[i] = slot < 0 ? 0 : (int)slot;
          }
          // requests that start on a page boundary put every 16-row group of the tile on one page: fetch it with one
          // tiled 16-row box instead of four gathers (8 instead of 32 TMA operations per A tile)
          const int base = __shfl_sync(0xffffffffu, r4[0], lane & ~3);
          const bool mine = r4[1] == r4[0] + 1 && r4[2] == r4[0] + 2 && r4[3] == r4[0] + 3 && r4[0] == base + 4 * (lane & 3) &&
                            m_tile * BLOCK_M + (lane | 3) * 4 + 3 < P.M;
          const unsigned all = __ballot_sync(0xffffffffu, mine);
          page_run = ((all >> (lane & ~3)) & 0xFu) == 0xFu;
        }
        const CUtensorMap* pm = &P.a_maps[TC_MAX_AMAPS / 2 + sg.a_map];     // the same pool with a 16-row box
        for (int kb = 0; kb < P.num_kb; ++kb) {
          ptx::mbar_wait_suspend(&bars->empty[stage], phase ^ 1);
          if (lane == 0) {
            ptx::mbar_expect_tx(&bars->full[stage], A_STAGE_BYTES + b_stage_bytes);
            ptx::tma_load_2d(smem_b + stage * b_stage_bytes, bm, &bars->full[stage], kb * BLOCK_K, n_tile * block_n);
          }
          __syncwarp();
          if (!page_run)
            ptx::tma_gather4_2d(smem_a + stage * A_STAGE_BYTES + lane * 512, am, &bars->full[stage], kb * BLOCK_K, r4[0], r4[1], r4[2], r4[3]);
          else if ((lane & 3) == 0)
            ptx::tma_load_2d(smem_a + stage * A_STAGE_BYTES + lane * 512, pm, &bars->full[stage], kb * BLOCK_K, r4[0]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    } else
    if (PAIR) {
      if (lane == 0) {
        int stage = 0;
        uint32_t phase = 0;
        for (int tile = walker; tile < total_tiles; tile += walk_stride) {
          int mp, n_tile, seg_i;
          tile_decode(P, walk_mt, tile, mp, n_tile, seg_i);
          const int m_tile = 2 * mp + (int)cta_rank;
          const TcSeg& sg = P.segs[seg_i];
          const CUtensorMap* am = &P.a_maps[sg.a_map];
          const CUtensorMap* bm = P.b_maps + sg.b_map;
          for (int kb = 0; kb < P.num_kb; ++kb) {
            ptx::mbar_wait_suspend(&bars->empty[stage], phase ^ 1);
            const uint32_t lead_full = ptx::mapa(ptx::smem_u32(&bars->full[stage]), 0);
            if (cta_rank == 0) ptx::mbar_expect_tx(&bars->full[stage], 2 * (A_STAGE_BYTES + b_stage_bytes));
            ptx::tma_load_3d_cg2(smem_a + stage * A_STAGE_BYTES, am, lead_full, kb * BLOCK_K, m_tile * BLOCK_M, sg.a_z);
            ptx::tma_load_2d_cg2(smem_b + stage * b_stage_bytes, bm, lead_full, kb * BLOCK_K,
                                 n_tile * block_n + (int)cta_rank * (block_n / 2));
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
        }
      }
    } else if (bres) {
      if (lane == 0) {
        int stage = 0, prev_key = -1;
        uint32_t phase = 0, groups = 0;                         // groups = (segment, n-tile) B tiles started so far
        for (int tile = t_begin; tile < t_end; ++tile) {
          int m_tile, n_tile, seg_i;
          tile_decode(P, walk_mt, tile, m_tile, n_tile, seg_i);
          const TcSeg& sg = P.segs[seg_i];
          const int key = seg_i * P.n_tiles + n_tile;
          const bool grp_first = key != prev_key;
          prev_key = key;
          for (int kb = 0; kb < P.num_kb; ++kb) {
            if (grp_first) {                                     // the B tile's k-block, once the previous group's MMAs are done with the slot
              if (groups > 0) ptx::mbar_wait_suspend(&bars->b_empty[kb], (groups - 1) & 1);
              ptx::mbar_expect_tx(&bars->b_full[kb], b_stage_bytes);
              ptx::tma_load_2d(smem_b + kb * b_stage_bytes, P.b_maps + sg.b_map, &bars->b_full[kb], kb * BLOCK_K, n_tile * block_n);
            }
            ptx::mbar_wait_suspend(&bars->empty[stage], phase ^ 1);
            ptx::mbar_expect_tx(&bars->full[stage], A_STAGE_BYTES);
            ptx::tma_load_3d(smem_a + stage * A_STAGE_BYTES, &P.a_maps[sg.a_map], &bars->full[stage], kb * BLOCK_K, m_tile * BLOCK_M, sg.a_z);
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
          if (grp_first) ++groups;
        }
      }
    } else
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      int sslot = 0;
      uint32_t sphase = 0;
      int tile = blockIdx.x;
      int next = dyn ? (int)gridDim.x + atomicAdd(P.sched, 1) : tile + (int)gridDim.x;
      for (;;) {
        // dynamic: claim the tile after next now (the atomic's latency hides under this tile's loads), publish this one
        int after = next + (int)gridDim.x;
        if (dyn) {
          after = next < total_tiles ? (int)gridDim.x + atomicAdd(P.sched, 1) : next;
          ptx::mbar_wait_suspend(&bars->sched_empty[sslot], sphase ^ 1);
          *(volatile int*)&bars->sched_tile[sslot] = tile < total_tiles ? tile : -1;
          ptx::mbar_arrive(&bars->sched_full[sslot]);
          if (++sslot == 4) { sslot = 0; sphase ^= 1; }
        }
        if (tile >= total_tiles) break;
        int m_tile, n_tile, seg_i;
        tile_decode(P, walk_mt, tile, m_tile, n_tile, seg_i);
        const TcSeg& sg = P.segs[seg_i];
        const CUtensorMap* am = &P.a_maps[sg.a_map];
        const CUtensorMap* bm = P.b_maps + sg.b_map;
        // the A operand streams from HBM: its k-block `pf` steps ahead (this tile's, or the next tile's) is pulled
        // into L2 now, so that the few shared-memory stages see L2 latency instead of HBM latency
        const int pf = P.a_prefetch < P.num_kb ? P.a_prefetch : P.num_kb;
        int nm_tile = 0, nn_tile = 0, nseg_i = 0;
        const bool has_next = next < total_tiles;
        if (pf > 0 && has_next) tile_decode(P, walk_mt, next, nm_tile, nn_tile, nseg_i);
        for (int kb = 0; kb < P.num_kb; ++kb) {
          if (pf > 0) {
            const bool same = kb + pf < P.num_kb;
            if (same || has_next) {
              const int pkb = same ? kb + pf : kb + pf - P.num_kb;
              const int pm = same ? m_tile : nm_tile;
              const TcSeg& ps = same ? sg : P.segs[nseg_i];
              if (P.a_kb_per_head > 0)
                ptx::tma_prefetch_l2_3d(&P.a_maps[ps.a_map], (pkb % P.a_kb_per_head) * BLOCK_K, pkb / P.a_kb_per_head, pm * BLOCK_M);
              else
                ptx::tma_prefetch_l2_3d(&P.a_maps[ps.a_map], pkb * BLOCK_K, pm * BLOCK_M, ps.a_z);
            }
          }
          ptx::mbar_wait_suspend(&bars->empty[stage], phase ^ 1);
          // A_CODES: the raw e4m3 tile [128 x 64 B] lands in the upper half of the stage and is expanded in place
          ptx::mbar_expect_tx(&bars->full[stage], (AMODE == A_CODES ? A_STAGE_BYTES / 2 : A_STAGE_BYTES) + b_stage_bytes);
          if (AMODE == A_CODES)
            ptx::tma_load_3d(smem_a + stage * A_STAGE_BYTES + A_STAGE_BYTES / 2, am, &bars->full[stage], kb * BLOCK_K,
                             m_tile * BLOCK_M, sg.a_z);
          else if (P.a_kb_per_head > 0)
            ptx::tma_load_3d(smem_a + stage * A_STAGE_BYTES, am, &bars->full[stage],
                             (kb % P.a_kb_per_head) * BLOCK_K, kb / P.a_kb_per_head, m_tile * BLOCK_M);
          else
            ptx::tma_load_3d(smem_a + stage * A_STAGE_BYTES, am, &bars->full[stage], kb * BLOCK_K,
                             m_tile * BLOCK_M, sg.a_z);
          ptx::tma_load_2d(smem_b + stage * b_stage_bytes, bm, &bars->full[stage], kb * BLOCK_K, n_tile * block_n);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        tile = next;
        next = after;
      }
      if (dyn) {                                  // the last CTA to stop claiming re-arms the counters for a later launch
        __threadfence();
        if (atomicAdd(P.sched + 1, 1) == (int)gridDim.x - 1) {
          P.sched[0] = 0;
          P.sched[1] = 0;
          __threadfence();
        }
      }
    }
  } else if (warp == 1) {
    // ============================== MMA issuer ==============================
    if (bres) {
      if (lane == 0) {
        const uint32_t idesc = ptx::umma_idesc_bf16(BLOCK_M, block_n);
        int stage = 0, it = 0;
        uint32_t phase = 0, groups = 0;                         // groups completed
        int m_tile, n_tile, seg_i;
        if (t_begin < t_end) tile_decode(P, walk_mt, t_begin, m_tile, n_tile, seg_i);
        int key = t_begin < t_end ? seg_i * P.n_tiles + n_tile : -1, prev_key = -1;
        for (int tile = t_begin; tile < t_end; ++tile, ++it) {
          int next_key = -1;
          if (tile + 1 < t_end) {
            tile_decode(P, walk_mt, tile + 1, m_tile, n_tile, seg_i);
            next_key = seg_i * P.n_tiles + n_tile;
          }
          const bool grp_first = key != prev_key, grp_last = next_key != key;
          const int acc = it & 1;
          ptx::mbar_wait_suspend(&bars->tmem_empty[acc], ((it >> 1) & 1) ^ 1);
          ptx::tc_fence_after();
          const uint32_t d_tmem = tmem_base + (uint32_t)(acc * 256);
          for (int kb = 0; kb < P.num_kb; ++kb) {
            if (grp_first) ptx::mbar_wait_suspend(&bars->b_full[kb], groups & 1);
            ptx::mbar_wait_suspend(&bars->full[stage], phase);
            ptx::tc_fence_after();
            const uint64_t da = ptx::umma_desc_sw128(ptx::smem_u32(smem_a + stage * A_STAGE_BYTES));
            const uint64_t db = ptx::umma_desc_sw128(ptx::smem_u32(smem_b + kb * b_stage_bytes));
#pragma unroll
            for (int k = 0; k < BLOCK_K / 16; ++k)
              ptx::mma_bf16(d_tmem, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, (kb | k) != 0);
            ptx::mma_commit(&bars->empty[stage]);
            if (grp_last) ptx::mma_commit(&bars->b_empty[kb]);   // the slot may take the next group's B tile
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
          ptx::mma_commit(&bars->tmem_full[acc]);
          if (grp_last) ++groups;
          prev_key = key;
          key = next_key;
        }
      }
    } else
    if (lane == 0 && cta_rank == 0) {
      const uint32_t idesc = ptx::umma_idesc_bf16(PAIR ? 2 * BLOCK_M : BLOCK_M, block_n);
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      int sslot = 0;
      uint32_t sphase = 0;
      for (int tile = walker; dyn || tile < total_tiles; tile += walk_stride, ++it) {
        if (dyn) {                                // the tile count is all this thread needs from the ring
          ptx::mbar_wait_suspend(&bars->sched_full[sslot], sphase);
          const int t = *(volatile int*)&bars->sched_tile[sslot];
          ptx::mbar_arrive(&bars->sched_empty[sslot]);
          if (++sslot == 4) { sslot = 0; sphase ^= 1; }
          if (t < 0) break;
        }
        const int acc = it & 1;
        const uint32_t acc_phase = (it >> 1) & 1;
        ptx::mbar_wait_suspend(&bars->tmem_empty[acc], acc_phase ^ 1);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(acc * 256);
        for (int kb = 0; kb < P.num_kb; ++kb) {
          ptx::mbar_wait_suspend(AMODE != A_PLAIN ? &bars->ready[stage] : &bars->full[stage], phase);
          ptx::tc_fence_after();
          const uint64_t da = ptx::umma_desc_sw128(ptx::smem_u32(smem_a + stage * A_STAGE_BYTES));
          const uint64_t db = ptx::umma_desc_sw128(ptx::smem_u32(smem_b + stage * b_stage_bytes));
#pragma unroll
          for (int k = 0; k < BLOCK_K / 16; ++k) {
            if (PAIR) ptx::mma_bf16_cg2(d_tmem, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, (kb | k) != 0);
            else ptx::mma_bf16(d_tmem, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, (kb | k) != 0);
          }
          if (PAIR) ptx::mma_commit_cg2(&bars->empty[stage]);      // frees the stage in both CTAs
          else ptx::mma_commit(&bars->empty[stage]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        if (PAIR) ptx::mma_commit_cg2(&bars->tmem_full[acc]);
        else ptx::mma_commit(&bars->tmem_full[acc]);
      }
    }
  }
  } else if (warp < 4 + NEPI) {
    // ============================== epilogue ==============================
    if (AMODE != A_PLAIN) ptx::setmaxnreg_inc<120>();
    // One token row per thread (TMEM lane); warps w and w+4 share a lane quadrant and split the
    // tile's work into two groups (columns, or RoPE frequencies for 2-head K tiles).  Per group:
    // TMEM -> registers -> fused math -> swizzled per-warp staging -> coalesced 16-B stores.
    // The per-row quantities of the NEXT tile (position, slot, scales, mean slice) are fetched
    // while the current tile is processed.
    const int ew = (warp - 4) & 3;                    // TMEM lane quadrant (= warp % 4)
    const int grp = (warp - 4) >> 2;                  // group 0 / 1
    const int half = P.head_dim / 2;
    const uint32_t stg = ptx::smem_u32(smem_stg + (warp - 4) * P.stg_warp_bytes);
    const uint32_t wvec = ptx::smem_u32(smem_vec + (warp - 4) * VEC_WARP_BYTES);
    const int out_eb = (EPI == EPI_CODES && P.code_dtype == SCD_E4M3_ROWSCALE) ? 1 : 2;
    // column split only when both halves keep whole heads (RoPE) and whole 32-column TMEM chunks
    const int gran = (EPI == EPI_KV && P.head_dim > 32) ? P.head_dim : 32;
    const bool split_cols = (block_n % (2 * gran)) == 0;
    const int grp_cols = split_cols ? block_n / 2 : block_n;

    struct RowInfo {
      int pos;
      float rs;
      unsigned long long row_ptr;                     // global address of this row's first tile column (0 = no row)
      float4 m0, m1;                                  // this lane's share of the tile's mean / bias slice
    };
    auto fetch = [&](int tile) -> RowInfo {
      RowInfo ri;
      ri.pos = 0; ri.rs = 1.0f; ri.row_ptr = 0ull;
      ri.m0 = make_float4(0.f, 0.f, 0.f, 0.f); ri.m1 = ri.m0;
      int m_tile, n_tile, seg_i;
      tile_decode(P, walk_mt, tile, m_tile, n_tile, seg_i);
      if (PAIR) m_tile = 2 * m_tile + (int)cta_rank;
      const TcSeg& sg = P.segs[seg_i];
      const int row = m_tile * BLOCK_M + ew * 32 + lane;
      const int n0 = n_tile * block_n;
      if (sg.col_vec) {
        ri.m0 = ldg_f4(sg.col_vec + n0 + lane * 4);
        if (block_n > 128) ri.m1 = ldg_f4(sg.col_vec + n0 + 128 + lane * 4);
      }
      if (row < P.M) {
        if (EPI == EPI_KV) {
          long long slot;
          row_to_pos_slot(P.batch, row, ri.pos, slot);
          const bool to1 = n0 >= P.split;
          if (slot >= 0)                                  // -1: page id outside the pool -> the row is not written
            ri.row_ptr = (unsigned long long)(to1 ? sg.out1 : sg.out0) +
                         ((unsigned long long)slot * P.pool_width + (to1 ? n0 - P.split : n0)) * 2ull;
        } else {
          ri.row_ptr = (unsigned long long)sg.out0 + ((unsigned long long)row * P.N + n0) * (unsigned long long)out_eb;
        }
        if ((EPI == EPI_KV || EPI == EPI_ACT) && sg.a_scale) ri.rs = __ldg(sg.a_scale + row);
        if (EPI == EPI_KV && sg.rowscale_in) {
          float ss = 0.0f;
          for (int p = 0; p < P.n_partials; ++p) ss += __ldg(sg.rowscale_in + (size_t)p * P.M + row);
          ri.rs *= rsqrtf(ss / (float)P.rms_dim + P.rms_eps);
        }
      }
      return ri;
    };

    // hand an accumulator buffer back to the MMA thread (PAIR: the leader's barrier collects both CTAs' warps)
    auto release_acc = [&](int acc) {
      if (PAIR) ptx::mbar_arrive_cluster(ptx::mapa(ptx::smem_u32(&bars->tmem_empty[acc]), 0));
      else ptx::mbar_arrive(&bars->tmem_empty[acc]);
    };
    if (bres) {
      // ---- PATCH GEMM-1, B-resident walk: consecutive tiles are consecutive m-tiles of one (segment, n-tile), so the tile
      // coordinates advance without divisions and the warp's 64-entry bias slice is staged once per (segment, n-tile) ----
      constexpr int CW = 256 / (NEPI / 4), PASSES = CW / 64;
      int m_tile = 0, n_tile = 0, seg_i = 0, prev_key = -1;
      if (t_begin < t_end) tile_decode(P, walk_mt, t_begin, m_tile, n_tile, seg_i);
      const bool silu = P.act == SCD_ACT_SILU;
      int it = 0;
      for (int tile = t_begin; tile < t_end; ++tile, ++it) {
        const TcSeg& sg = P.segs[seg_i];
        const int n0 = n_tile * block_n;
        const int key = seg_i * P.n_tiles + n_tile;
        if (key != prev_key) {
          prev_key = key;
          __syncwarp();
          for (int i = lane; i < CW / 4; i += 32) {
            float4 b4 = sg.col_vec ? ldg_f4(sg.col_vec + n0 + grp * CW + i * 4) : make_float4(0.f, 0.f, 0.f, 0.f);
            if (silu) { b4.x *= 0.5f; b4.y *= 0.5f; b4.z *= 0.5f; b4.w *= 0.5f; }   // SiLU works on h = x / 2
            asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(wvec + i * 16), "f"(b4.x), "f"(b4.y), "f"(b4.z), "f"(b4.w) : "memory");
          }
          __syncwarp();
        }
        const int acc = it & 1;
        ptx::mbar_wait_suspend(&bars->tmem_full[acc], (it >> 1) & 1);
        ptx::tc_fence_after();
        const uint32_t t_row = tmem_base + (uint32_t)(acc * 256) + ((uint32_t)(ew * 32) << 16);
        const int row0 = m_tile * BLOCK_M + ew * 32;
        const unsigned long long out_q = (unsigned long long)sg.out0 + ((unsigned long long)row0 * P.N + n0 + grp * CW) * 2ull;
#pragma unroll
        for (int ps = 0; ps < PASSES; ++ps) {
          if (silu) act_stage64<true>(t_row + grp * CW + ps * 64, stg, wvec + ps * 256, 0.5f, lane);
          else act_stage64<false>(t_row + grp * CW + ps * 64, stg, wvec + ps * 256, 1.0f, lane);
          if (ps == PASSES - 1) ptx::tc_fence_before();
          __syncwarp();
          if (ps == PASSES - 1 && lane == 0) release_acc(acc);
          rowmajor_copy_out_128(stg, out_q + (unsigned long long)ps * 128ull, (unsigned long long)P.N * 2ull, P.M - row0, lane);
          __syncwarp();
        }
        if (++m_tile == walk_mt) {                              // plain m-fastest order (the host checks msb >= m-tiles)
          m_tile = 0;
          if (++n_tile == P.n_tiles) { n_tile = 0; ++seg_i; }
        }
      }
    } else {
    int it = 0;
    RowInfo cur;
    int sslot = 0;
    uint32_t sphase = 0;
    if (!dyn && t_begin < t_end) cur = fetch(t_begin);
    for (int tile = t_begin; dyn || tile < t_end; tile += t_step, ++it) {
      if (dyn) {                                  // claimed tiles arrive through the ring; no look-ahead on the next one
        ptx::mbar_wait_suspend(&bars->sched_full[sslot], sphase);
        tile = *(volatile int*)&bars->sched_tile[sslot];
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&bars->sched_empty[sslot]);
        if (++sslot == 4) { sslot = 0; sphase ^= 1; }
        if (tile < 0) break;
        cur = fetch(tile);
      }
      int m_tile, n_tile, seg_i;
      tile_decode(P, walk_mt, tile, m_tile, n_tile, seg_i);
      if (PAIR) m_tile = 2 * m_tile + (int)cta_rank;
      const TcSeg& sg = P.segs[seg_i];
      const int acc = it & 1;
      const uint32_t acc_phase = (it >> 1) & 1;
      const int row = m_tile * BLOCK_M + ew * 32 + lane;
      const bool valid = row < P.M;
      const int n0 = n_tile * block_n;
      const int n_end = min(block_n, P.N - n0);              // valid columns in this tile
      const int g_begin = grp * grp_cols;                     // this warp's columns [g_begin, g_end) of the tile
      const int g_end = min(n_end, g_begin + grp_cols);
      const bool has_work = (grp == 0 || split_cols) && g_begin < n_end;
      const int pos = cur.pos;
      const float rs = cur.rs;
      const unsigned long long row_ptr = cur.row_ptr;

      // this warp's copy of the tile's mean / bias slice: wvec[c] for tile column c
      // PATCH GEMM-1 fast path (below): whole 256-column tiles of the aligner's first layer
      const bool act_fast = EPI == EPI_ACT && block_n == 256 && n_end == 256;
      __syncwarp();
      if (vec_smem) {
      if (act_fast && P.act == SCD_ACT_SILU) {             // SiLU works on h = x / 2: the bias is staged halved
        cur.m0.x *= 0.5f; cur.m0.y *= 0.5f; cur.m0.z *= 0.5f; cur.m0.w *= 0.5f;
        cur.m1.x *= 0.5f; cur.m1.y *= 0.5f; cur.m1.z *= 0.5f; cur.m1.w *= 0.5f;
      }
      asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(wvec + lane * 16), "f"(cur.m0.x), "f"(cur.m0.y),
                   "f"(cur.m0.z), "f"(cur.m0.w) : "memory");
      asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(wvec + 512 + lane * 16), "f"(cur.m1.x), "f"(cur.m1.y),
                   "f"(cur.m1.z), "f"(cur.m1.w) : "memory");
      }
      __syncwarp();

      ptx::mbar_wait_suspend(&bars->tmem_full[acc], acc_phase);
      ptx::tc_fence_after();
      const uint32_t t_row = tmem_base + (uint32_t)(acc * 256) + ((uint32_t)(ew * 32) << 16);

      // prefetch the next tile's per-row quantities; consumed at the bottom of the loop
      RowInfo nxt = cur;
      if (!dyn && tile + t_step < t_end) nxt = fetch(tile + t_step);

      if (EPI == EPI_KV && n0 < sg.rope_cols && P.rope_style == SCD_ROPE_HALF && P.head_dim == 128 && block_n == 256 &&
          n_end == 256) {
        // ---- 2-head K tile: frequency split between the warp pair ----
        if (P.kv_compact) {
          const float* bias = sg.col_vec ? sg.col_vec + n0 : nullptr;
          if (grp == 0) rope_tile_h128_compact<0>(P, t_row, stg, bias, pos, rs, row_ptr, lane);
          else rope_tile_h128_compact<1>(P, t_row, stg, bias, pos, rs, row_ptr, lane);
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) release_acc(acc);
          cur = nxt;
          continue;
        }
        if (grp == 0) rope_tile_h128<0>(P, t_row, stg, wvec, pos, rs, lane);
        else rope_tile_h128<1>(P, t_row, stg, wvec, pos, rs, lane);
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) release_acc(acc);
        if (grp == 0) rope_tile_h128_copy_out<0>(stg, row_ptr, lane);
        else rope_tile_h128_copy_out<1>(stg, row_ptr, lane);
        cur = nxt;
        continue;
      }

      if (act_fast) {
        // ---- PATCH GEMM-1: TMEM -> scale / bias / SiLU -> bf16 -> staging, accumulator handed back, row-major copy-out ----
        // warp (quadrant ew, group grp) owns columns [grp * cw, (grp + 1) * cw), cw = 64 (sixteen warps) or 128 (eight)
        constexpr int CW = 256 / (NEPI / 4), PASSES = CW / 64;
        const int row0 = m_tile * BLOCK_M + ew * 32;
        const unsigned long long out_q = (unsigned long long)sg.out0 + ((unsigned long long)row0 * P.N + n0 + grp * CW) * 2ull;
#pragma unroll
        for (int ps = 0; ps < PASSES; ++ps) {
          const int c0 = grp * CW + ps * 64;
          if (P.act == SCD_ACT_SILU) act_stage64<true>(t_row + c0, stg, wvec + c0 * 4, 0.5f * rs, lane);
          else act_stage64<false>(t_row + c0, stg, wvec + c0 * 4, rs, lane);
          if (ps == PASSES - 1) ptx::tc_fence_before();
          __syncwarp();
          if (ps == PASSES - 1 && lane == 0) release_acc(acc);
          rowmajor_copy_out_128(stg, out_q + (unsigned long long)ps * 128ull, (unsigned long long)P.N * 2ull, P.M - row0, lane);
          __syncwarp();
        }
        cur = nxt;
        continue;
      }

      // e4m3 codes: the row scale needs the amax over all of N first (tile spans N).  Columns
      // beyond N hold acc = 0 (zero-filled operand rows) and c = 0 (padded vector): no masks needed.
      float e4_scale = 1.0f, e4_inv = 1.0f;
      if (EPI == EPI_CODES && P.code_dtype == SCD_E4M3_ROWSCALE && has_work) {
        float amax = 0.0f;
        for (int c = 0; c < n_end; c += 32) {
          uint32_t r[32];
          ptx::tmem_ld32(t_row + c, r);
          ptx::tmem_ld_wait();
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            const float4 m4 = vec_smem ? ptx::lds_f4(wvec + (c + q * 4) * 4)
                                       : (sg.col_vec ? ldg_f4(sg.col_vec + n0 + c + q * 4) : make_float4(0.f, 0.f, 0.f, 0.f));
            amax = fmaxf(amax, fmaxf(fmaxf(fabsf(__uint_as_float(r[q * 4]) - m4.x), fabsf(__uint_as_float(r[q * 4 + 1]) - m4.y)),
                                     fmaxf(fabsf(__uint_as_float(r[q * 4 + 2]) - m4.z), fabsf(__uint_as_float(r[q * 4 + 3]) - m4.w))));
          }
        }
        e4_scale = amax > 0.0f ? amax / 448.0f : 1.0f;
        if (valid && grp == 0) sg.aux[row] = e4_scale;
        e4_inv = __fdiv_rn(1.0f, e4_scale);     // one division per row; the codes multiply (<= 1.5 ulp of fp32 from z / s)
      }
      float ss_u = 0.0f;

      if (!has_work) {                                        // nothing to read: release the accumulator
        if (EPI == EPI_U && valid && sg.aux) sg.aux[(size_t)(n_tile * 2 + grp) * P.M + row] = 0.0f;
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) release_acc(acc);
        cur = nxt;
        continue;
      }
      for (int c0 = g_begin; c0 < g_end; c0 += P.sub_n) {
        const int sub_cols = min(P.sub_n, g_begin + grp_cols - c0);
        const int row_bytes = sub_cols * out_eb;
        const int pitch = (row_bytes + 127) & ~127;            // whole 128-B swizzle spans
        const bool last_sub = c0 + P.sub_n >= g_end;

        if (EPI == EPI_KV && (n0 + c0) < sg.rope_cols && P.rope_style == SCD_ROPE_HALF) {
          // ---- RoPE, HALF pairing (generic): heads of this sub-tile, 16 pairs at a time ----
          for (int hc = 0; hc < sub_cols; hc += P.head_dim)
            for (int j0 = 0; j0 < half; j0 += 16) {
              uint32_t ra[16], rb[16];
              ptx::tmem_ld16(t_row + c0 + hc + j0, ra);
              ptx::tmem_ld16(t_row + c0 + hc + half + j0, rb);
              ptx::tmem_ld_wait();
              uint32_t oa[8], ob[8];
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                const float4 ma = ptx::lds_f4(wvec + (c0 + hc + j0 + q * 4) * 4);
                const float4 mb = ptx::lds_f4(wvec + (c0 + hc + half + j0 + q * 4) * 4);
                const float am[4] = {ma.x, ma.y, ma.z, ma.w}, bm[4] = {mb.x, mb.y, mb.z, mb.w};
                float va[4], vb[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                  const int i = q * 4 + e;
                  const float2 cs = rope_cs(pos, P.rope_g[j0 + i]);
                  const float a = fmaf(__uint_as_float(ra[i]), rs, am[e]);
                  const float b = fmaf(__uint_as_float(rb[i]), rs, bm[e]);
                  va[e] = a * cs.x - b * cs.y;
                  vb[e] = b * cs.x + a * cs.y;
                }
                oa[q * 2] = pack_bf16x2(va[0], va[1]); oa[q * 2 + 1] = pack_bf16x2(va[2], va[3]);
                ob[q * 2] = pack_bf16x2(vb[0], vb[1]); ob[q * 2 + 1] = pack_bf16x2(vb[2], vb[3]);
              }
              const int ca = (hc + j0) >> 3, cb = (hc + half + j0) >> 3;
              stg_put(stg, pitch, lane, ca, make_uint4(oa[0], oa[1], oa[2], oa[3]));
              stg_put(stg, pitch, lane, ca + 1, make_uint4(oa[4], oa[5], oa[6], oa[7]));
              stg_put(stg, pitch, lane, cb, make_uint4(ob[0], ob[1], ob[2], ob[3]));
              stg_put(stg, pitch, lane, cb + 1, make_uint4(ob[4], ob[5], ob[6], ob[7]));
            }
        } else {
          // ---- 32 columns at a time: plain epilogues, or INTERLEAVED RoPE (adjacent pairs) ----
          // SiLU(v) = v (1/2 + 1/2 tanh(v/2)) = h + h tanh(h) with h = v/2: the halving rides on the scale / bias FMA
          const bool silu = EPI == EPI_ACT && P.act == SCD_ACT_SILU;
          const float rsh = silu ? 0.5f * rs : rs;
          const unsigned long long rs2 = f2_pack(rsh, rsh);
          const unsigned long long half2 = f2_pack(0.5f, 0.5f);
          for (int c = c0; c < c0 + sub_cols; c += 32) {
            uint32_t r[32];
            ptx::tmem_ld32(t_row + c, r);
            ptx::tmem_ld_wait();
            float v[32];
#pragma unroll
            for (int q = 0; q < 8; ++q) {
              const float4 m4 = vec_smem ? ptx::lds_f4(wvec + (c + q * 4) * 4)
                                         : (sg.col_vec ? ldg_f4(sg.col_vec + n0 + c + q * 4) : make_float4(0.f, 0.f, 0.f, 0.f));
              if (EPI == EPI_CODES) {
                v[q * 4] = __uint_as_float(r[q * 4]) - m4.x; v[q * 4 + 1] = __uint_as_float(r[q * 4 + 1]) - m4.y;
                v[q * 4 + 2] = __uint_as_float(r[q * 4 + 2]) - m4.z; v[q * 4 + 3] = __uint_as_float(r[q * 4 + 3]) - m4.w;
              } else {
                unsigned long long b01 = f2_pack(m4.x, m4.y), b23 = f2_pack(m4.z, m4.w);
                if (silu) { b01 = f2_mul(b01, half2); b23 = f2_mul(b23, half2); }
                f2_unpack(f2_fma(f2_pack(__uint_as_float(r[q * 4]), __uint_as_float(r[q * 4 + 1])), rs2, b01), v[q * 4], v[q * 4 + 1]);
                f2_unpack(f2_fma(f2_pack(__uint_as_float(r[q * 4 + 2]), __uint_as_float(r[q * 4 + 3])), rs2, b23), v[q * 4 + 2], v[q * 4 + 3]);
              }
            }
            if (EPI == EPI_ACT && P.act == SCD_ACT_SILU) {
#pragma unroll
              for (int i = 0; i < 32; ++i) {      // v[i] holds h = x / 2: x sigmoid(x) = h + h tanh(h), one MUFU op (2^-11 rel.)
                float t;
                asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(v[i]));
                v[i] = fmaf(v[i], t, v[i]);
              }
            }
            if (EPI == EPI_U) {
#pragma unroll
              for (int i = 0; i < 32; ++i) ss_u = fmaf(v[i], v[i], ss_u);
            }
            if (EPI == EPI_KV && (n0 + c) < sg.rope_cols) {
              const int f0 = ((n0 + c) % P.head_dim) >> 1;
#pragma unroll
              for (int i = 0; i < 16; ++i) {
                const float2 cs = rope_cs(pos, P.rope_g[f0 + i]);
                const float a = v[2 * i], b = v[2 * i + 1];
                v[2 * i] = a * cs.x - b * cs.y;
                v[2 * i + 1] = b * cs.x + a * cs.y;
              }
            }
            if (EPI == EPI_CODES && P.code_dtype == SCD_E4M3_ROWSCALE) {
#pragma unroll
              for (int q = 0; q < 2; ++q) {
                uint32_t w[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                  w[e] = float2_to_e4m3x2_sat(v[q * 16 + e * 4] * e4_inv, v[q * 16 + e * 4 + 1] * e4_inv) |
                         (float2_to_e4m3x2_sat(v[q * 16 + e * 4 + 2] * e4_inv, v[q * 16 + e * 4 + 3] * e4_inv) << 16);
                }
                stg_put(stg, pitch, lane, ((c - c0) >> 4) + q, make_uint4(w[0], w[1], w[2], w[3]));
              }
            } else {
#pragma unroll
              for (int q = 0; q < 4; ++q)
                stg_put(stg, pitch, lane, ((c - c0) >> 3) + q,
                        make_uint4(pack_bf16x2(v[q * 8], v[q * 8 + 1]), pack_bf16x2(v[q * 8 + 2], v[q * 8 + 3]),
                                   pack_bf16x2(v[q * 8 + 4], v[q * 8 + 5]), pack_bf16x2(v[q * 8 + 6], v[q * 8 + 7])));
            }
          }
        }
        if (last_sub) {
          // all TMEM reads of this tile are done: hand the accumulator back before the copy-out
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) release_acc(acc);
        } else {
          __syncwarp();
        }
        // valid bytes: the N tail, and never more than this warp staged (a 96-column group rounds its lanes-per-row
        // up to 16 chunks; the 4 extra chunks are the other group's columns)
        stg_copy_out(stg, pitch, row_bytes, min(row_bytes, (n_end - c0) * out_eb), row_ptr, (unsigned long long)c0 * out_eb, lane,
                     EPI == EPI_KV || EPI == EPI_CODES);
        __syncwarp();
      }
      if (EPI == EPI_U && valid && sg.aux) sg.aux[(size_t)(n_tile * 2 + grp) * P.M + row] = ss_u;
      cur = nxt;
    }
    }
  } else if (AMODE == A_CODES) {
    // ============================== A transform: e4m3 -> bf16 in shared memory ==============================
    // The raw tile (row-major, 64 B per token row) sits in bytes [8192, 16384) of the stage.  Thread (row, quarter)
    // takes 16 codes, all 512 threads meet (the expansion overwrites the raw bytes), then it writes chunks
    // 2 quarter, 2 quarter + 1 of the row in the 128-byte-swizzled K-major layout the MMA descriptor expects.
    // e4m3 s.eeee.mmm -> bf16 s.0000eeee.mmm0000 is the same number times 2^-120 (normals and subnormals alike);
    // one exact bf16 multiply by 2^120 finishes the conversion.  The row scale is applied in the epilogue.
    ptx::setmaxnreg_dec<56>();
    const int dt = threadIdx.x - (4 + EPI_WARPS) * 32;
    const int row = dt >> 2, qt = dt & 3;
    const uint32_t src_off = A_STAGE_BYTES / 2 + (uint32_t)dt * 16;
    const uint32_t row_off = (uint32_t)(row >> 3) * 1024 + (uint32_t)(row & 7) * 128;
    const uint32_t dst0 = row_off + (uint32_t)(((2 * qt) ^ (row & 7)) << 4), dst1 = row_off + (uint32_t)(((2 * qt + 1) ^ (row & 7)) << 4);
    const uint32_t a_base = ptx::smem_u32(smem_a);
    int stage = 0;
    uint32_t phase = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
      for (int kb = 0; kb < P.num_kb; ++kb) {
        ptx::mbar_wait_suspend(&bars->full[stage], phase);
        const uint32_t sb = a_base + (uint32_t)stage * A_STAGE_BYTES;
        const uint4 raw = ptx::lds128(sb + src_off);
        ptx::named_bar_sync(1, DEROPE_WARPS * 32);
        const uint32_t w[4] = {raw.x, raw.y, raw.z, raw.w};
        uint32_t o[8];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          o[2 * i] = e4m3x2_to_bf16x2(__byte_perm(w[i], 0u, 0x1404));       // bytes 0, 1 -> high bytes of two halves
          o[2 * i + 1] = e4m3x2_to_bf16x2(__byte_perm(w[i], 0u, 0x3424));   // bytes 2, 3
        }
        ptx::sts128(sb + dst0, make_uint4(o[0], o[1], o[2], o[3]));
        ptx::sts128(sb + dst1, make_uint4(o[4], o[5], o[6], o[7]));
        ptx::fence_proxy_async_smem();
        ptx::mbar_arrive(&bars->ready[stage]);
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
    }
  } else if (AMODE == A_DEROPE) {
    // ============================== A transform: deRoPE in shared memory ==============================
    ptx::setmaxnreg_dec<56>();
    // Four threads per token row (the rotation, not the MMA, is what has to keep up with HBM here).  A k-block
    // row is 128 B = 8 chunks of 16 B, chunk c stored at position c ^ (row & 7) (128-byte swizzle).  Channel
    // pairs (j, j + d_h/2) of a head:
    //   d_h = 128: same chunk / element of two consecutive k-blocks (stages s, s+1)
    //   d_h =  64: chunks c and c + 4 of one k-block;  d_h = 32: chunks c and c + 2 (two heads per block)
    // Thread `sp` of a row owns `per` of the `pair_chunks` "a"-half chunks (8 frequencies each); its (cos, sin)
    // of the row's position are computed once per tile and kept in registers.
    const int dt = threadIdx.x - (4 + EPI_WARPS) * 32;
    const int tr = dt & 127;                                            // row in tile
    const int sp = dt >> 7;                                             // 0..3
    const int half = P.head_dim / 2;
    const int step = P.head_dim == 128 ? 2 : 1;                         // k-blocks consumed per iteration
    const int pair_chunks = P.head_dim == 128 ? 8 : half / 8;           // chunks in the "a" half: 8 / 4 / 2
    const int groups = P.head_dim == 128 ? 1 : BLOCK_K / P.head_dim;    // heads per k-block
    const int nsplit = pair_chunks < 4 ? pair_chunks : 4;
    const int per = pair_chunks / nsplit;                               // 2 / 1 / 1
    const bool active = sp < nsplit;
    const uint32_t row_off = (uint32_t)(tr >> 3) * 1024 + (uint32_t)(tr & 7) * 128;
    int stage = 0;
    uint32_t phase = 0;
    if (P.head_dim == 128) {
      // d_h = 128 (every BASELINE model): thread sp owns chunks 2sp, 2sp+1 of the "a" k-block and of the "b" k-block that
      // follows it, i.e. frequencies [16 sp, 16 sp + 16).  Shared-space 16-B accesses, (cos, sin) as fp32 pairs in
      // registers, the rotation in packed fp32 (2 FMUL2 + 2 FFMA2 per two channel pairs).
      const uint32_t a0 = ptx::smem_u32(smem_a) + row_off;
      const uint32_t sw = (uint32_t)(tr & 7);
      const uint32_t off0 = ((uint32_t)(2 * sp) ^ sw) << 4, off1 = ((uint32_t)(2 * sp + 1) ^ sw) << 4;
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        int m_tile, n_tile_unused, seg_unused;
        tile_decode(P, walk_mt, tile, m_tile, n_tile_unused, seg_unused);
        const int row = m_tile * BLOCK_M + tr;
        int pos = 0;
        long long slot;
        if (row < P.M) row_to_pos_slot(P.batch, row, pos, slot);
        unsigned long long cc[8], ss[8];                  // (cos_j, cos_j+1), (sin_j, sin_j+1), j = 16 sp + 2 i
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const float2 v0 = rope_cs(pos, P.rope_g[sp * 16 + 2 * i]), v1 = rope_cs(pos, P.rope_g[sp * 16 + 2 * i + 1]);
          cc[i] = f2_pack(v0.x, v1.x);
          ss[i] = f2_pack(v0.y, v1.y);
        }
        for (int kb = 0; kb < P.num_kb; kb += 2) {
          const int s0 = stage, s1 = stage + 1 == STAGES ? 0 : stage + 1;
          ptx::mbar_wait_suspend(&bars->full[s0], phase);
          ptx::mbar_wait_suspend(&bars->full[s1], (s1 == 0) ? (phase ^ 1) : phase);
          const uint32_t ra = a0 + (uint32_t)s0 * A_STAGE_BYTES, rb = a0 + (uint32_t)s1 * A_STAGE_BYTES;
#pragma unroll
          for (int c = 0; c < 2; ++c) {
            const uint32_t off = c == 0 ? off0 : off1;
            uint4 xa = ptx::lds128(ra + off), xb = ptx::lds128(rb + off);
            uint32_t* wa = reinterpret_cast<uint32_t*>(&xa);
            uint32_t* wb = reinterpret_cast<uint32_t*>(&xb);
#pragma unroll
            for (int w = 0; w < 4; ++w) {
              const unsigned long long a2 = f2_pack(__uint_as_float(wa[w] << 16), __uint_as_float(wa[w] & 0xffff0000u));
              const unsigned long long b2 = f2_pack(__uint_as_float(wb[w] << 16), __uint_as_float(wb[w] & 0xffff0000u));
              // rotation by -phi:  a' = a cos + b sin ; b' = b cos - a sin
              const unsigned long long na = f2_fma(a2, cc[c * 4 + w], f2_mul(b2, ss[c * 4 + w]));
              const unsigned long long nb = f2_fma(b2, cc[c * 4 + w], f2_neg(f2_mul(a2, ss[c * 4 + w])));
              float a_lo, a_hi, b_lo, b_hi;
              f2_unpack(na, a_lo, a_hi);
              f2_unpack(nb, b_lo, b_hi);
              wa[w] = pack_bf16x2(a_lo, a_hi);
              wb[w] = pack_bf16x2(b_lo, b_hi);
            }
            ptx::sts128(ra + off, xa);
            ptx::sts128(rb + off, xb);
          }
          ptx::fence_proxy_async_smem();
          ptx::mbar_arrive(&bars->ready[s0]);
          ptx::mbar_arrive(&bars->ready[s1]);
          for (int q = 0; q < 2; ++q)
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    } else
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
      int m_tile, n_tile_unused, seg_unused;
      tile_decode(P, walk_mt, tile, m_tile, n_tile_unused, seg_unused);
      const int row = m_tile * BLOCK_M + tr;
      int pos = 0;
      long long slot;
      if (row < P.M && active) row_to_pos_slot(P.batch, row, pos, slot);
      __half2 cs[16];                                   // fp16 (2^-12 abs) is below the bf16 operand rounding
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const int f = sp * per * 8 + j;
        const float2 v = (active && j < per * 8) ? rope_cs(pos, P.rope_g[f & 63]) : make_float2(1.f, 0.f);
        cs[j] = __floats2half2_rn(v.x, v.y);
      }
      for (int kb = 0; kb < P.num_kb; kb += step) {
        const int s0 = stage, s1 = (stage + 1) % STAGES;
        ptx::mbar_wait_suspend(&bars->full[s0], phase);
        if (step == 2) ptx::mbar_wait_suspend(&bars->full[s1], (s1 == 0) ? (phase ^ 1) : phase);
        if (active) {
          uint8_t* ra = smem_a + s0 * A_STAGE_BYTES + row_off;
          uint8_t* rb = step == 2 ? smem_a + s1 * A_STAGE_BYTES + row_off : ra;
          for (int gidx = 0; gidx < groups; ++gidx)
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              if (c >= per) break;
              const int cl = sp * per + c;                            // chunk within the "a" half
              const int ca = P.head_dim == 128 ? cl : gidx * (P.head_dim / 8) + cl;
              const int cb = P.head_dim == 128 ? cl : ca + pair_chunks;
              uint4* pa = reinterpret_cast<uint4*>(ra + ((ca ^ (tr & 7)) << 4));
              uint4* pb = reinterpret_cast<uint4*>(rb + ((cb ^ (tr & 7)) << 4));
              uint4 xa = *pa, xb = *pb;
              uint32_t* wa = reinterpret_cast<uint32_t*>(&xa);
              uint32_t* wb = reinterpret_cast<uint32_t*>(&xb);
#pragma unroll
              for (int w = 0; w < 4; ++w) {
                const float2 a2 = __bfloat1622float2(*reinterpret_cast<__nv_bfloat162*>(&wa[w]));
                const float2 b2 = __bfloat1622float2(*reinterpret_cast<__nv_bfloat162*>(&wb[w]));
                const float2 c0 = __half22float2(cs[c * 8 + 2 * w]), c1 = __half22float2(cs[c * 8 + 2 * w + 1]);
                // rotation by -phi:  a' = a cos + b sin ; b' = b cos - a sin
                wa[w] = pack_bf16x2(a2.x * c0.x + b2.x * c0.y, a2.y * c1.x + b2.y * c1.y);
                wb[w] = pack_bf16x2(b2.x * c0.x - a2.x * c0.y, b2.y * c1.x - a2.y * c1.y);
              }
              *pa = xa;
              *pb = xb;
            }
          ptx::fence_proxy_async_smem();
        }
        ptx::mbar_arrive(&bars->ready[s0]);
        if (step == 2) ptx::mbar_arrive(&bars->ready[s1]);
        for (int q = 0; q < step; ++q)
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
    }
  }

  // ============================== teardown ==============================
  ptx::tc_fence_before();
  if (P.dep_wait_late && threadIdx.x == 0) ptx::grid_dep_wait();
  if (PAIR) {
    ptx::cluster_sync();                // neither CTA leaves while the other may still signal its barriers / read its TMEM
    if (warp == 2) ptx::tmem_dealloc_cg2<TMEM_COLS>(tmem_base);
  } else {
    __syncthreads();
    if (warp == 2) ptx::tmem_dealloc<TMEM_COLS>(tmem_base);
  }
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

// scd_fit.cu: bf16 matrix [rows][cols] (cols contiguous, row pitch in bytes), box {64, box_rows}, 128-B swizzle
scd_status_t tc_make_map_2d_bf16(CUtensorMap* m, const void* base, uint64_t cols, uint64_t rows, uint64_t row_pitch_bytes,
                                 uint32_t box_rows) {
  return make_map(m, base, cols, rows, 1, row_pitch_bytes, row_pitch_bytes * rows, box_rows, 1);
}

// paged producer pool [n_slots][width] (row pitch in bytes): 2-D, box {64, 1} for tile::gather4, 128-B swizzle
static scd_status_t make_gather_map(CUtensorMap* m, const void* base, uint64_t width, uint64_t n_slots, uint64_t pitch_bytes,
                                    uint32_t box_rows = 1) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return fail(SCD_E_CUDA, "cuTensorMapEncodeTiled entry point not found");
  cuuint64_t dims[2] = {width, n_slots};
  cuuint64_t strides[1] = {pitch_bytes};
  cuuint32_t box[2] = {BLOCK_K, box_rows};
  cuuint32_t es[2] = {1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, es,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(SCD_E_CUDA, "cuTensorMapEncodeTiled (gather %llu x %llu) failed (%d)", (unsigned long long)n_slots,
                                     (unsigned long long)width, (int)r);
  return SCD_OK;
}

// e4m3 code segments [n_seg][T][r] (1 byte per code): box {64, 128, 1}, no swizzle (expanded in shared memory)
static scd_status_t make_code_map_u8(CUtensorMap* m, const void* base, uint64_t r, uint64_t T, uint64_t n_seg,
                                     uint64_t seg_stride) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return fail(SCD_E_CUDA, "cuTensorMapEncodeTiled entry point not found");
  cuuint64_t dims[3] = {r, T, n_seg};
  cuuint64_t strides[2] = {r, seg_stride};
  cuuint32_t box[3] = {BLOCK_K, BLOCK_M, 1};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult rc = fn(m, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(base), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (rc != CUDA_SUCCESS)
    return fail(SCD_E_CUDA, "cuTensorMapEncodeTiled (u8 codes %llu x %llu x %llu) failed (%d)", (unsigned long long)r,
                (unsigned long long)T, (unsigned long long)n_seg, (int)rc);
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

#ifndef G3_GENERIC
#define G3_GENERIC 1
#endif
#ifndef TC_PAIRS
#define TC_PAIRS 1
#endif
#ifndef TC_ENC_PAIRS
#define TC_ENC_PAIRS 1
#endif
#ifndef TC_ENC_DYN
#define TC_ENC_DYN 1
#endif
#ifndef TC_ENC_OVERLAP
#define TC_ENC_OVERLAP 1
#endif
#ifndef TC_G1_BRES
#define TC_G1_BRES 1
#endif
#ifndef TC_A_PREFETCH
#define TC_A_PREFETCH 4
#endif
static int pick_block_n_div(int n) {            // largest tile width that divides n (paged / split epilogues)
  for (int b : {256, 128, 64, 32})
    if (n % b == 0) return b;
  return 0;
}
// Smallest multiple of 32 covering n, capped at 256.  32, not the MMA's own granularity of 16: the epilogue reads TMEM
// in 32-column chunks, and TMEM is not cleared between kernels -- every column it reads must have been written by this
// tile's MMA (columns in [N, block_n) are written as exact zeros: their B rows are zero-filled by the TMA).
static int pick_block_n_cover(int n) {
  int b = (n + 31) / 32 * 32;
  return b > 256 ? 256 : b;
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
  // + per PATCH layer: W2^T and [W_k ; W_v] with 128-row boxes, + per segment the encoder with half-tile boxes (CTA pairs)
  std::vector<CUtensorMap> maps((size_t)3 * nseg + 5 * np);
  memset(maps.data(), 0, maps.size() * sizeof(CUtensorMap));
  scd_status_t st;
  for (int i = 0; i < nseg; ++i) {
    const SegPlan& sp = p->segs[i];
    if ((st = make_b_map(&maps[i], sp.enc_t, sp.rank, sp.width, pick_block_n_cover(sp.rank))) != SCD_OK) return st;
    if ((st = make_b_map(&maps[2 * nseg + 5 * np + i], sp.enc_t, sp.rank, sp.width, pick_block_n_cover(sp.rank) / 2)) != SCD_OK) return st;
    if (sp.dec_t)
      if ((st = make_b_map(&maps[nseg + i], sp.dec_t, p->D, sp.rank, pick_block_n_div(p->D))) != SCD_OK) return st;
  }
  for (int j = 0; j < np; ++j) {
    const PatchPlan& pp = p->patches[j];
    if ((st = make_b_map(&maps[2 * nseg + 3 * j], pp.w1_t, pp.d_a, pp.r_h, pick_block_n_cover(pp.d_a))) != SCD_OK) return st;
    if ((st = make_b_map(&maps[2 * nseg + 3 * j + 1], pp.w2_t, m.d_model, pp.d_a, pick_block_n_cover(m.d_model))) != SCD_OK) return st;
    if ((st = make_b_map(&maps[2 * nseg + 3 * j + 2], pp.wkv, 2 * p->D, m.d_model, pick_block_n_div(p->D))) != SCD_OK) return st;
    if ((st = make_b_map(&maps[2 * nseg + 3 * np + 2 * j], pp.w2_t, m.d_model, pp.d_a, 128)) != SCD_OK) return st;
    if ((st = make_b_map(&maps[2 * nseg + 3 * np + 2 * j + 1], pp.wkv, 2 * p->D, m.d_model, 128)) != SCD_OK) return st;
  }
  void* d = nullptr;
  if (cudaMalloc(&d, maps.size() * sizeof(CUtensorMap) + 64) != cudaSuccess) return fail(SCD_E_NOMEM, "cudaMalloc(tensor maps)");
  p->allocs.push_back(d);
  // stream-ordered on the plan's stream (pageable source: staged before the call returns), like every other plan write
  if (cudaMemcpyAsync(d, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, s) != cudaSuccess)
    return fail(SCD_E_CUDA, "cudaMemcpyAsync(tensor maps)");
  p->tc_bmaps = d;
  void* sc = nullptr;
  if (cudaMalloc(&sc, KV_SCHED_SETS * 2 * sizeof(int32_t)) != cudaSuccess) return fail(SCD_E_NOMEM, "cudaMalloc(kv scheduler)");
  p->allocs.push_back(sc);
  if (cudaMemsetAsync(sc, 0, KV_SCHED_SETS * 2 * sizeof(int32_t), s) != cudaSuccess) return fail(SCD_E_CUDA, "cudaMemsetAsync(kv scheduler)");
  p->kv_sched = (int32_t*)sc;
  return SCD_OK;
}

// ---------------------------------------------------------------------------------
// launch helper
// ---------------------------------------------------------------------------------
// CTA-pair launch: clusters of 2, one cluster per TPC, grid = 2 x min(pair tiles, resident clusters)
template <int EPI>
static scd_status_t launch_tc_pair(const scd_plan_t* p, TcParams& P, size_t smem, int pair_tiles, cudaStream_t s) {
  if (EPI != EPI_U && EPI != EPI_KV && EPI != EPI_CODES) return fail(SCD_E_UNSUPPORTED, "internal: CTA pairs for this epilogue");
  constexpr int E = (EPI == EPI_U || EPI == EPI_KV || EPI == EPI_CODES) ? EPI : EPI_U;
  auto kernel = tc_gemm_kernel<E, A_PLAIN, true>;
  static std::atomic<size_t> configured[SCD_MAX_DEVICES];
  static std::atomic<int> clusters[SCD_MAX_DEVICES];
  if (configured[p->device].load(std::memory_order_relaxed) < smem) {
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return fail(SCD_E_CUDA, "cudaFuncSetAttribute(pair smem %zu): %s", smem, cudaGetErrorString(e));
    int n = max_active_clusters(kernel, 384, smem, 2);
    if (n <= 0) n = p->sm_count / 2;
    clusters[p->device].store(n, std::memory_order_relaxed);
    configured[p->device].store(smem, std::memory_order_relaxed);
  }
  const int grid = 2 * std::min(pair_tiles, std::min(clusters[p->device].load(std::memory_order_relaxed), p->sm_count / 2));
  prof_begin(s);
  launch_pdl(kernel, grid, 384, smem, s, 2, P);
  prof_end(s, P.prof_id);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(SCD_E_CUDA, "tc_gemm_kernel (CTA pairs) launch: %s", cudaGetErrorString(e));
  count_launch();
  return SCD_OK;
}

template <int EPI, int AMODE>
static scd_status_t launch_tc(const scd_plan_t* p, TcParams& P, cudaStream_t s) {
  P.m_tiles = (P.M + BLOCK_M - 1) / BLOCK_M;
  P.n_tiles = (P.N + P.block_n - 1) / P.block_n;
  P.num_kb = (P.K + BLOCK_K - 1) / BLOCK_K;
  const int total = P.n_segs * P.m_tiles * P.n_tiles;
  if (total <= 0) return SCD_OK;
  // compact paged-KV epilogue: long-K tiles of two 128-wide heads (PATCH GEMM-3)
  const bool compact = EPI == EPI_KV && P.num_kb >= 16 && P.block_n == 256 && P.head_dim == 128 && P.rope_style == SCD_ROPE_HALF &&
                       (P.N % 256) == 0;
  P.kv_compact = compact ? 1 : 0;
  P.sub_n = tc_sub_n(EPI, compact);
  P.stg_warp_bytes = tc_stg_warp_bytes(EPI, P.block_n, compact, (EPI == EPI_CODES && P.code_dtype == SCD_E4M3_ROWSCALE) ? 1 : 2);
  // CTA pairs (the caller asked and pointed the segments at the 128-row-box B maps): whole 256-column tiles only
  const bool pair = P.pair && AMODE == A_PLAIN &&
                    (((EPI == EPI_U || (EPI == EPI_KV && compact)) && P.block_n == 256 && (P.N % 256) == 0) ||
                     (EPI == EPI_CODES && (P.block_n % 32) == 0));
  if (P.pair && !pair) return fail(SCD_E_UNSUPPORTED, "internal: CTA-pair launch requested for a shape it does not take");
  const int b_rows = pair ? P.block_n / 2 : P.block_n;
  constexpr int NEPI = tc_epi_warps(EPI, AMODE, false);
  P.stages = tc_pick_stages(b_rows, P.num_kb, P.stg_warp_bytes, tc_vec_warp_bytes(EPI, compact), pair ? EPI_WARPS : NEPI);
  // PATCH GEMM-1 with short K: B tile resident, A tiles streamed (see the kernel); needs a few tiles per CTA to pay
  const bool bres = TC_G1_BRES && EPI == EPI_ACT && AMODE == A_PLAIN && !pair && P.num_kb <= 4 && P.a_kb_per_head == 0 &&
                    total >= 4 * p->sm_count && P.block_n == 256 && (P.N % 256) == 0 &&
                    tc_pick_stages_bres(b_rows, P.num_kb, P.stg_warp_bytes, tc_vec_warp_bytes(EPI, compact), NEPI) >= 2 * P.num_kb;
  if (bres) {
    P.b_res = 1;
    P.stages = tc_pick_stages_bres(b_rows, P.num_kb, P.stg_warp_bytes, tc_vec_warp_bytes(EPI, compact), NEPI);
  }
  // super-block so that its A rows take <= 32 MB of the 126 MB L2 (whole CTA waves: a multiple of the grid's share)
  P.a_prefetch = (EPI == EPI_CODES && !P.a_gather) ? TC_A_PREFETCH : 0;   // encode: A is the HBM stream
  const int walk_mt = pair ? (P.m_tiles + 1) / 2 : P.m_tiles;      // m-tiles of the walk (pair tiles of 256 rows)
  P.msb = walk_mt;
  if (P.n_tiles > 1) {
    const long long a_tile_bytes = (long long)BLOCK_M * P.K * 2 * (pair ? 2 : 1);
    int msb = (int)std::max<long long>(1, (32ll << 20) / a_tile_bytes);
    if (msb < walk_mt) P.msb = msb;
  }
  if (bres) P.msb = walk_mt;                                       // plain m-fastest order (A is K <= 256 wide: nothing to block)
  const size_t smem = bres ? tc_smem_bytes_bres(b_rows, P.num_kb, P.stages, P.stg_warp_bytes, tc_vec_warp_bytes(EPI, compact), NEPI)
                           : tc_smem_bytes(b_rows, P.stages, P.stg_warp_bytes, tc_vec_warp_bytes(EPI, compact), pair ? EPI_WARPS : NEPI);
  if (pair) return launch_tc_pair<EPI>(p, P, smem, P.n_segs * P.n_tiles * walk_mt, s);
  // the attribute belongs to (function, device): cached per instantiation and device ordinal
  static std::atomic<size_t> configured[SCD_MAX_DEVICES];
  if (configured[p->device].load(std::memory_order_relaxed) < smem) {
    cudaError_t e = cudaFuncSetAttribute(tc_gemm_kernel<EPI, AMODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return fail(SCD_E_CUDA, "cudaFuncSetAttribute(smem %zu): %s", smem, cudaGetErrorString(e));
    configured[p->device].store(smem, std::memory_order_relaxed);
  }
  const int grid = std::min(total, p->sm_count);
  prof_begin(s);
  launch_pdl(tc_gemm_kernel<EPI, AMODE>, grid, AMODE != A_PLAIN ? DEROPE_NTHREADS : (4 + NEPI) * 32, smem, s, 1, P);
  prof_end(s, P.prof_id);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(SCD_E_CUDA, "tc_gemm_kernel launch: %s", cudaGetErrorString(e));
  count_launch();
  return SCD_OK;
}

static void fill_common(const scd_plan_t* p, const scd_batch_t* b, bool pages, bool producer, TcParams& P, int n_blocks = 0) {
  memset(&P, 0, sizeof(P));
  P.b_maps = (const CUtensorMap*)p->tc_bmaps;
  P.batch.cu_seqlens = b->cu_seqlens;
  P.batch.page_table = pages ? b->page_table : nullptr;
  P.batch.pos_offset = b->pos_offset;
  P.batch.n_seqs = b->n_seqs;
  P.batch.total_tokens = b->total_tokens;
  P.batch.max_pages_per_seq = b->max_pages_per_seq;
  P.batch.block_size = p->model.block_size;
  P.batch.n_blocks = n_blocks;
  P.pool_slots = (long long)n_blocks * p->model.block_size;
  {
    // frequencies as Q0.32 fractions of a turn, from fp64 (exact modular angle arithmetic in the kernel)
    const double theta = producer ? p->model.rope_theta_producer : p->model.rope_theta_consumer;
    for (int j = 0; j < p->model.head_dim / 2 && j < 64; ++j) {
      double turns = pow(theta, -2.0 * j / p->model.head_dim) / 6.283185307179586476925286766559;
      turns -= floor(turns);
      P.rope_g[j] = (uint32_t)llround(turns * 4294967296.0);
    }
  }
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
  int n_launched = 0;
  const size_t nseg = p->segs.size();
  // Launch order K, H, V: the launches overlap at their seams (dep_wait_late) and the plain ones claim their tiles
  // dynamically, so the V launch -- many short tiles -- goes last and fills the hole the H launch leaves (config 2: 192
  // tiles of 64 k-blocks on 148 SMs, a second wave of 44)
  // (measured on config 2 with dynamic claiming: K, H, V 0.257 ms; H, K, V 0.263 ms; K, V, H 0.291 ms)
  static const int kPassBranch[3] = {SCD_BRANCH_K, SCD_BRANCH_H, SCD_BRANCH_V};
  for (int pass = 0; pass < 3; ++pass) {
  i = 0;
  while (i < nseg) {
    if (!layer_in_window(p->segs[i].layer) || p->segs[i].branch != kPassBranch[pass]) { ++i; continue; }
    // a launch = run of segments (inside the call's layer window) with the same branch, rank and width
    size_t j = i;
    // (a paged source needs two descriptors per segment: half as many segments per launch)
    const size_t max_run = (src->page_table && p->segs[i].branch != SCD_BRANCH_H) ? (size_t)TC_MAX_AMAPS / 2 : (size_t)TC_MAX_SEGS;
    while (j < nseg && j - i < max_run && p->segs[j].branch == p->segs[i].branch &&
           p->segs[j].rank == p->segs[i].rank && layer_in_window(p->segs[j].layer))
      ++j;
    const SegPlan& s0 = p->segs[i];
    static thread_local TcParams P;
    fill_common(p, batch, false, true, P);
    P.n_segs = (int)(j - i);
    P.N = s0.rank;
    P.K = s0.width;
    P.block_n = pick_block_n_cover(s0.rank);
    P.a_kb_per_head = (s0.branch != SCD_BRANCH_H && !dense_kv) ? m.head_dim / BLOCK_K : 0;
    const bool gather = src->page_table != nullptr && s0.branch != SCD_BRANCH_H;
    if (gather) {                       // rows of the K / V tiles come through the producer's page table
      P.a_gather = 1;
      P.batch.page_table = src->page_table;
      P.batch.max_pages_per_seq = src->max_pages_per_seq;
      P.batch.n_blocks = src->n_blocks;
    }
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
        if (gather) {
          st = make_gather_map(am, a, p->D, (uint64_t)src->n_blocks * m.block_size, (uint64_t)src->kv_token_stride * 2);
          if (st == SCD_OK)
            st = make_gather_map(&P.a_maps[TC_MAX_AMAPS / 2 + (q - i)], a, p->D, (uint64_t)src->n_blocks * m.block_size,
                                 (uint64_t)src->kv_token_stride * 2, 16);
        }
        else if (dense_kv)
          st = make_map(am, a, p->D, T, 1, (uint64_t)src->kv_token_stride * 2, (uint64_t)src->kv_token_stride * 2 * T,
                        BLOCK_M, 1);
        else
          st = make_map(am, a, m.head_dim, m.n_kv_heads, T, (uint64_t)src->kv_head_stride * 2,
                        (uint64_t)src->kv_token_stride * 2, 1, BLOCK_M);
      }
      if (st != SCD_OK) return st;
    }
    P.prof_id = (s0.branch == SCD_BRANCH_K && m.k_is_roped) ? SCD_PROF_ENCODE_K : SCD_PROF_ENCODE;
    P.dep_wait_late = (TC_ENC_OVERLAP && n_launched > 0) ? 1 : 0;      // the call's launches are independent of one another
    ++n_launched;
    if (s0.branch == SCD_BRANCH_K && m.k_is_roped) {
      if (m.rope_style != SCD_ROPE_HALF)
        return fail(SCD_E_UNSUPPORTED, "deRoPE-on-load implements the HALF pairing only on the bf16 path");
      st = launch_tc<EPI_CODES, A_DEROPE>(p, P, s);
    } else {
      // wide ranks (256-column tiles): CTA pairs, half of the W_enc^T tile per CTA (config 4: V 0.453 -> 0.420 ms, H 0.258 ->
      // 0.220 ms; at r = 128 the plain kernel with its L2 prefetch of the A stream is as fast: 0.098 vs 0.101 ms)
      if (TC_ENC_PAIRS && P.block_n == 256 && !gather && P.a_kb_per_head == 0 && T > BLOCK_M) {
        P.pair = 1;
        for (size_t q = i; q < j; ++q) P.segs[q - i].b_map = 2 * (int)nseg + 5 * (int)p->patches.size() + p->segs[q].seg_index;
      }
      if (TC_ENC_DYN && !P.pair && !gather)      // dynamic tile claiming: a plan-owned counter pair per launch in flight
        P.sched = p->kv_sched + 2 * (p->kv_sched_next.fetch_add(1) % KV_SCHED_SETS);
      st = launch_tc<EPI_CODES, A_PLAIN>(p, P, s);
    }
    if (st != SCD_OK) return st;
    i = j;
  }
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
  const bool e4 = m.code_dtype == SCD_E4M3_ROWSCALE;
  scd_status_t st;
  const int nseg_all = (int)p->segs.size();
  size_t i = 0;
  std::vector<int> reuse;
  for (int q = 0; q < nseg_all; ++q)
    if (p->segs[q].branch != SCD_BRANCH_H && layer_in_window(p->segs[q].layer)) reuse.push_back(q);
  while (i < reuse.size()) {
    size_t j = i;
    while (j < reuse.size() && j - i < (size_t)TC_MAX_SEGS && p->segs[reuse[j]].rank == p->segs[reuse[i]].rank) ++j;
    const SegPlan& s0 = p->segs[reuse[i]];
    static thread_local TcParams P;
    fill_common(p, batch, true, false, P, kv->n_blocks);
    P.n_segs = (int)(j - i);
    P.N = p->D;
    P.K = s0.rank;
    P.block_n = pick_block_n_div(p->D);
    P.split = P.N;
    P.pool_width = p->D;
    // segments of a run are consecutive in the code buffer with a uniform stride: one 3-D map
    const size_t seg_stride = align_up((size_t)T * s0.rank * (e4 ? 1 : 2), 128);
    const int key0 = s0.layer * 3 + s0.branch;
    bool uniform = true;
    for (size_t q = i; q < j; ++q) {
      const SegPlan& sp = p->segs[reuse[q]];
      if (off[sp.layer * 3 + sp.branch] != off[key0] + (q - i) * seg_stride) uniform = false;
    }
    if (uniform) {
      st = e4 ? make_code_map_u8(&P.a_maps[0], (const char*)codes + off[key0], s0.rank, T, j - i, seg_stride)
              : make_map(&P.a_maps[0], (const char*)codes + off[key0], s0.rank, T, j - i, (uint64_t)s0.rank * 2, seg_stride,
                         BLOCK_M, 1);
      if (st != SCD_OK) return st;
    }
    for (size_t q = i; q < j; ++q) {
      const SegPlan& sp = p->segs[reuse[q]];
      const int key = sp.layer * 3 + sp.branch;
      TcSeg& sg = P.segs[q - i];
      sg.col_vec = sp.mean_dst;
      sg.out0 = sp.branch == SCD_BRANCH_K ? kv->k_pool[sp.layer] : kv->v_pool[sp.layer];
      if (kv->pool_e4m3) sg.scale0 = sp.branch == SCD_BRANCH_K ? kv->k_scale[sp.layer] : kv->v_scale[sp.layer];
      sg.rope_cols = (sp.branch == SCD_BRANCH_K && m.rope_on_reuse_k) ? p->D : 0;
      sg.b_map = nseg_all + sp.seg_index;
      sg.a_scale = e4 ? (const float*)((const char*)codes + soff[key]) : nullptr;
      if (uniform) {
        sg.a_map = 0;
        sg.a_z = (int)(q - i);
      } else {
        sg.a_map = (int)(q - i);
        sg.a_z = 0;
        st = e4 ? make_code_map_u8(&P.a_maps[q - i], (const char*)codes + off[key], sp.rank, T, 1, seg_stride)
                : make_map(&P.a_maps[q - i], (const char*)codes + off[key], sp.rank, T, 1, (uint64_t)sp.rank * 2, seg_stride,
                           BLOCK_M, 1);
        if (st != SCD_OK) return st;
      }
    }
    P.prof_id = SCD_PROF_REUSE_DECODE;
    P.head_rank = m.reuse_per_head ? s0.rank / m.n_kv_heads : 0;
    P.a_is_codes = 1;
    P.pool_e4m3 = kv->pool_e4m3 ? 1 : 0;
    if (P.pool_e4m3 && !tc_kv_eligible(p, P)) return fail(SCD_E_UNSUPPORTED, "fp8 pools: D must be a multiple of 256");
    // the paged-KV kernel takes 256-column tiles of 128-wide heads (e4m3 codes: widened in shared memory by its own
    // warps); anything else runs on the generic kernel
    // a call with more than TC_MAX_SEGS (layer, branch) segments takes several launches over disjoint layers: like the
    // encode's, they overlap at their seams (dep_wait_late)
    P.dep_wait_late = (TC_ENC_OVERLAP && i > 0) ? 1 : 0;
    if (tc_kv_eligible(p, P)) st = launch_tc_kv(p, P, s);
    else st = e4 ? launch_tc<EPI_KV, A_CODES>(p, P, s) : launch_tc<EPI_KV, A_PLAIN>(p, P, s);
    if (st != SCD_OK) return st;
    i = j;
  }
  return SCD_OK;
}

// ---------------------------------------------------------------------------------
// scd_patch on tensor cores: GEMM-1 (aligner in) -> GEMM-2 (aligner out, row sum of squares) -> GEMM-3
// ([gamma.W_k | gamma.W_v], row scale, RoPE, paged write).  PATCH layers are independent of one another
// (Alg. 1), so each stage runs for a GROUP of layers as one multi-segment launch: three
// launches per group instead of three per layer, and GEMM-3's 512 tiles per layer (3.46 waves on 148 SMs)
// become 512 x group tiles.  A group = consecutive PATCH layers of equal (r_h, d_a), at most `group` of them
// (what the workspace holds).
// ---------------------------------------------------------------------------------
scd_status_t tc_patch(const scd_plan_t* p, const scd_batch_t* batch, const void* codes, const scd_paged_kv_t* kv,
                      void* ws_act, void* ws_u, float* ws_ss, int group, size_t act_stride, size_t u_stride, size_t ss_stride,
                      const size_t* off, const size_t* soff, cudaStream_t s) {
  const scd_model_desc_t& m = p->model;
  const int T = batch->total_tokens, d = m.d_model, D = p->D;
  const bool e4 = m.code_dtype == SCD_E4M3_ROWSCALE;
  const bool rms = m.patch_norm == SCD_NORM_RMS;
  const int nseg = (int)p->segs.size();
  scd_status_t st;
  if (group < 1) group = 1;
  if (group > TC_MAX_SEGS) group = TC_MAX_SEGS;
  size_t j0 = 0;
  int n_groups_done = 0;
  while (j0 < p->patches.size()) {
    if (!layer_in_window(p->patches[j0].layer)) { ++j0; continue; }
    size_t j1 = j0;
    while (j1 < p->patches.size() && j1 - j0 < (size_t)group && p->patches[j1].r_h == p->patches[j0].r_h &&
           p->patches[j1].d_a == p->patches[j0].d_a && layer_in_window(p->patches[j1].layer))
      ++j1;
    const PatchPlan& p0 = p->patches[j0];
    const int g = (int)(j1 - j0);
    static thread_local TcParams P;
    // GEMM-1: [T, r_h] x [r_h, d_a] per layer
    fill_common(p, batch, true, false, P);
    P.n_segs = g; P.N = p0.d_a; P.K = p0.r_h; P.block_n = pick_block_n_cover(p0.d_a);
    for (int q = 0; q < g; ++q) {
      const PatchPlan& pp = p->patches[j0 + q];
      const int key = pp.layer * 3 + SCD_BRANCH_H;
      st = e4 ? make_code_map_u8(&P.a_maps[q], (const char*)codes + off[key], pp.r_h, T, 1, align_up((size_t)T * pp.r_h, 128))
              : make_map(&P.a_maps[q], (const char*)codes + off[key], pp.r_h, T, 1, (uint64_t)pp.r_h * 2,
                         align_up((size_t)T * pp.r_h * 2, 128), BLOCK_M, 1);
      if (st != SCD_OK) return st;
      TcSeg& sg = P.segs[q];
      sg.a_map = q; sg.col_vec = pp.b1; sg.out0 = (char*)ws_act + q * act_stride; sg.b_map = 2 * nseg + 3 * (int)(j0 + q);
      sg.a_scale = e4 ? (const float*)((const char*)codes + soff[key]) : nullptr;
    }
    P.prof_id = SCD_PROF_PATCH_GEMM1;
    // a later group's GEMM-1 reads codes and overwrites activation slices whose reader (the previous group's GEMM-2) completed
    // before that group's GEMM-3 started: independent of its stream predecessor, the previous group's GEMM-3 (dep_wait_late)
    P.dep_wait_late = (TC_ENC_OVERLAP && n_groups_done > 0) ? 1 : 0;
    ++n_groups_done;
    if ((st = e4 ? launch_tc<EPI_ACT, A_CODES>(p, P, s) : launch_tc<EPI_ACT, A_PLAIN>(p, P, s)) != SCD_OK) return st;
    // GEMM-2: [T, d_a] x [d_a, d] per layer
    fill_common(p, batch, true, false, P);
    P.n_segs = g; P.N = d; P.K = p0.d_a; P.block_n = pick_block_n_cover(d);
    const int n_partials = 2 * ((d + P.block_n - 1) / P.block_n);   // two column groups per n-tile
    for (int q = 0; q < g; ++q) {
      const PatchPlan& pp = p->patches[j0 + q];
      if ((st = make_map(&P.a_maps[q], (char*)ws_act + q * act_stride, pp.d_a, T, 1, (uint64_t)pp.d_a * 2,
                         (uint64_t)pp.d_a * 2 * T, BLOCK_M, 1)) != SCD_OK) return st;
      TcSeg& sg = P.segs[q];
      sg.a_map = q; sg.col_vec = pp.b2; sg.out0 = (char*)ws_u + q * u_stride;
      sg.aux = rms ? (float*)((char*)ws_ss + q * ss_stride) : nullptr;
      sg.b_map = 2 * nseg + 3 * (int)(j0 + q) + 1;
    }
    P.prof_id = SCD_PROF_PATCH_GEMM2;
    if (TC_PAIRS && (d % 256) == 0 && P.block_n == 256 && T > BLOCK_M) {       // CTA pairs: B maps with 128-row boxes
      P.pair = 1;
      for (int q = 0; q < g; ++q) P.segs[q].b_map = 2 * nseg + 3 * (int)p->patches.size() + 2 * (int)(j0 + q);
    }
    if ((st = launch_tc<EPI_U, A_PLAIN>(p, P, s)) != SCD_OK) return st;
    // GEMM-3: [T, d] x [d, 2D] per layer
    fill_common(p, batch, true, false, P, kv->n_blocks);
    P.n_segs = g; P.N = 2 * D; P.K = d; P.block_n = pick_block_n_div(D);
    P.split = D; P.pool_width = D; P.n_partials = n_partials; P.rms_dim = d; P.rms_eps = m.rms_eps;
    for (int q = 0; q < g; ++q) {
      const PatchPlan& pp = p->patches[j0 + q];
      if ((st = make_map(&P.a_maps[q], (char*)ws_u + q * u_stride, d, T, 1, (uint64_t)d * 2, (uint64_t)d * 2 * T, BLOCK_M, 1)) != SCD_OK)
        return st;
      TcSeg& sg = P.segs[q];
      sg.a_map = q; sg.col_vec = pp.bkv; sg.out0 = kv->k_pool[pp.layer]; sg.out1 = kv->v_pool[pp.layer];
      if (kv->pool_e4m3) { sg.scale0 = kv->k_scale[pp.layer]; sg.scale1 = kv->v_scale[pp.layer]; }
      sg.rowscale_in = rms ? (const float*)((const char*)ws_ss + q * ss_stride) : nullptr;
      sg.rope_cols = D;
      sg.b_map = 2 * nseg + 3 * (int)(j0 + q) + 2;
    }
    P.prof_id = SCD_PROF_PATCH_GEMM3;
    // long K (d_model >= 1024): the generic kernel with the compact epilogue runs four pipeline stages where the
    // paged-KV kernel has room for three; short K: the paged-KV kernel's faster epilogue wins
    P.pool_e4m3 = kv->pool_e4m3 ? 1 : 0;
    if (P.pool_e4m3 && !tc_kv_eligible(p, P)) return fail(SCD_E_UNSUPPORTED, "fp8 pools: D must be a multiple of 256");
    const bool long_k = G3_GENERIC && d >= 16 * BLOCK_K && !P.pool_e4m3;   // fp8 pools: only the paged-KV kernel quantises
    if (TC_PAIRS && long_k && P.block_n == 256 && (P.N % 256) == 0 && m.head_dim == 128 && m.rope_style == SCD_ROPE_HALF && T > BLOCK_M) {
      P.pair = 1;
      for (int q = 0; q < g; ++q) P.segs[q].b_map = 2 * nseg + 3 * (int)p->patches.size() + 2 * (int)(j0 + q) + 1;
    }
    if ((st = (!long_k && tc_kv_eligible(p, P)) ? launch_tc_kv(p, P, s)
                                                                                       : launch_tc<EPI_KV, A_PLAIN>(p, P, s)) != SCD_OK)
      return st;
    j0 = j1;
  }
  return SCD_OK;
}

}  // namespace scd
