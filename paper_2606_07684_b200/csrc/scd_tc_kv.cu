// Paged-KV specialisation of the tcgen05 GEMM: REUSE decode (Eq. 9) and short-K PATCH
// GEMM-3 (Eq. 12a/b) for head_dim 128, HALF RoPE, 256-column (two-head) tiles.  (Long-K GEMM-3
// runs on scd_tc.cu's kernel with its compact epilogue, which leaves room for a fourth pipeline stage.)
//
// Same TMA -> tcgen05 -> TMEM main loop as scd_tc.cu; what differs is the tile order and the epilogue,
// which is where this kernel's time goes (it writes 8x what it reads):
//
//   * tiles are walked m-slowest (m-tile, segment, n-tile) and each CTA owns one contiguous range, so
//     a CTA sees at most a handful of m-tiles: the per-row quantities (position, slot, RMS scale) and
//     the row's (cos, sin) are computed when the m-tile changes and then live in registers;
//   * 16 epilogue warps: warp (q, g) owns TMEM lane quadrant q (32 token rows, one per lane) and,
//     for K tiles, RoPE frequencies [16g, 16g+16) of both heads -- every (cos, sin) is used for two
//     heads and for every layer of the m-tile; for V tiles, columns [64g, 64g+64);
//   * the four warps of a quadrant stage bf16 results in one swizzled [32 x 512 B] buffer, meet at a
//     named barrier, and each copies 8 complete 512-B row segments to the rows' slots of the paged
//     pool with fully coalesced 16-B stores.
#include <algorithm>
#include <cstring>

#include "scd_tc_common.cuh"

#ifndef KV_ARES
#define KV_ARES 1
#endif
#ifndef KV_ARES_BF16
#define KV_ARES_BF16 1
#endif
#ifndef KV_STATIC_PCT
#define KV_STATIC_PCT 60
#endif

namespace scd {

namespace {

constexpr int KV_BLOCK_N = 256;
constexpr int KV_EPI_WARPS = 16;
constexpr int KV_B_STAGE_BYTES = KV_BLOCK_N * BLOCK_K * 2;   // 32 KB
constexpr int KV_ROW_PITCH = 512;
constexpr int KV_STG_BYTES = 4 * 32 * KV_ROW_PITCH;          // 4 quadrants x [32 rows x 512 B] = 64 KB
constexpr int KV_VEC_BYTES = KV_EPI_WARPS * 64 * 4;          // per-warp slice of the tile's mean / bias: 64 floats
constexpr int KV_SLOT_BYTES = KV_EPI_WARPS * 32 * 4;         // per-warp copy of its quadrant's 32 slot numbers (-1 = no row)

struct __align__(8) KvBarriers {
  uint64_t full[MAX_STAGES], empty[MAX_STAGES], ready[MAX_STAGES];
  uint64_t tmem_full[2], tmem_empty[2];
  uint64_t sched_full[4], sched_empty[4];                    // chunk ring (KV_SCHED_SLOTS)
  int32_t sched_begin[4], sched_end[4];                      // tile range of the entry; begin < 0 = no more work
  uint64_t a_full[4], a_ready[4], a_empty[4];                // ARES: the resident code tile's k-block slots
  uint32_t tmem_base;
};
constexpr int KV_SCHED_SLOTS = 4;

size_t kv_smem_bytes(int stages) {
  return 1024 + (size_t)stages * (A_STAGE_BYTES + KV_B_STAGE_BYTES) + KV_STG_BYTES + KV_VEC_BYTES + KV_SLOT_BYTES + sizeof(KvBarriers);
}
// ARES (code tile resident across the n-tiles of its (m-tile, segment)): num_kb slots of 16 KB + a ring of basis stages
// Its shared memory is laid out tightly so that K = 256 gets a THIRD basis stage (two left main loop and epilogue adding up
// instead of overlapping: 0.88 + 1.06 -> 1.68 ms on config 4): the small regions come first -- barriers (<= 512 B), ONE slot
// table per lane quadrant (4 x 128 B) and the mean slices per column group, double-buffered by accumulator (4 x 2 x 256 B),
// 3 KB in all instead of 6.4 KB of per-warp copies -- then the 1024-byte-aligned tiles.  With the dynamic shared memory
// starting on a 1024-byte boundary (if it ever does not, the kernel runs with one stage less) that is exactly 227 KB at K = 256,
// three stages.
constexpr int KVA_SMALL_BYTES = 3072, KVA_SLOT_OFF = 512, KVA_VEC_OFF = 1024;
static_assert(sizeof(KvBarriers) <= KVA_SLOT_OFF, "barriers outgrew their 512 bytes");
size_t kva_smem_bytes(int b_stages, int num_kb) {
  const size_t need = KVA_SMALL_BYTES + (size_t)num_kb * A_STAGE_BYTES + (size_t)b_stages * KV_B_STAGE_BYTES + KV_STG_BYTES;
  // wherever it costs no stage (every rank but 256), 1 KB of slack makes the carve-up independent of the window's alignment
  return need + 1024 <= 232448 ? need + 1024 : need;
}
int kva_pick_stages(int num_kb) {
  const size_t budget = 232448 - KVA_SMALL_BYTES - KV_STG_BYTES - (size_t)num_kb * A_STAGE_BYTES;
  int st = (int)(budget / KV_B_STAGE_BYTES);
  return st > MAX_STAGES ? MAX_STAGES : st;
}
int kv_pick_stages(int num_kb) {
  const size_t budget = 232448 - 1024 - KV_STG_BYTES - KV_VEC_BYTES - KV_SLOT_BYTES - sizeof(KvBarriers);
  int st = (int)(budget / (A_STAGE_BYTES + KV_B_STAGE_BYTES));
  if (st > MAX_STAGES) st = MAX_STAGES;
  if (st > 2 * num_kb) st = 2 * num_kb;
  return st < 2 ? 2 : st;
}

// quadrant staging buffer: 32 rows x 512 B, 16-byte chunks XOR-swizzled with the row's low 3 bits:
// row-per-lane writes and row-per-warp reads are both conflict free
__device__ __forceinline__ uint32_t qstg_addr(uint32_t stg, int row, int chunk) {
  return stg + row * 512 + (((chunk & ~7) | ((chunk ^ row) & 7)) << 4);
}

struct TileCoord {
  int m_tile, seg, n_tile;
};
// Tile order.  SEG_SLOWEST = false (REUSE decode): (m-tile, segment, n-tile) -- a CTA's contiguous share stays on a
// handful of m-tiles, so per-row state is computed once for all layers.  SEG_SLOWEST = true (PATCH GEMM-3 over a group
// of layers): (segment, m-tile, n-tile) -- one layer's 33 MB weight slab at a time stays L2-resident.
template <bool SEG_SLOWEST>
__device__ __forceinline__ void tile_next(const TcParams& P, TileCoord& c) {
  if (++c.n_tile == P.n_tiles) {
    c.n_tile = 0;
    if (SEG_SLOWEST) {
      if (++c.m_tile == P.m_tiles) { c.m_tile = 0; ++c.seg; }
    } else {
      if (++c.seg == P.n_segs) { c.seg = 0; ++c.m_tile; }
    }
  }
}
// k-blocks a tile needs.  Per-head REUSE (P.head_rank = r > 0): the operands are block-diagonal, a 256-column tile is
// heads 2 n_tile and 2 n_tile + 1, whose codes are columns [2 n_tile r, (2 n_tile + 2) r) of the code row.
__device__ __forceinline__ void tile_kb_range(const TcParams& P, int n_tile, int& kb0, int& kb1) {
  kb0 = 0;
  kb1 = P.num_kb;
  if (P.head_rank > 0) {
    kb0 = (2 * n_tile * P.head_rank) / BLOCK_K;
    kb1 = min(P.num_kb, ((2 * n_tile + 2) * P.head_rank + BLOCK_K - 1) / BLOCK_K);
  }
}
template <bool SEG_SLOWEST>
__device__ __forceinline__ TileCoord tile_coord(const TcParams& P, int tile) {
  TileCoord c;
  if (SEG_SLOWEST) {
    const int per_seg = P.m_tiles * P.n_tiles;
    c.seg = tile / per_seg;
    const int rem = tile - c.seg * per_seg;
    c.m_tile = rem / P.n_tiles;
    c.n_tile = rem - c.m_tile * P.n_tiles;
  } else {
    const int per_m = P.n_segs * P.n_tiles;
    c.m_tile = tile / per_m;
    const int rem = tile - c.m_tile * per_m;
    c.seg = rem / P.n_tiles;
    c.n_tile = rem - c.seg * P.n_tiles;
  }
  return c;
}

}  // namespace

// ---------------------------------------------------------------------------------
// the kernel: warp 0 = TMEM allocator + TMA producer, warp 1 = MMA issuer, warps 2-3 idle, warps 4..19 =
// epilogue.  Registers live per SM sub-partition (16 K each, 5 warps): warpgroup 0 shrinks to 32 registers so
// that the four epilogue warps of each sub-partition can hold 112 (setmaxnreg).
// ---------------------------------------------------------------------------------
constexpr int KV_FIRST_EPI_WARP = 4;
constexpr int KV_NTHREADS = (KV_FIRST_EPI_WARP + KV_EPI_WARPS) * 32;   // 640
#ifndef KV_XF_WARPS_N
#define KV_XF_WARPS_N 8
#endif
constexpr int KV_XF_WARPS = KV_XF_WARPS_N;                              // AE4: code-widening warps (two per SM sub-partition)
constexpr int KV_XF_ITEMS = 512 / (KV_XF_WARPS * 32);                   // 16-code items per thread and k-block
constexpr int KV_NTHREADS_E4 = KV_NTHREADS + KV_XF_WARPS * 32;          // 896

// DYN: dynamic tile scheduling (hybrid static share + claimed chunks) -- used where tiles are long (PATCH GEMM-3,
// K = d_model) and SMs drift apart; the REUSE decode keeps the static split, whose epilogue has no registers
// to spare for the scheduler state.
// SCALED: rows carry a scale (e4m3 code scales and / or the RMS scale of PATCH GEMM-3); REUSE decode of bf16 codes
// compiles it out (no per-tile scale fetch, mean added with one packed add).
// AE4: the A operand is a segment of e4m3 codes (config 4).  tcgen05 has no bf16 x fp8 MMA and the basis must stay bf16,
// so the raw tile [128 rows x 64 B] lands in the upper half of the A stage and four extra warps (24 in all; registers
// re-dealt 24 / 104 / 40) widen it in place to the swizzled bf16 tile before the MMA may read it -- exactly (all 254
// finite codes, test_e4m3_operand_expansion_is_exact_for_every_code); the row scale is applied in the epilogue.
// P8: the pools are e4m3 bytes with one fp32 scale per (slot, head) (fp8 pools, scd.h): the copy-out, which holds a
// complete bf16 row segment of two heads per warp pass, takes the head's amax over its 16 lanes, and stores 8 bytes per
// lane plus the scale.
// ARES (e4m3 codes, K <= 256): the code tile of an (m-tile, segment) serves all of its n-tiles, which are consecutive in
// the walk; widening it once per n-tile is what bounds the e4m3 decode (profiles/r02_decode_history.md).  Here its k-blocks
// get slots of their own: loaded and widened ONCE when the CTA enters the (m-tile, segment), released by the MMAs of the last
// n-tile; only the basis tiles go through the ring.
template <bool DYN, bool SCALED, bool AE4, bool P8, bool ARES = false>
__global__ void __launch_bounds__(AE4 ? KV_NTHREADS_E4 : KV_NTHREADS, 1) tc_kv_kernel(const __grid_constant__ TcParams P) {
  static_assert(!AE4 || (SCALED && !DYN), "e4m3 codes carry row scales; static split");
  static_assert(!ARES || !DYN, "resident code tiles: static split (REUSE decode)");
  static_assert(!P8 || SCALED, "fp8 pools are built on the scaled variants only");
  extern __shared__ uint8_t smem_raw[];
  // ARES: small regions first, then the aligned tiles (see kva_smem_bytes)
  uint8_t* smem = ARES ? (uint8_t*)(((uintptr_t)smem_raw + KVA_SMALL_BYTES + 1023) & ~(uintptr_t)1023)
                       : (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  int stages_fit = P.stages;
  if (ARES) {
    // The host sizes the window for tiles that start on a 1024-byte boundary right after the small regions.  Should the
    // window itself not start on one, the ring gives up a stage instead of running past the end (every role takes the same
    // decision from the same addresses).
    uint32_t dyn;
    asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn));
    while (stages_fit > 1 && smem + (size_t)P.num_kb * A_STAGE_BYTES + (size_t)stages_fit * KV_B_STAGE_BYTES + KV_STG_BYTES > smem_raw + dyn)
      --stages_fit;
  }
  const int STAGES = stages_fit;
  uint8_t* smem_a = smem;
  uint8_t* smem_b = smem + (ARES ? P.num_kb : STAGES) * A_STAGE_BYTES;      // ARES: STAGES counts basis stages only
  uint8_t* smem_stg = smem_b + STAGES * KV_B_STAGE_BYTES;
  uint8_t* smem_vec = ARES ? smem_raw + KVA_VEC_OFF : smem_stg + KV_STG_BYTES;
  uint8_t* smem_slot = ARES ? smem_raw + KVA_SLOT_OFF : smem_vec + KV_VEC_BYTES;
  KvBarriers* bars = ARES ? (KvBarriers*)smem_raw : (KvBarriers*)(smem_slot + KV_SLOT_BYTES);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int total_tiles = P.m_tiles * P.n_segs * P.n_tiles;
  // static mode: one contiguous share per CTA
  const int s_begin = (int)((long long)total_tiles * blockIdx.x / gridDim.x);
  const int s_end = (int)((long long)total_tiles * (blockIdx.x + 1) / gridDim.x);

  if (warp == 1 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) {
      ptx::mbar_init(&bars->full[s], 1);
      ptx::mbar_init(&bars->empty[s], 1);
      ptx::mbar_init(&bars->ready[s], KV_XF_WARPS * 32);
    }
    for (int a = 0; a < 2; ++a) {
      ptx::mbar_init(&bars->tmem_full[a], 1);
      ptx::mbar_init(&bars->tmem_empty[a], 4);          // one arrival per lane quadrant
    }
    for (int a = 0; a < 4; ++a) {
      ptx::mbar_init(&bars->a_full[a], 1);
      ptx::mbar_init(&bars->a_ready[a], KV_XF_WARPS * 32);
      ptx::mbar_init(&bars->a_empty[a], 1);
    }
    for (int a = 0; a < KV_SCHED_SLOTS; ++a) {
      ptx::mbar_init(&bars->sched_full[a], 1);
      ptx::mbar_init(&bars->sched_empty[a], 1 + KV_EPI_WARPS);   // MMA thread + one lane per epilogue warp
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
  // the previous kernel of the stream has completed and flushed (P.dep_wait_late: a later launch of one scd_reuse_decode
  // call, independent of its predecessor -- it waits at its END instead, see tc_gemm_kernel)
  if (!P.dep_wait_late) ptx::grid_dep_wait();
  ptx::grid_dep_launch_dependents();    // the next one may start its prologue as SMs free up

  if (warp < KV_FIRST_EPI_WARP) {
    // 128 x 32 + 512 x 112 = 640 x 96 (AE4: 128 x 24 + 512 x 104 + 256 x 32 = 64512 <= 896 x 72): the pool the launch allocated
    if (AE4) ptx::setmaxnreg_dec<24>();
    else ptx::setmaxnreg_dec<32>();
  if (warp == 0) {
    // ============================== TMA producer ==============================
    if (ARES) {
      if (lane == 0) {
        int stage = 0;
        uint32_t phase = 0, groups = 0;                       // groups = (m-tile, segment) code tiles started so far
        TileCoord tc = tile_coord<false>(P, s_begin);
        for (int tile = s_begin; tile < s_end; ++tile, tile_next<false>(P, tc)) {
          const TcSeg& sg = P.segs[tc.seg];
          const bool grp_first = tile == s_begin || tc.n_tile == 0;
          if (grp_first && tile + (P.n_tiles - tc.n_tile) < s_end) {
            // the NEXT group's code tile comes from HBM and its load sits on the critical path at the group boundary (the
            // slots free only then): pull it into L2 now, a whole group ahead
            int nseg = tc.seg + 1, nm = tc.m_tile;
            if (nseg == P.n_segs) { nseg = 0; ++nm; }
            const TcSeg& ng = P.segs[nseg];
            for (int kb = 0; kb < P.num_kb; ++kb) ptx::tma_prefetch_l2_3d(&P.a_maps[ng.a_map], kb * BLOCK_K, nm * BLOCK_M, ng.a_z);
          }
          for (int kb = 0; kb < P.num_kb; ++kb) {
            if (grp_first) {                                   // the code tile's k-block, once its slot has been released
              if (groups > 0) ptx::mbar_wait_suspend(&bars->a_empty[kb], (groups - 1) & 1);
              // e4m3 codes: the raw tile lands in the upper half of its slot and is widened in place; bf16 codes: the slot itself
              ptx::mbar_expect_tx(&bars->a_full[kb], AE4 ? A_STAGE_BYTES / 2 : A_STAGE_BYTES);
              ptx::tma_load_3d(smem_a + kb * A_STAGE_BYTES + (AE4 ? A_STAGE_BYTES / 2 : 0), &P.a_maps[sg.a_map], &bars->a_full[kb], kb * BLOCK_K,
                               tc.m_tile * BLOCK_M, sg.a_z);
            }
            ptx::mbar_wait_suspend(&bars->empty[stage], phase ^ 1);
            ptx::mbar_expect_tx(&bars->full[stage], KV_B_STAGE_BYTES);
            ptx::tma_load_2d(smem_b + stage * KV_B_STAGE_BYTES, P.b_maps + sg.b_map, &bars->full[stage], kb * BLOCK_K, tc.n_tile * KV_BLOCK_N);
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
          if (grp_first) ++groups;
        }
      }
    } else
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      int slot = 0;
      uint32_t sphase = 0;
      // dynamic mode: every CTA owns a static contiguous share first (per-row state is computed once per m-tile), then
      // claims small chunks of the remainder; the next claim is always in flight under the current loads
      int next_chunk = DYN ? atomicAdd(P.sched, 1) : 0;
      for (int round = 0;; ++round) {
        int t_begin, t_end;
        if (!DYN) {
          if (round) break;
          t_begin = s_begin;
          t_end = s_end;
        } else {
        if (round == 0) {
          t_begin = (int)blockIdx.x * P.static_tiles;
          t_end = t_begin + P.static_tiles;
        } else {
          const int chunk = next_chunk;
          if (chunk < P.n_chunks) next_chunk = atomicAdd(P.sched, 1);
          t_begin = chunk < P.n_chunks ? P.dyn_begin + chunk * P.chunk_tiles : -1;
          t_end = t_begin + P.chunk_tiles;
        }
        ptx::mbar_wait_suspend(&bars->sched_empty[slot], sphase ^ 1);
        *(volatile int*)&bars->sched_begin[slot] = t_begin;
        *(volatile int*)&bars->sched_end[slot] = t_end;
        ptx::mbar_arrive(&bars->sched_full[slot]);
        if (++slot == KV_SCHED_SLOTS) { slot = 0; sphase ^= 1; }
        if (t_begin < 0) break;
        }
      TileCoord tc = tile_coord<DYN>(P, t_begin);
      for (int tile = t_begin; tile < t_end; ++tile, tile_next<DYN>(P, tc)) {
        const TcSeg& sg = P.segs[tc.seg];
        const CUtensorMap* am = &P.a_maps[sg.a_map];
        const CUtensorMap* bm = P.b_maps + sg.b_map;
        int kb0, kb1;
        tile_kb_range(P, tc.n_tile, kb0, kb1);
        for (int kb = kb0; kb < kb1; ++kb) {
          ptx::mbar_wait_suspend(&bars->empty[stage], phase ^ 1);
          ptx::mbar_expect_tx(&bars->full[stage], (AE4 ? A_STAGE_BYTES / 2 : A_STAGE_BYTES) + KV_B_STAGE_BYTES);
          ptx::tma_load_3d(smem_a + stage * A_STAGE_BYTES + (AE4 ? A_STAGE_BYTES / 2 : 0), am, &bars->full[stage], kb * BLOCK_K,
                           tc.m_tile * BLOCK_M, sg.a_z);
          ptx::tma_load_2d(smem_b + stage * KV_B_STAGE_BYTES, bm, &bars->full[stage], kb * BLOCK_K,
                           tc.n_tile * KV_BLOCK_N);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
      }
      if (DYN) {
        // the last CTA to stop claiming work re-arms the counters for the next launch
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
    if (ARES) {
      if (lane == 0) {
        const uint32_t idesc = ptx::umma_idesc_bf16(BLOCK_M, KV_BLOCK_N);
        int stage = 0, it = 0;
        uint32_t phase = 0, groups = 0;                       // groups completed
        int n_tile = s_begin % P.n_tiles;
        for (int tile = s_begin; tile < s_end; ++tile, ++it) {
          const bool grp_first = tile == s_begin || n_tile == 0;
          const bool grp_last = tile == s_end - 1 || n_tile == P.n_tiles - 1;
          if (++n_tile == P.n_tiles) n_tile = 0;
          const int acc = it & 1;
          ptx::mbar_wait_suspend(&bars->tmem_empty[acc], ((it >> 1) & 1) ^ 1);
          ptx::tc_fence_after();
          const uint32_t d_tmem = tmem_base + (uint32_t)(acc * KV_BLOCK_N);
          for (int kb = 0; kb < P.num_kb; ++kb) {
            if (grp_first) ptx::mbar_wait_suspend(AE4 ? &bars->a_ready[kb] : &bars->a_full[kb], groups & 1);   // landed (and widened), once per group
            ptx::mbar_wait_suspend(&bars->full[stage], phase);
            ptx::tc_fence_after();
            const uint64_t da = ptx::umma_desc_sw128(ptx::smem_u32(smem_a + kb * A_STAGE_BYTES));
            const uint64_t db = ptx::umma_desc_sw128(ptx::smem_u32(smem_b + stage * KV_B_STAGE_BYTES));
#pragma unroll
            for (int k = 0; k < BLOCK_K / 16; ++k)
              ptx::mma_bf16(d_tmem, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, (kb | k) != 0);
            ptx::mma_commit(&bars->empty[stage]);
            if (grp_last) ptx::mma_commit(&bars->a_empty[kb]);                           // the slot may take the next code tile
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
          ptx::mma_commit(&bars->tmem_full[acc]);
          if (grp_last) ++groups;
        }
      }
    } else
    if (lane == 0) {
      const uint32_t idesc = ptx::umma_idesc_bf16(BLOCK_M, KV_BLOCK_N);
      int stage = 0;
      uint32_t phase = 0;
      int it = 0;
      int slot = 0;
      uint32_t sphase = 0;
      for (int round = 0;; ++round) {
        int t_begin = s_begin, t_end = s_end;
        if (!DYN) {
          if (round) break;
        } else {
          ptx::mbar_wait_suspend(&bars->sched_full[slot], sphase);
          t_begin = *(volatile int*)&bars->sched_begin[slot];
          t_end = *(volatile int*)&bars->sched_end[slot];
          ptx::mbar_arrive(&bars->sched_empty[slot]);
          if (++slot == KV_SCHED_SLOTS) { slot = 0; sphase ^= 1; }
          if (t_begin < 0) break;
        }
      int n_tile = t_begin % P.n_tiles;                    // the only tile coordinate the MMA loop needs
      for (int tile = t_begin; tile < t_end; ++tile, ++it) {
        const int acc = it & 1;
        const uint32_t acc_phase = (it >> 1) & 1;
        ptx::mbar_wait_suspend(&bars->tmem_empty[acc], acc_phase ^ 1);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(acc * KV_BLOCK_N);
        int kb0, kb1;
        tile_kb_range(P, n_tile, kb0, kb1);
        if (++n_tile == P.n_tiles) n_tile = 0;
        for (int kb = kb0; kb < kb1; ++kb) {
          ptx::mbar_wait_suspend(AE4 ? &bars->ready[stage] : &bars->full[stage], phase);   // ready: landed and widened
          ptx::tc_fence_after();
          const uint64_t da = ptx::umma_desc_sw128(ptx::smem_u32(smem_a + stage * A_STAGE_BYTES));
          const uint64_t db = ptx::umma_desc_sw128(ptx::smem_u32(smem_b + stage * KV_B_STAGE_BYTES));
#pragma unroll
          for (int k = 0; k < BLOCK_K / 16; ++k)
            ptx::mma_bf16(d_tmem, da + (uint64_t)(k * 2), db + (uint64_t)(k * 2), idesc, (kb > kb0) || k != 0);
          ptx::mma_commit(&bars->empty[stage]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        ptx::mma_commit(&bars->tmem_full[acc]);
      }
      }
    }
  }
  } else if (AE4 && warp >= KV_FIRST_EPI_WARP + KV_EPI_WARPS) {
    // ============================== A transform: e4m3 -> bf16 in shared memory ==============================
    // 512 items of 16 codes per k-block (row = item / 4, quarter = item % 4), KV_XF_ITEMS per thread, read conflict-free from
    // the raw tile in bytes [8192, 16384) of the stage; all widening threads meet (the widened rows overwrite the raw
    // bytes); then each item becomes chunks 2 quarter, 2 quarter + 1 of its row in the 128-byte-swizzled K-major layout.
    if (KV_XF_WARPS == 4) ptx::setmaxnreg_dec<40>();
    else ptx::setmaxnreg_dec<32>();
    const int xt = threadIdx.x - (KV_FIRST_EPI_WARP + KV_EPI_WARPS) * 32;
    const uint32_t a_base = ptx::smem_u32(smem_a);
    int stage = 0;
    uint32_t phase = 0;
    int n_tile = s_begin % P.n_tiles;
    uint32_t groups = 0;
    for (int tile = s_begin; tile < s_end; ++tile) {
      int kb0, kb1;
      tile_kb_range(P, n_tile, kb0, kb1);
      const bool grp_first = tile == s_begin || n_tile == 0;
      if (++n_tile == P.n_tiles) n_tile = 0;
      if (ARES && !grp_first) continue;                       // the code tile of this (m-tile, segment) is already widened
      for (int kb = kb0; kb < kb1; ++kb) {
        if (ARES) { stage = kb; phase = groups & 1; }
        ptx::mbar_wait_suspend(ARES ? &bars->a_full[kb] : &bars->full[stage], phase);
        const uint32_t sb = a_base + (uint32_t)stage * A_STAGE_BYTES;
        uint4 raw[KV_XF_ITEMS];
#pragma unroll
        for (int j = 0; j < KV_XF_ITEMS; ++j) raw[j] = ptx::lds128(sb + A_STAGE_BYTES / 2 + (uint32_t)(xt + KV_XF_WARPS * 32 * j) * 16);
        ptx::named_bar_sync(5, KV_XF_WARPS * 32);
#pragma unroll
        for (int j = 0; j < KV_XF_ITEMS; ++j) {
          const int item = xt + KV_XF_WARPS * 32 * j, row = item >> 2, qt = item & 3;
          const uint32_t row_off = (uint32_t)(row >> 3) * 1024 + (uint32_t)(row & 7) * 128;
          const uint32_t w[4] = {raw[j].x, raw[j].y, raw[j].z, raw[j].w};
          uint32_t o[8];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            o[2 * i] = e4m3x2_to_bf16x2(__byte_perm(w[i], 0u, 0x1404));       // bytes 0, 1 -> high bytes of two halves
            o[2 * i + 1] = e4m3x2_to_bf16x2(__byte_perm(w[i], 0u, 0x3424));   // bytes 2, 3
          }
          ptx::sts128(sb + row_off + (uint32_t)(((2 * qt) ^ (row & 7)) << 4), make_uint4(o[0], o[1], o[2], o[3]));
          ptx::sts128(sb + row_off + (uint32_t)(((2 * qt + 1) ^ (row & 7)) << 4), make_uint4(o[4], o[5], o[6], o[7]));
        }
        ptx::fence_proxy_async_smem();
        if (ARES) {
          ptx::mbar_arrive(&bars->a_ready[kb]);
        } else {
          ptx::mbar_arrive(&bars->ready[stage]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
      if (ARES) ++groups;
    }
  } else {
    // ============================== epilogue ==============================
    if (AE4) ptx::setmaxnreg_inc<104>();
    else ptx::setmaxnreg_inc<112>();
    const int q = warp & 3;                                   // TMEM lane quadrant this warp may read
    const int g = (warp - KV_FIRST_EPI_WARP) >> 2;            // frequency / column group 0..3
    const uint32_t stg = ptx::smem_u32(smem_stg) + (uint32_t)q * (32 * KV_ROW_PITCH);
    // ARES: one slice per column group g (the four quadrants' warps write identical bytes), two buffers picked by the tile's
    // accumulator; else one private slice per warp
    const uint32_t wvec = ARES ? ptx::smem_u32(smem_vec) + (uint32_t)g * 512 : ptx::smem_u32(smem_vec) + (uint32_t)(warp - KV_FIRST_EPI_WARP) * 256;
    // the quadrant's 32 slot numbers, one private copy per warp (no cross-warp ordering needed): the copy-out reads the
    // slot of the row it stores with one broadcast LDS instead of shuffling a 64-bit address out of the owning lane
    // (ARES: one table per quadrant, written by its four warps -- identical values -- between the tile's two quadrant barriers)
    const uint32_t wslot = ARES ? ptx::smem_u32(smem_slot) + (uint32_t)q * 128 : ptx::smem_u32(smem_slot) + (uint32_t)(warp - KV_FIRST_EPI_WARP) * 128;
    int slot_reg = -1;
    bool slot_dirty = false;
    const uint32_t bar_id = 1 + q;
    const uint32_t row_stride = (uint32_t)P.pool_width * (P8 ? 1u : 2u);  // bytes per slot
    // this lane's float4 of the warp's mean / bias slice: tile column for K tiles (runs a | b of both heads) / V tiles
    const int vcol_k = ((lane >> 3) & 1) * 128 + ((lane >> 2) & 1) * 64 + 16 * g + (lane & 3) * 4;
    const int vcol_v = 64 * g + lane * 4;

    // per-row state, recomputed when the m-tile changes (DYN: or the segment -- the RMS scale belongs to a layer)
    int cur_m = -1, cur_seg = -1;
    float rs_row = 1.0f;
    unsigned long long c2[8], s2[8];                          // (cos, sin) of frequencies 16g + {2i, 2i+1}, packed pairs
#pragma unroll
    for (int i = 0; i < 8; ++i) c2[i] = s2[i] = 0ull;

    // per-tile prefetch: this lane's float4 of the warp's mean / bias slice, e4m3 row scale
    struct Pre {
      float4 vec;
      float a_scale;
    };
    auto fetch = [&](const TileCoord& tc) -> Pre {
      Pre pr;
      pr.vec = make_float4(0.f, 0.f, 0.f, 0.f);
      pr.a_scale = 1.0f;
      const TcSeg& sg = P.segs[tc.seg];
      const int n0 = tc.n_tile * KV_BLOCK_N;
      if (sg.col_vec && lane < 16) pr.vec = ldg_f4(sg.col_vec + n0 + ((n0 < sg.rope_cols) ? vcol_k : vcol_v));
      if (SCALED && sg.a_scale) {
        const int row = tc.m_tile * BLOCK_M + q * 32 + lane;
        if (row < P.M) pr.a_scale = __ldg(sg.a_scale + row);
      }
      return pr;
    };

    int it = 0;
    int sslot = 0;
    uint32_t sphase = 0;
    for (int round = 0;; ++round) {
      int t_begin = s_begin, t_end = s_end;
      if (!DYN) {
        if (round) break;
      } else {
        ptx::mbar_wait_suspend(&bars->sched_full[sslot], sphase);
        t_begin = *(volatile int*)&bars->sched_begin[sslot];
        t_end = *(volatile int*)&bars->sched_end[sslot];
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&bars->sched_empty[sslot]);
        if (++sslot == KV_SCHED_SLOTS) { sslot = 0; sphase ^= 1; }
        if (t_begin < 0) break;
      }
    Pre cur;
    TileCoord tc = tile_coord<DYN>(P, t_begin);
    if (t_begin < t_end) cur = fetch(tc);
    for (int tile = t_begin; tile < t_end; ++tile, ++it) {
      TileCoord tn = tc;
      tile_next<DYN>(P, tn);
      const TcSeg& sg = P.segs[tc.seg];
      const int acc = it & 1;
      const uint32_t acc_phase = (it >> 1) & 1;
      const int n0 = tc.n_tile * KV_BLOCK_N;
      const bool is_k = n0 < sg.rope_cols;

      if (tc.m_tile != cur_m || (DYN && tc.seg != cur_seg)) {
        cur_m = tc.m_tile;
        cur_seg = tc.seg;
        const int row = cur_m * BLOCK_M + q * 32 + lane;
        int pos = 0;
        long long slot = -1;                                    // stays -1 for rows beyond M and page ids outside the pool
        rs_row = 1.0f;
        if (row < P.M) {
          row_to_pos_slot(P.batch, row, pos, slot);
          if (SCALED && sg.rowscale_in) {                       // NORM_RMS (PATCH GEMM-3; several segments only with DYN)
            float ss = 0.0f;
            for (int p = 0; p < P.n_partials; ++p) ss += __ldg(sg.rowscale_in + (size_t)p * P.M + row);
            rs_row = rsqrtf(ss / (float)P.rms_dim + P.rms_eps);
          }
        }
        if (ARES) {                                             // written once the previous tile's copy-out has drained
          slot_reg = (int)slot;
          slot_dirty = true;
        } else {
          __syncwarp();
          asm volatile("st.shared.b32 [%0], %1;" ::"r"(wslot + lane * 4), "r"((int)slot) : "memory");
          __syncwarp();
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const float2 x = rope_cs(pos, P.rope_g[16 * g + 2 * i]), y = rope_cs(pos, P.rope_g[16 * g + 2 * i + 1]);
          c2[i] = f2_pack(x.x, y.x);
          s2[i] = f2_pack(x.y, y.y);
        }
      }
      const float rs = rs_row * cur.a_scale;
      const unsigned long long rs2 = f2_pack(rs, rs);
      const bool to1 = n0 >= P.split;
      // address of this lane's 16 bytes in slot 0 of the tile's pool columns; a row adds slot * row_stride
      const unsigned long long tile_base = (unsigned long long)(to1 ? sg.out1 : sg.out0) +
                                           (unsigned long long)(to1 ? n0 - P.split : n0) * (P8 ? 1ull : 2ull) +
                                           (unsigned long long)(P8 ? (lane & 15) : lane) * 16ull;
      // fp8 pools: scale of this lane's head = [slot][head]
      float* scale_base = nullptr;
      if (P8) scale_base = (to1 ? sg.scale1 : sg.scale0) + ((to1 ? n0 - P.split : n0) >> 7) + ((lane >> 3) & 1);
      const uint32_t scale_stride = (uint32_t)(P.pool_width >> 7);

      // this warp's slice of the tile's mean / bias: wv[16 * run + i].  ARES: the slice is shared by the column group's four
      // warps and written AFTER the accumulator has arrived -- by then every quadrant has handed back the tile before last,
      // the previous user of this buffer
      const uint32_t wv = ARES ? wvec + (uint32_t)acc * 256 : wvec;
      if (!ARES) {
        __syncwarp();
        if (lane < 16)
          asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(wv + lane * 16), "f"(cur.vec.x), "f"(cur.vec.y),
                       "f"(cur.vec.z), "f"(cur.vec.w) : "memory");
        __syncwarp();
      }

      ptx::mbar_wait_suspend(&bars->tmem_full[acc], acc_phase);
      ptx::tc_fence_after();
      if (ARES) {
        if (lane < 16)
          asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(wv + lane * 16), "f"(cur.vec.x), "f"(cur.vec.y),
                       "f"(cur.vec.z), "f"(cur.vec.w) : "memory");
        __syncwarp();
      }
      const uint32_t t_row = tmem_base + (uint32_t)(acc * KV_BLOCK_N) + ((uint32_t)(q * 32) << 16);

      Pre nxt = cur;
      if (tile + 1 < t_end) nxt = fetch(tn);

      if (is_k) {
        // ---- K tile: rotate pairs (j, j + 64) of both heads, j in [16g, 16g + 16), eight pairs at a time ----
#pragma unroll
        for (int hh = 0; hh < 4; ++hh) {
          const int h = hh >> 1, hf = hh & 1;                   // head of the tile, half of the warp's 16 frequencies
          uint32_t ra[8], rb[8];
          const int ca = h * 128 + 16 * g + 8 * hf;
          ptx::tmem_ld8(t_row + ca, ra);
          ptx::tmem_ld8(t_row + ca + 64, rb);
          ptx::tmem_ld_wait();
          uint32_t oa[4], ob[4];
#pragma unroll
          for (int q4 = 0; q4 < 2; ++q4) {
            const float4 ma = ptx::lds_f4(wv + ((2 * h) * 16 + 8 * hf + q4 * 4) * 4);
            const float4 mb = ptx::lds_f4(wv + ((2 * h + 1) * 16 + 8 * hf + q4 * 4) * 4);
#pragma unroll
            for (int e = 0; e < 2; ++e) {
              const int i = q4 * 4 + e * 2, k = q4 * 2 + e, kf = 4 * hf + k;
              const unsigned long long am = e ? f2_pack(ma.z, ma.w) : f2_pack(ma.x, ma.y);
              const unsigned long long bm = e ? f2_pack(mb.z, mb.w) : f2_pack(mb.x, mb.y);
              const unsigned long long av = f2_pack(__uint_as_float(ra[i]), __uint_as_float(ra[i + 1]));
              const unsigned long long bv = f2_pack(__uint_as_float(rb[i]), __uint_as_float(rb[i + 1]));
              const unsigned long long a = SCALED ? f2_fma(av, rs2, am) : f2_add(av, am);
              const unsigned long long b = SCALED ? f2_fma(bv, rs2, bm) : f2_add(bv, bm);
              float x0, x1, y0, y1, t0, t1;
              f2_unpack(f2_mul(b, s2[kf]), t0, t1);
              f2_unpack(f2_fma(a, c2[kf], f2_pack(-t0, -t1)), x0, x1);    // a cos - b sin
              f2_unpack(f2_fma(a, s2[kf], f2_mul(b, c2[kf])), y0, y1);    // b cos + a sin
              oa[k] = pack_bf16x2(x0, x1);
              ob[k] = pack_bf16x2(y0, y1);
            }
          }
          if (hh == 0) {
            ptx::named_bar_sync(bar_id, 128);                   // the quadrant's previous copy-out has drained
            if (ARES && slot_dirty) {
              asm volatile("st.shared.b32 [%0], %1;" ::"r"(wslot + lane * 4), "r"(slot_reg) : "memory");
              slot_dirty = false;
            }
          }
          const int k0 = h * 16 + 2 * g + hf;                   // 16-B chunk of run (h, a); run (h, b) = +8
          ptx::sts128(qstg_addr(stg, lane, k0), make_uint4(oa[0], oa[1], oa[2], oa[3]));
          ptx::sts128(qstg_addr(stg, lane, k0 + 8), make_uint4(ob[0], ob[1], ob[2], ob[3]));
        }
      } else {
        // ---- V tile (or K without RoPE): columns [64g, 64g + 64), 16 at a time (32 at a time cost 12 B of spills at the
        // epilogue's 112-register cap, and a spill reload queues behind the copy-out stores) ----
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          uint32_t r[16];
          ptx::tmem_ld16(t_row + 64 * g + 16 * c, r);
          ptx::tmem_ld_wait();
          uint32_t o[8];
#pragma unroll
          for (int q4 = 0; q4 < 4; ++q4) {
            const float4 m4 = ptx::lds_f4(wv + (c * 16 + q4 * 4) * 4);
            float v0, v1, v2, v3;
            const unsigned long long r01 = f2_pack(__uint_as_float(r[q4 * 4]), __uint_as_float(r[q4 * 4 + 1]));
            const unsigned long long r23 = f2_pack(__uint_as_float(r[q4 * 4 + 2]), __uint_as_float(r[q4 * 4 + 3]));
            f2_unpack(SCALED ? f2_fma(r01, rs2, f2_pack(m4.x, m4.y)) : f2_add(r01, f2_pack(m4.x, m4.y)), v0, v1);
            f2_unpack(SCALED ? f2_fma(r23, rs2, f2_pack(m4.z, m4.w)) : f2_add(r23, f2_pack(m4.z, m4.w)), v2, v3);
            o[q4 * 2] = pack_bf16x2(v0, v1);
            o[q4 * 2 + 1] = pack_bf16x2(v2, v3);
          }
          if (c == 0) {
            ptx::named_bar_sync(bar_id, 128);
            if (ARES && slot_dirty) {
              asm volatile("st.shared.b32 [%0], %1;" ::"r"(wslot + lane * 4), "r"(slot_reg) : "memory");
              slot_dirty = false;
            }
          }
          const int k0 = 8 * g + 2 * c;
          ptx::sts128(qstg_addr(stg, lane, k0), make_uint4(o[0], o[1], o[2], o[3]));
          ptx::sts128(qstg_addr(stg, lane, k0 + 1), make_uint4(o[4], o[5], o[6], o[7]));
        }
      }
      // staging complete and all TMEM reads of the quadrant done: hand the accumulator back, copy out
      ptx::tc_fence_before();
      ptx::named_bar_sync(bar_id, 128);
      if (g == 0 && lane == 0) ptx::mbar_arrive(&bars->tmem_empty[acc]);
      if (P8) {
        // fp8 pools: a warp pass covers TWO rows -- lanes 0-15 the even row, 16-31 the odd one -- and a lane converts 16
        // columns (two staged chunks) into one 16-byte store, so the store instructions carry full 16-byte lanes as in
        // the bf16 path.  A head is 8 lanes: its amax takes 3 shuffles; s = amax / 448, bytes = e4m3(x * (1 / s)).
        const int hl = lane & 15;
#pragma unroll
        for (int p2 = 0; p2 < 4; ++p2) {
          const int r = 8 * g + 2 * p2 + (lane >> 4);
          int slot;
          asm volatile("ld.shared.b32 %0, [%1];" : "=r"(slot) : "r"(wslot + r * 4) : "memory");
          const uint4 x0 = ptx::lds128(qstg_addr(stg, r, 2 * hl)), x1 = ptx::lds128(qstg_addr(stg, r, 2 * hl + 1));
          const uint32_t w[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
          float a = 0.0f;
#pragma unroll
          for (int j = 0; j < 8; ++j) a = fmaxf(a, fmaxf(fabsf(__uint_as_float(w[j] << 16)), fabsf(__uint_as_float(w[j] & 0xffff0000u))));
#pragma unroll
          for (int o = 1; o < 8; o <<= 1) a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, o));
          const float sc = a > 0.0f ? __fdiv_rn(a, 448.0f) : 1.0f;
          const float inv = __fdiv_rn(1.0f, sc);
          uint32_t o4[4];
#pragma unroll
          for (int j = 0; j < 4; ++j)
            o4[j] = float2_to_e4m3x2_sat(__fmul_rn(__uint_as_float(w[2 * j] << 16), inv), __fmul_rn(__uint_as_float(w[2 * j] & 0xffff0000u), inv)) |
                    (float2_to_e4m3x2_sat(__fmul_rn(__uint_as_float(w[2 * j + 1] << 16), inv), __fmul_rn(__uint_as_float(w[2 * j + 1] & 0xffff0000u), inv)) << 16);
          if (slot >= 0) {
            ptx::stg128_cs(tile_base + (unsigned long long)(uint32_t)slot * row_stride, make_uint4(o4[0], o4[1], o4[2], o4[3]));
            if ((lane & 7) == 0) scale_base[(size_t)(uint32_t)slot * scale_stride] = sc;
          }
        }
      } else {
        uint4 v[8];
        int sl[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const int r = 8 * g + i;
          asm volatile("ld.shared.b32 %0, [%1];" : "=r"(sl[i]) : "r"(wslot + r * 4) : "memory");
          v[i] = ptx::lds128(qstg_addr(stg, r, lane));
        }
#pragma unroll
        for (int i = 0; i < 8; ++i)
          if (sl[i] >= 0) ptx::stg128_cs(tile_base + (unsigned long long)(uint32_t)sl[i] * row_stride, v[i]);
      }
      cur = nxt;
      tc = tn;
    }
    }
  }

  // ============================== teardown ==============================
  ptx::tc_fence_before();
  if (P.dep_wait_late && threadIdx.x == 0) ptx::grid_dep_wait();
  __syncthreads();
  if (warp == 0) ptx::tmem_dealloc<TMEM_COLS>(tmem_base);
}

// ---------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------
bool tc_kv_eligible(const scd_plan_t* p, const TcParams& P) {
  if (p->model.head_dim != 128 || p->model.rope_style != SCD_ROPE_HALF) return false;
  if (P.block_n != KV_BLOCK_N || (P.N % KV_BLOCK_N) || (P.split % KV_BLOCK_N) || P.a_kb_per_head != 0) return false;
  for (int i = 0; i < P.n_segs; ++i) {
    if (P.segs[i].rope_cols % KV_BLOCK_N) return false;
  }
  return true;
}

scd_status_t launch_tc_kv(const scd_plan_t* p, TcParams& P, cudaStream_t s) {
  P.m_tiles = (P.M + BLOCK_M - 1) / BLOCK_M;
  P.n_tiles = P.N / KV_BLOCK_N;
  P.num_kb = (P.K + BLOCK_K - 1) / BLOCK_K;
  const int total = P.n_segs * P.m_tiles * P.n_tiles;
  if (total <= 0) return SCD_OK;
  P.stages = kv_pick_stages(P.num_kb);
  const size_t smem = kv_smem_bytes(P.stages);
  static std::atomic<size_t> configured[SCD_MAX_DEVICES];      // the attribute belongs to (function, device)
  if (configured[p->device].load(std::memory_order_relaxed) < smem) {
    cudaError_t e = cudaFuncSetAttribute(tc_kv_kernel<false, false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(tc_kv_kernel<false, true, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(tc_kv_kernel<true, true, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(tc_kv_kernel<false, true, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(tc_kv_kernel<false, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(tc_kv_kernel<true, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(tc_kv_kernel<false, true, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return fail(SCD_E_CUDA, "cudaFuncSetAttribute(kv smem %zu): %s", smem, cudaGetErrorString(e));
    configured[p->device].store(smem, std::memory_order_relaxed);
  }
  // bf16 codes on bf16 pools, plain REUSE decode (no row scales): resident code tile as well -- the ring then holds basis tiles
  // only and a code tile leaves L2 once per (m-tile, segment) instead of once per n-tile.  Measured on config-2 geometry
  // (profiles/r02_decode_history.md section 17): faster at one k-block per tile (r <= 64: four tiles' basis in flight instead of two
  // whole stages; config 3 0.508 -> 0.469 ms) and at three or four (r = 192, 256: +1-2 %), slower at two (r = 96, 128: -4 %,
  // where three 48 KB stages already hold 1.5 tiles) -- so two k-blocks keep the plain kernel
  {
    bool any_scale = false;
    for (int i = 0; i < P.n_segs; ++i) any_scale |= P.segs[i].rowscale_in != nullptr || P.segs[i].a_scale != nullptr;
    if (KV_ARES_BF16 && P.code_dtype == SCD_BF16 && P.a_is_codes && !any_scale && !P.pool_e4m3 && P.head_rank == 0 && P.num_kb <= 4 &&
        P.num_kb != 2 && P.n_tiles > 1) {
      P.stages = kva_pick_stages(P.num_kb);
      const size_t smem_b_ = kva_smem_bytes(P.stages, P.num_kb);
      static std::atomic<size_t> conf_b[SCD_MAX_DEVICES];
      if (conf_b[p->device].load(std::memory_order_relaxed) < smem_b_) {
        cudaError_t e = cudaFuncSetAttribute(tc_kv_kernel<false, false, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_b_);
        if (e != cudaSuccess) return fail(SCD_E_CUDA, "cudaFuncSetAttribute(kv resident bf16 smem %zu): %s", smem_b_, cudaGetErrorString(e));
        conf_b[p->device].store(smem_b_, std::memory_order_relaxed);
      }
      if ((long long)P.pool_slots >= (1ll << 31)) return fail(SCD_E_UNSUPPORTED, "pools of more than 2^31 slots");
      prof_begin(s);
      launch_pdl(tc_kv_kernel<false, false, false, false, true>, std::min(total, p->sm_count), KV_NTHREADS, smem_b_, s, 1, P);
      prof_end(s, P.prof_id);
      cudaError_t e = cudaGetLastError();
      if (e != cudaSuccess) return fail(SCD_E_CUDA, "tc_kv_kernel (resident bf16 code tile) launch: %s", cudaGetErrorString(e));
      count_launch();
      return SCD_OK;
    }
  }
  // e4m3 codes of rank <= 256 on bf16 pools: the code tile stays resident across its n-tiles
  if (KV_ARES && P.code_dtype == SCD_E4M3_ROWSCALE && P.a_is_codes && !P.pool_e4m3 && P.head_rank == 0 && P.num_kb <= 4 && P.n_tiles > 1) {
    P.stages = kva_pick_stages(P.num_kb);
    const size_t smem_a_ = kva_smem_bytes(P.stages, P.num_kb);
    static std::atomic<size_t> conf_a[SCD_MAX_DEVICES];
    if (conf_a[p->device].load(std::memory_order_relaxed) < smem_a_) {
      cudaError_t e = cudaFuncSetAttribute(tc_kv_kernel<false, true, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_a_);
      if (e != cudaSuccess) return fail(SCD_E_CUDA, "cudaFuncSetAttribute(kv resident smem %zu): %s", smem_a_, cudaGetErrorString(e));
      conf_a[p->device].store(smem_a_, std::memory_order_relaxed);
    }
    if ((long long)P.pool_slots >= (1ll << 31)) return fail(SCD_E_UNSUPPORTED, "pools of more than 2^31 slots");
    prof_begin(s);
    launch_pdl(tc_kv_kernel<false, true, true, false, true>, std::min(total, p->sm_count), KV_NTHREADS_E4, smem_a_, s, 1, P);
    prof_end(s, P.prof_id);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SCD_E_CUDA, "tc_kv_kernel (resident code tile) launch: %s", cudaGetErrorString(e));
    count_launch();
    return SCD_OK;
  }
  const int grid = std::min(total, p->sm_count);
  // long tiles (K = d_model: PATCH GEMM-3): KV_STATIC_PCT % of an even split is owned statically, the rest is
  // claimed tile by tile; short tiles (REUSE decode): static split only
  bool multi_rowscale = false, scaled = false;              // several layers' RMS scales: only the DYN variant tracks the segment
  for (int i = 0; i < P.n_segs; ++i) {
    multi_rowscale |= P.n_segs > 1 && P.segs[i].rowscale_in != nullptr;
    scaled |= P.segs[i].rowscale_in != nullptr || P.segs[i].a_scale != nullptr;
  }
  if ((long long)P.pool_slots >= (1ll << 31)) return fail(SCD_E_UNSUPPORTED, "pools of more than 2^31 slots");
  const bool dyn = (P.num_kb >= 16 && total > grid) || multi_rowscale;
  const bool ae4 = P.code_dtype == SCD_E4M3_ROWSCALE && P.a_is_codes;
  if (ae4 && dyn) return fail(SCD_E_UNSUPPORTED, "internal: e4m3 codes on the dynamically scheduled paged-KV kernel");
  prof_begin(s);
  const bool p8 = P.pool_e4m3 != 0;
  if (dyn) {
    P.chunk_tiles = 1;
    P.static_tiles = (int)((long long)total * KV_STATIC_PCT / 100 / grid);
    P.dyn_begin = grid * P.static_tiles;
    P.n_chunks = total - P.dyn_begin;
    P.sched = p->kv_sched + 2 * (p->kv_sched_next.fetch_add(1) % KV_SCHED_SETS);
  }
  if (ae4) {
    if (p8) launch_pdl(tc_kv_kernel<false, true, true, true>, grid, KV_NTHREADS_E4, smem, s, 1, P);
    else launch_pdl(tc_kv_kernel<false, true, true, false>, grid, KV_NTHREADS_E4, smem, s, 1, P);
  } else if (dyn) {
    if (p8) launch_pdl(tc_kv_kernel<true, true, false, true>, grid, KV_NTHREADS, smem, s, 1, P);
    else launch_pdl(tc_kv_kernel<true, true, false, false>, grid, KV_NTHREADS, smem, s, 1, P);
  } else if (p8) {
    launch_pdl(tc_kv_kernel<false, true, false, true>, grid, KV_NTHREADS, smem, s, 1, P);
  } else if (scaled) {
    launch_pdl(tc_kv_kernel<false, true, false, false>, grid, KV_NTHREADS, smem, s, 1, P);
  } else {
    launch_pdl(tc_kv_kernel<false, false, false, false>, grid, KV_NTHREADS, smem, s, 1, P);
  }
  prof_end(s, P.prof_id);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(SCD_E_CUDA, "tc_kv_kernel launch: %s", cudaGetErrorString(e));
  count_launch();
  return SCD_OK;
}

}  // namespace scd
