// Persistent, warp-specialised tcgen05 GEMM for the four vocab-sized contractions of the GRPO step
// (SURVEY.md §8(a) rows A2, A4, A5, A6), with the method's epilogues fused behind the TMEM accumulator.
//
//   warps 0..3  : epilogue       (tcgen05.ld 32x32b: one accumulator row per thread; warp w owns TMEM lanes 32w..)
//   warp 4      : TMA producer   (cp.async.bulk.tensor -> 128B-swizzled smem ring, mbarrier complete_tx)
//   warp 5      : MMA issuer     (tcgen05.mma kind::f16, fp32 accumulators in TMEM, 2 accumulator stages)
//   warp 6      : drift gate     (one thread polls the launch's epoch counters, see "Drift bound" below)
// Producer and MMA warps walk their loops with all 32 lanes converged and ONE elected lane issuing, so that
// addresses, coordinates and descriptors are warp-uniform (uniform registers; a lane-0-only producer loop paid
// an ELECT + four R2UR.BROADCAST per TMA instruction and starved the tensor pipe).  The two issuing warps have
// the highest warp ids of their scheduler partitions, so the arbiter never parks them behind an epilogue warp.
//
// Shared memory: ring stages | 16 KB staging for the A6 epilogue (one 32 x 32 fp32 block per epilogue warp,
// reduced into dW by a TMA reduce-add) | barriers.
//
// CG = 1: one CTA per SM, C tile = 128 x 256, K block = 64 bf16 (one 128-byte swizzle row), 4-stage
//         smem ring of 48 KB stages.
// CG = 2: CTA pairs (cluster of 2 = one TPC), tcgen05 cta_group::2, pair tile = 256 x 256: CTA r of the
//         pair stages A rows [r*128, +128) and B rows [r*128, +128) of the tile (32 KB per stage, 7-stage
//         ring; 6 for A6), the leader's MMA thread issues M=256 N=256 instructions that read both CTAs' smem, and
//         each CTA holds its own 128 accumulator rows in its TMEM.  Per-SM L2->smem traffic and smem
//         operand reads drop by a third against CG = 1 at the same per-SM MMA rate.
// Both: 2 x 256 TMEM columns so the epilogue of tile i overlaps the MMAs of tile i+1.
//
// Operand layouts (template): K-major (row = M/N index, 64 contiguous k) or MN-major (row = k index,
// 64 contiguous m/n per 8 KB box).  Row-major tensors are consumed as they are; nothing is transposed
// in memory:
//   A2/A4  z  = H W^T        A = H  [T,d]  K-major   B = W  [V,d]  K-major    K = d
//   A5     dH = dZ W         A = dZ [Tc,V] K-major   B = W  [V,d]  MN-major   K = V
//   A6     dW += dZ^T H      A = dZ [Tc,V] MN-major  B = H  [Tc,d] MN-major   K = Tc
#pragma once
#include "ptx_sm100.cuh"

namespace grpo {

constexpr int BM = 128, BN = 256, BK = 64;
constexpr int kMaxStages = 8;
constexpr int kABytes = BM * BK * 2;        // 16 KB
constexpr int kGemmThreads = 224;
constexpr int kProducerWarp = 4, kMmaWarp = 5, kGateWarp = 6;
constexpr int kTmemCols = 512;
constexpr int kRedStageBytes = 4 * 32 * 32 * 4;   // A6 epilogue: one 32 x 32 fp32 block per epilogue warp (16 KB)
// Ring depth: as many 32 KB stages as the 227 KB of shared memory hold - 7, or 6 for the A6 instance, whose
// epilogue needs 16 KB of staging (A/B on one box, 3 runs each: 7 stages A4 -2 %, A2 / A5 -0.6 % against 6).
template <int CG, int EPI> struct GemmShape {
  static constexpr int kBRows = BN / CG;                       // B rows (N index) staged by one CTA
  static constexpr int kBBytes = kBRows * BK * 2;              // 32 KB / 16 KB
  static constexpr int kStageBytes = kABytes + kBBytes;        // 48 KB / 32 KB
  static constexpr int kRedBytes = EPI == 3 ? kRedStageBytes : 0;   // only the A6 epilogue stages its blocks
  static constexpr int kStages = CG == 1 ? 4 : (EPI == 3 ? 6 : 7);
  static constexpr int kSmemBytes = kStages * kStageBytes + kRedBytes + 1024 /*align slack*/ + 256 /*barriers*/;
};
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

enum Epi : int { EPI_LSE = 0, EPI_DZ = 1, EPI_STORE = 2, EPI_RED_F32 = 3, EPI_LSE_STASH = 4 };
// EPI_LSE_STASH (3-contraction variant): EPI_LSE that also writes, for every logit, the
// exponential e = 2^(z2 - m) it adds to the running sum (z2 = z s log2(e), m = the row's running max after the
// element's 256-column tile) as fp16 into the chunk buffer `dz`, and m per (row, tile) into `stash_shift`;
// stash_to_dz_kernel later turns e into dZ = k (1[v = y] - e 2^(m - lse2)) in place.  Stashing e instead of the
// logit keeps the relative error of every probability at fp16's 2^-11 whatever the magnitude of the logits.
__host__ __device__ constexpr bool is_lse(int epi) { return epi == EPI_LSE || epi == EPI_LSE_STASH; }

struct GemmParams {
  int m_total, n_total;              // valid rows / cols of C
  int m_tiles, n_tiles, k_blocks;
  int n_fastest;                     // unit order: 1 = n tile fastest (A5/A6), 0 = m tile fastest (A2/A4)
  // L2 working-set bounds of the unit ORDER (never of a reduction: results do not depend on them).  n_fastest = 1:
  // the n tiles are walked in groups of n_group (all m tiles of a group before the next group), so that the B
  // panels a wave re-reads from L2 - A6: the chunk's hidden-state columns - stay what they are at d = 2048 when d
  // is larger.  n_fastest = 0: the m tiles are walked in blocks of m_block (all n tiles of a block before the next
  // block; A4: the block's hidden-state rows stay L2-resident while W streams).  0 = one group / block.
  int n_group, m_block;
  // EPI_LSE: a unit is (m tile, contiguous range of n tiles).  The vocab split is a function of V ALONE (never of
  // the launch's row count), so a token's log-sum-exp is summed in the same order whatever launch it is part of
  // (batch invariance).  Units are walked in blocks of `lse_block` m tiles (= CTA pairs of the
  // grid): inside a block the m tile is fastest, then the split, so that the pairs running together share W tiles
  // through L2 while the block's H rows stay L2-resident and W is streamed once per block.
  int n_split, tiles_per_split, lse_block;
  // split-K (A5): the reduction is cut into k_split contiguous ranges of kb_per_split k blocks, again a function
  // of the problem's K alone; split ks stores its fp32 partial tile at c_out + ks * c_split_stride, and
  // splitk_reduce_kernel adds the partials in a fixed order.  k_split <= 1: off.
  int k_split, kb_per_split;
  int64_t c_split_stride;
  // rows (A4 / A5: m_total; A6: reduction length) of this launch read from device memory (written by
  // compact_rows_kernel: token-granular zero-coefficient compaction).  nullptr: the static
  // m_total / k_blocks.  m_alloc: rows the dZ buffer holds (EPI_DZ zero-fills the rows of its last walked tile
  // beyond the dynamic row count, which A6 reads as part of its last k block).
  const int* dyn_rows;
  int m_alloc;
  // per-token arrays are indexed by (row_offset + local row)
  int64_t row_offset;
  const int32_t* targets;
  float scale_log2e;                 // logit_scale * log2(e)
  float logit_scale;
  // FP8 study (DT = 1): the accumulator is (H8 W8^T)[t, v]; the logit is that times the
  // token's quantisation scale row_scale[t] times the vocab matrix' scale *w_scale.  nullptr: 1.
  const float* row_scale;
  const float* w_scale;
  // EPI_LSE outputs (log2 domain running max / sum per split) + the target logit
  float* part_m;
  float* part_s;
  float* part_u;                     // nullable: sum 2^(z2 - max) z2 per split, for the entropy output (R28)
  int64_t part_stride;
  float* zy;
  // EPI_DZ
  const float* lse;
  const float* coeff;
  float coeff_mul;                   // logit_scale * grad_scale
  __nv_bfloat16* dz;
  int64_t dz_pitch;
  float* stash_shift;                // EPI_LSE_STASH: running max (log2 domain) per (row, 256-column tile)
  int64_t shift_pitch;
  // EPI_STORE / EPI_RED_F32: fp32 C
  void* c_out;
  int64_t c_pitch;                   // elements
  // drift bound between the CTA pairs of one launch (see the producer loop); sync == nullptr: off
  unsigned int* sync;
  int sync_epoch_kb;                 // k blocks per epoch
  int sync_epochs;                   // counters in `sync` (epochs any pair can reach)
  int sync_lag;                      // a pair may run this many epochs ahead of the slowest pair (>= 1)
};

struct alignas(8) GemmBarriers {
  uint64_t full[kMaxStages];
  uint64_t empty[kMaxStages];
  uint64_t tmem_full[2];
  uint64_t tmem_empty[2];
  uint32_t tmem_base;
  int gate_open;                     // highest epoch the producer may enter (written by the gate warp)
};

// Effective extent of a launch under row compaction: the rows of C that exist, the number of m
// tiles walked (A4/A5), the k blocks per unit (A6) and the unit count.  Uniform over the grid (one global load).
struct Extent { int m_total, m_tiles, k_blocks, n_units; };
template <int CG, int EPI>
__device__ __forceinline__ Extent launch_extent(const GemmParams& p, int n_units) {
  Extent e{p.m_total, p.m_tiles, p.k_blocks, n_units};
  if constexpr (is_lse(EPI)) return e;
  const int ks = p.k_split > 1 ? p.k_split : 1;
  if (p.dyn_rows != nullptr) {
    const int rows = *p.dyn_rows;
    if constexpr (EPI == EPI_RED_F32) {
      e.k_blocks = min(p.k_blocks, (rows + BK - 1) / BK);
      if (e.k_blocks == 0) e.n_units = 0;              // nothing to add: no MMA, so no epilogue either
    } else {
      e.m_total = min(p.m_total, rows);
      e.m_tiles = min(p.m_tiles, (e.m_total + BM * CG - 1) / (BM * CG));
      e.n_units = e.m_tiles * p.n_tiles * ks;
    }
  }
  return e;
}
// One scheduling unit: output tile(s) [m_tile] x [n0, n1) reduced over k blocks [kb0, kb1); `part` is the vocab
// split (EPI_LSE) or the K split (split-K stores) the unit belongs to.
struct Unit { int m_tile, n0, n1, kb0, kb1, part; };
template <int EPI>
__device__ __forceinline__ Unit unit_to_tiles(const GemmParams& p, const Extent& e, int u) {
  Unit t;
  t.kb0 = 0;
  t.kb1 = e.k_blocks;
  t.part = 0;
  if constexpr (is_lse(EPI)) {
    const int per_block = p.lse_block * p.n_split;       // only the last block of m tiles can be short
    const int b = u / per_block, r = u - b * per_block;
    const int mb = min(p.lse_block, p.m_tiles - b * p.lse_block);
    t.part = r / mb;
    t.m_tile = b * p.lse_block + (r - t.part * mb);
    t.n0 = t.part * p.tiles_per_split;
    t.n1 = min(p.n_tiles, t.n0 + p.tiles_per_split);
    return t;
  }
  if (p.k_split > 1) {                                    // K split slowest: a wave streams one K range
    const int per_split = e.m_tiles * p.n_tiles;
    t.part = u / per_split;
    u -= t.part * per_split;
    t.kb0 = t.part * p.kb_per_split;
    t.kb1 = min(e.k_blocks, t.kb0 + p.kb_per_split);
  }
  int m_idx;
  if (p.n_fastest) {                                      // groups of n tiles; inside a group: m tile, then n tile fastest
    const int ng = p.n_group > 0 ? min(p.n_group, p.n_tiles) : p.n_tiles;
    const int per_group = ng * e.m_tiles;                 // only the last group can be short
    const int g = u / per_group, r = u - g * per_group;
    const int gsz = min(ng, p.n_tiles - g * ng);
    m_idx = r / gsz;
    t.n0 = g * ng + (r - m_idx * gsz);
  } else {                                                // blocks of m tiles; inside a block: n tile, then m tile fastest
    const int mb = p.m_block > 0 ? min(p.m_block, e.m_tiles) : e.m_tiles;
    const int per_block = mb * p.n_tiles;                 // only the last block can be short
    const int b = u / per_block, r = u - b * per_block;
    const int bsz = min(mb, e.m_tiles - b * mb);
    t.n0 = r / bsz;
    m_idx = b * mb + (r - t.n0 * bsz);
  }
  t.n1 = t.n0 + 1;
  t.m_tile = m_idx;
  return t;
}

// Drift bound.  The CTA pairs of a launch that share operand panels through L2 (the 8 d-tiles of one dZ
// row panel in A5/A6, every pair's W tile in A2/A4) only hit in L2 while they stream the same k blocks at
// about the same time; pairs that start late (the previous kernel's tail) or drift re-fetch the panels
// from HBM (measured: 16.6 GB instead of 5.4 GB per A5 launch), which costs DRAM power on a power-capped
// board.  Every `sync_epoch_kb` k blocks the producer of each pair arrives on the global counter of its
// epoch e and enters it only once every pair has arrived on epoch e-1.  The polling is done by a
// separate warp that publishes the open epoch in shared memory, so the producer never waits on a
// global load in steady state.  This is a performance gate, never a correctness one: every wait is
// bounded (pairs of two launches on different streams may not all be co-resident), and after
// kGateMaxTimeouts timeouts a pair stops gating; a pair that is done arrives for all later epochs.
constexpr long long kGateTimeoutClk = 600000;   // ~0.4 ms
constexpr int kGateMaxTimeouts = 2;
constexpr int kGateOff = 0x7fffffff;

__device__ __forceinline__ int ld_volatile_shared_i32(const int* p) {
  int v;
  asm volatile("ld.volatile.shared.b32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
  return v;
}
__device__ __forceinline__ void st_volatile_shared_i32(int* p, int v) {
  asm volatile("st.volatile.shared.b32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}

// DT: operand type of the contraction: 0 = bf16 (kind::f16, 64 elements per 128-byte k block), 1 = e4m3
// (kind::f8f6f4, 128 elements per k block; K-major operands only).  Shared-memory layout, descriptors and the four
// K = 32-byte MMAs per k block are byte-identical.
template <int CG, bool A_MN, bool B_MN, int EPI, int DT = 0>
__global__ void __launch_bounds__(kGemmThreads, 1)
grpo_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                 const __grid_constant__ CUtensorMap tmC, const GemmParams p, const int n_units_dense) {
  using Shape = GemmShape<CG, EPI>;
  constexpr int kStages = Shape::kStages;
  constexpr int kStageBytes = Shape::kStageBytes;
  constexpr int kBRows = Shape::kBRows;
  constexpr int kBKe = DT == 1 ? 2 * BK : BK;                    // elements per k block (128 bytes)
  static_assert(DT == 0 || (!A_MN && !B_MN), "the e4m3 instance is K-major only");
  // L2 eviction priorities (measured with ncu, profiles/r02c_l2_hints.md).  A6 streams its dZ column panel once
  // (evict_first), re-reads the chunk's H rows for every vocab panel (evict_last) and touches every dW line once
  // (reduce-add evict_first): DRAM reads per launch 6.7 -> 5.1 GB.  The other instances are best WITHOUT a hint:
  // evict_first on the dZ panel of A5 or on the W tiles of A4 evicts lines before the other pairs of the wave
  // have read them (A5 5.6 -> 9.7 GB, A4 0.7 -> 1.4 GB).
  constexpr int kHintA = EPI == EPI_RED_F32 ? kL2EvictFirst : kL2None;
  constexpr int kHintB = EPI == EPI_RED_F32 ? kL2EvictLast : kL2None;
  extern __shared__ uint8_t smem_raw[];
  // SWIZZLE_128B atoms need 1024-byte alignment of the tile bases (same offset in both CTAs of a pair)
  const uint32_t raw_addr = smem_u32(smem_raw);
  const uint32_t pad = (1024u - (raw_addr & 1023u)) & 1023u;
  uint8_t* smem = smem_raw + pad;
  const uint32_t tiles_addr = raw_addr + pad;
  GemmBarriers* bars = reinterpret_cast<GemmBarriers*>(smem + kStages * kStageBytes + Shape::kRedBytes);

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const uint32_t cta_rank = CG == 2 ? cluster_ctarank() : 0u;   // 0 = leader (issues the MMAs)
  const int unit0 = blockIdx.x / CG;                             // CTA pairs walk the unit list together
  const int unit_step = gridDim.x / CG;
  const Extent ext = launch_extent<CG, EPI>(p, n_units_dense);
  const int n_units = ext.n_units;

  if (warp == kProducerWarp && lane == 0) {
    prefetch_tmap(&tmA);
    prefetch_tmap(&tmB);
    for (int i = 0; i < kStages; ++i) {
      mbar_init(&bars->full[i], 1);
      mbar_init(&bars->empty[i], 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&bars->tmem_full[i], 1);
      mbar_init(&bars->tmem_empty[i], 4 * CG);  // one arrive per epilogue warp of every CTA of the pair
    }
    bars->gate_open = 0;
    fence_barrier_init();
  }
  if (warp == kMmaWarp) tmem_alloc<CG>(&bars->tmem_base, kTmemCols);
  tc_fence_before();
  if constexpr (CG == 2) cluster_sync_all(); else __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = bars->tmem_base;

  if (warp == kProducerWarp) {
    // ================================================================ TMA producer
    // Like the MMA warp, the whole warp walks the loop converged and one elected lane issues: every
    // address and coordinate is then warp-uniform and lives in uniform registers (a lane-0-only loop costs
    // an ELECT + four R2UR.BROADCAST per TMA instruction, which made this thread the bottleneck of A6).
    {
      const bool leader_lane = elect_one();
      const uint64_t pol_a = l2_policy<kHintA>(), pol_b = l2_policy<kHintB>();
      const uint32_t full0 = CG == 2 ? mapa_cluster(smem_u32(&bars->full[0]), 0) : smem_u32(&bars->full[0]);
      int stage = 0;
      uint32_t phase = 0;
      bool sync_on = p.sync != nullptr && cta_rank == 0;
      int epoch = 0, to_epoch = 1;
      for (int u = unit0; u < n_units; u += unit_step) {
        const Unit un = unit_to_tiles<EPI>(p, ext, u);
        const int a_row = (un.m_tile * CG + static_cast<int>(cta_rank)) * BM;
        for (int n_tile = un.n0; n_tile < un.n1; ++n_tile) {
          const int b_row = n_tile * BN + static_cast<int>(cta_rank) * kBRows;
          for (int kbw = un.kb0; kbw < un.kb1; ++kbw) {
            const int kb = kbw;
            if (sync_on && --to_epoch == 0) {
              to_epoch = p.sync_epoch_kb;
              if (leader_lane) red_add_u32(p.sync + epoch, 1u);
              const int need = epoch - (p.sync_lag - 1);         // every pair has arrived on epoch need - 1
              if (ld_volatile_shared_i32(&bars->gate_open) < need) {
                const long long t0 = clock64();
                while (ld_volatile_shared_i32(&bars->gate_open) < need)
                  if (clock64() - t0 > 2 * kGateMaxTimeouts * kGateTimeoutClk) { sync_on = false; break; }
                sync_on = __shfl_sync(0xffffffffu, sync_on ? 1 : 0, 0) != 0;   // one decision for the warp
              }
              ++epoch;
            }
            mbar_wait(&bars->empty[stage], phase ^ 1);
            if (leader_lane) {
              // the leader CTA's barrier collects the bytes of both CTAs (one arrival: the leader's)
              if (cta_rank == 0) mbar_arrive_expect_tx(&bars->full[stage], kStageBytes * CG);
              const uint32_t a_dst = tiles_addr + stage * kStageBytes;
              const uint32_t b_dst = a_dst + kABytes;
              const uint32_t bar = full0 + stage * 8;
              if constexpr (!A_MN) {
                tma_load_2d_t<CG, kHintA>(a_dst, &tmA, bar, kb * kBKe, a_row, pol_a);
              } else {
#pragma unroll
                for (int i = 0; i < BM / 64; ++i) tma_load_2d_t<CG, kHintA>(a_dst + i * 8192, &tmA, bar, a_row + i * 64, kb * BK, pol_a);
              }
              if constexpr (!B_MN) {
                tma_load_2d_t<CG, kHintB>(b_dst, &tmB, bar, kb * kBKe, b_row, pol_b);
              } else {
#pragma unroll
                for (int i = 0; i < kBRows / 64; ++i) tma_load_2d_t<CG, kHintB>(b_dst + i * 8192, &tmB, bar, b_row + i * 64, kb * BK, pol_b);
              }
            }
            __syncwarp();
            if (++stage == kStages) { stage = 0; phase ^= 1; }
          }
        }
      }
      // pairs with fewer units must not hold the others back: arrive for every epoch not reached
      if (p.sync != nullptr && cta_rank == 0 && leader_lane)
        for (; epoch < p.sync_epochs; ++epoch) red_add_u32(p.sync + epoch, 1u);
    }
  } else if (warp == kMmaWarp) {
    // ================================================================ MMA issuer (leader CTA only)
    // The whole warp walks the loop converged (waits are warp-wide); one elected lane issues the MMAs and
    // the commits.  Descriptors are a 32-bit add away from a per-kernel constant: the high word and the
    // LBO field never change, the start-address field advances by (bytes >> 4) and cannot carry out of
    // its 14 bits (shared memory is < 256 KB).
    if (cta_rank == 0) {
      constexpr uint32_t idesc = DT == 1 ? make_idesc_e4m3(BM * CG, BN) : make_idesc_bf16(BM * CG, BN, A_MN ? 1 : 0, B_MN ? 1 : 0);
      constexpr uint32_t kDescHi = smem_desc_hi(1024);
      constexpr uint32_t kAdvA = (A_MN ? 2048u : 32u) >> 4, kAdvB = (B_MN ? 2048u : 32u) >> 4;
      const uint32_t a_lo0 = smem_desc_lo(tiles_addr, A_MN ? 8192u : 16u);
      const uint32_t b_lo0 = smem_desc_lo(tiles_addr + kABytes, B_MN ? 8192u : 16u);
      const bool leader_lane = elect_one();
      int stage = 0;
      uint32_t phase = 0;
      int acc = 0;
      uint32_t acc_phase = 0;
      for (int u = unit0; u < n_units; u += unit_step) {
        const Unit un = unit_to_tiles<EPI>(p, ext, u);
        const int n_kb = un.kb1 - un.kb0;
        for (int n_tile = un.n0; n_tile < un.n1; ++n_tile) {
          mbar_wait(&bars->tmem_empty[acc], acc_phase ^ 1);
          tc_fence_after();
          const uint32_t d_tmem = tmem_base + acc * BN;
          for (int kb = 0; kb < n_kb; ++kb) {
            mbar_wait(&bars->full[stage], phase);
            tc_fence_after();
            if (leader_lane) {
              const uint32_t a_lo = a_lo0 + stage * (kStageBytes >> 4);
              const uint32_t b_lo = b_lo0 + stage * (kStageBytes >> 4);
#pragma unroll
              for (int k = 0; k < BK / 16; ++k) {
                if constexpr (DT == 1)
                  umma_f8<CG>(d_tmem, make_desc64(a_lo + k * kAdvA, kDescHi), make_desc64(b_lo + k * kAdvB, kDescHi),
                              idesc, (kb | k) != 0 ? 1u : 0u);
                else
                  umma_bf16<CG>(d_tmem, make_desc64(a_lo + k * kAdvA, kDescHi), make_desc64(b_lo + k * kAdvB, kDescHi),
                                idesc, (kb | k) != 0 ? 1u : 0u);
              }
              umma_commit_t<CG>(&bars->empty[stage]);    // smem slot (of both CTAs) reusable once these MMAs retire
            }
            __syncwarp();
            if (++stage == kStages) { stage = 0; phase ^= 1; }
          }
          if (leader_lane) umma_commit_t<CG>(&bars->tmem_full[acc]);   // accumulator complete -> epilogue (both CTAs)
          __syncwarp();
          acc ^= 1;
          if (acc == 0) acc_phase ^= 1;
        }
      }
    }
  } else if (warp == kGateWarp) {
    // ================================================================ drift gate (leader CTA, one thread)
    if (lane == 0 && cta_rank == 0 && p.sync != nullptr) {
      // epochs this pair's producer enters: ceil(k blocks it issues / epoch length)
      long long my_kb = 0;
      for (int u = unit0; u < n_units; u += unit_step) {
        const Unit un = unit_to_tiles<EPI>(p, ext, u);
        my_kb += static_cast<long long>(un.n1 - un.n0) * (un.kb1 - un.kb0);
      }
      const int my_epochs = static_cast<int>((my_kb + p.sync_epoch_kb - 1) / p.sync_epoch_kb);
      const unsigned int n_pairs = gridDim.x / CG;
      int timeouts = 0;
      for (int e = 1; e < my_epochs; ++e) {
        const long long t0 = clock64();
        while (ld_volatile_u32(p.sync + e - 1) < n_pairs) {
          if (clock64() - t0 > kGateTimeoutClk) { ++timeouts; break; }
          __nanosleep(100);
        }
        if (timeouts >= kGateMaxTimeouts) { st_volatile_shared_i32(&bars->gate_open, kGateOff); break; }
        st_volatile_shared_i32(&bars->gate_open, e);
      }
    }
  } else {
    // ================================================================ epilogue (4 warps, 128 rows)
    const int quad = warp;                             // TMEM lane quarter this warp may access (warp id % 4)
    const int row_in_tile = quad * 32 + lane;
    int acc = 0;
    uint32_t acc_phase = 0;
    [[maybe_unused]] const uint64_t pol_c = l2_policy<kL2EvictFirst>();
    for (int u = unit0; u < n_units; u += unit_step) {
      const Unit un = unit_to_tiles<EPI>(p, ext, u);
      const int m_tile = un.m_tile, n0 = un.n0, n1 = un.n1;
      const int row_local = (m_tile * CG + static_cast<int>(cta_rank)) * BM + row_in_tile;   // row within this launch's C
      const bool row_ok = row_local < ext.m_total;
      const int64_t row_g = p.row_offset + row_local;            // index into per-token arrays

      [[maybe_unused]] int y = -1;
      [[maybe_unused]] float run_m = -INFINITY, run_s = 0.f, run_u = 0.f;   // EPI_LSE running stats (log2 domain)
      [[maybe_unused]] float lse2 = 0.f, kcoef = 0.f;            // EPI_DZ per-row constants
      if constexpr (is_lse(EPI) || EPI == EPI_DZ) {
        if (row_ok) {
          y = p.targets[row_g];
          if (y >= p.n_total) y = -1;
        }
      }
      if constexpr (EPI == EPI_DZ) {
        if (row_ok) {
          lse2 = p.lse[row_g] * kLog2e;
          kcoef = p.coeff[row_g] * p.coeff_mul;
        }
      }
      // logit = accumulator x sl (natural units) = accumulator x sl2 (log2 domain); DT = 1 folds the row's and the
      // vocab matrix' quantisation scales in
      [[maybe_unused]] float sl2 = p.scale_log2e, sl = p.logit_scale;
      if constexpr (DT == 1) {
        if (row_ok) {
          const float rs = p.row_scale[row_g] * *p.w_scale;
          sl2 *= rs;
          sl *= rs;
        }
      }

      for (int n_tile = n0; n_tile < n1; ++n_tile) {
        mbar_wait(&bars->tmem_full[acc], acc_phase);
        tc_fence_after();
        const uint32_t t_addr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + acc * BN;
        const int col_tile = n_tile * BN;
        if constexpr (EPI == EPI_LSE_STASH) {
          // first pass over the accumulator: the tile's maximum, so that one running max covers the whole tile
          float tmax = -INFINITY;
#pragma unroll 1
          for (int c = 0; c < BN / 32; ++c) {
            const int cbase = col_tile + c * 32;
            if (cbase >= p.n_total) break;
            float v[32];
            tmem_ld32(t_addr + c * 32, v);
            tmem_ld_wait();
            const int nvalid = p.n_total - cbase;
            if (nvalid < 32) {
#pragma unroll
              for (int i = 0; i < 32; ++i) v[i] = i < nvalid ? v[i] : -INFINITY;
            }
#pragma unroll
            for (int i = 0; i < 32; i += 2) tmax = max3(tmax, v[i], v[i + 1]);
          }
          const float new_m = fmaxf(run_m, tmax * sl2);             // sl2 > 0: the max commutes with the scale
          const float rescale = ex2_approx(run_m - new_m);
          run_s *= rescale;
          run_u *= rescale;
          run_m = new_m;
          if (row_ok) p.stash_shift[static_cast<int64_t>(row_local) * p.shift_pitch + n_tile] = new_m;
        }
#pragma unroll 1
        for (int c = 0; c < BN / 32; ++c) {
          const int cbase = col_tile + c * 32;
          if (cbase >= p.n_total) break;                          // warp-uniform
          float v[32];
          tmem_ld32(t_addr + c * 32, v);
          tmem_ld_wait();
          const int nvalid = p.n_total - cbase;                   // >= 1; columns >= nvalid are padding

          if constexpr (is_lse(EPI)) {
            // z2 = v s log2(e) is never formed on its own: the running maximum is taken over the raw accumulator
            // (the scale is positive) and every exponent is ONE fused multiply-add, 2^(v s log2e - m), issued two
            // logits per instruction (FFMA2 / FADD2 / FMNMX3).  Padding columns hold -inf: 2^-inf = 0.
            if (nvalid < 32) {
#pragma unroll
              for (int i = 0; i < 32; ++i) v[i] = i < nvalid ? v[i] : -INFINITY;
            }
            float new_m = run_m;                                   // stash: the tile max is already in run_m
            if constexpr (EPI != EPI_LSE_STASH) {
              float cmax = v[0];
#pragma unroll
              for (int i = 1; i < 31; i += 2) cmax = max3(cmax, v[i], v[i + 1]);
              new_m = fmaxf(run_m, fmaxf(cmax, v[31]) * sl2);
            }
            const float rescale = ex2_approx(run_m - new_m);
            const f32x2 sc2 = pack2(sl2, sl2), nm2 = pack2(-new_m, -new_m);
            float e[32];
            f32x2 acc = pack2(0.f, 0.f);
#pragma unroll
            for (int i = 0; i < 32; i += 2) {
              float t0, t1;
              unpack2(fma2(pack2(v[i], v[i + 1]), sc2, nm2), t0, t1);
              e[i] = ex2_approx(t0);
              e[i + 1] = ex2_approx(t1);
              acc = add2(acc, pack2(e[i], e[i + 1]));
            }
            float s0, s1;
            unpack2(acc, s0, s1);
            const float s = s0 + s1;
            if (p.part_u != nullptr) {   // entropy = lse - sum_v p_v z_v: one more running sum, rescaled like run_s
              float uc = 0.f;
#pragma unroll
              for (int i = 0; i < 32; ++i) uc = fmaf(e[i], i < nvalid ? v[i] * sl2 : 0.f, uc);   // 0 * -inf is NaN
              run_u = (EPI == EPI_LSE_STASH ? run_u : run_u * rescale) + uc;
            }
            if constexpr (EPI == EPI_LSE_STASH) {
              if (row_ok) {
                __nv_bfloat16* dst = p.dz + static_cast<int64_t>(row_local) * p.dz_pitch + cbase;
#pragma unroll
                for (int g = 0; g < 2; ++g)
                  st_global_v8(dst + g * 16, pack_f16x2(e[g * 16 + 0], e[g * 16 + 1]), pack_f16x2(e[g * 16 + 2], e[g * 16 + 3]),
                               pack_f16x2(e[g * 16 + 4], e[g * 16 + 5]), pack_f16x2(e[g * 16 + 6], e[g * 16 + 7]),
                               pack_f16x2(e[g * 16 + 8], e[g * 16 + 9]), pack_f16x2(e[g * 16 + 10], e[g * 16 + 11]),
                               pack_f16x2(e[g * 16 + 12], e[g * 16 + 13]), pack_f16x2(e[g * 16 + 14], e[g * 16 + 15]));
              }
            }
            run_s = run_s * rescale + s;
            run_m = new_m;
            if (static_cast<uint32_t>(y - cbase) < 32u) {          // rare: target column in this chunk
              float zy = 0.f;
#pragma unroll
              for (int i = 0; i < 32; ++i) zy = (y - cbase == i) ? v[i] : zy;
              p.zy[row_g] = zy * sl;                               // natural units: s * z
            }
          } else if constexpr (EPI == EPI_DZ) {
            // dz = k (1[v = y] - p),  p = 2^(z s log2e - lse log2e)
            float dzv[32];
            const f32x2 sc2 = pack2(sl2, sl2), nl2 = pack2(-lse2, -lse2), nk2 = pack2(-kcoef, -kcoef);
#pragma unroll
            for (int i = 0; i < 32; i += 2) {
              float t0, t1;
              unpack2(fma2(pack2(v[i], v[i + 1]), sc2, nl2), t0, t1);
              unpack2(mul2(pack2(ex2_approx(t0), ex2_approx(t1)), nk2), dzv[i], dzv[i + 1]);
            }
            if (static_cast<uint32_t>(y - cbase) < 32u) {
#pragma unroll
              for (int i = 0; i < 32; ++i) dzv[i] = (y - cbase == i) ? dzv[i] + kcoef : dzv[i];
            }
            uint32_t pk[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) pk[j] = pack_bf16x2(dzv[2 * j], dzv[2 * j + 1]);
            if (row_ok) {
              __nv_bfloat16* dst = p.dz + static_cast<int64_t>(row_local) * p.dz_pitch + cbase;
              // 2 x 32-byte stores (STG.256): whole aligned sectors (the row pitch is a multiple of 128 bytes)
#pragma unroll
              for (int g = 0; g < 2; ++g)
                st_global_v8(dst + g * 16, pk[8 * g], pk[8 * g + 1], pk[8 * g + 2], pk[8 * g + 3], pk[8 * g + 4],
                             pk[8 * g + 5], pk[8 * g + 6], pk[8 * g + 7]);
            } else if (row_local < p.m_alloc) {
              // rows of the last walked tile beyond the (dynamic) row count: A6 reads them as the tail of its last
              // k block, so they must hold zeros, not what an earlier chunk left there
              __nv_bfloat16* dst = p.dz + static_cast<int64_t>(row_local) * p.dz_pitch + cbase;
#pragma unroll
              for (int g = 0; g < 2; ++g) st_global_v8(dst + g * 16, 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u);
            }
          } else if constexpr (EPI == EPI_STORE) {
            if (row_ok) {   // fp32 partial tile of the unit's K range (A5; the test hook's plain product)
              float* dst = reinterpret_cast<float*>(p.c_out) + un.part * p.c_split_stride +
                           static_cast<int64_t>(row_local) * p.c_pitch + cbase;
              // 32-byte stores: the pitch keeps them aligned (c_pitch % 8 == 0) and nvalid is a multiple of 8
#pragma unroll
              for (int g = 0; g < 4; ++g)
                if (g * 8 < nvalid)
                  st_global_v8(dst + g * 8, __float_as_uint(v[g * 8]), __float_as_uint(v[g * 8 + 1]),
                               __float_as_uint(v[g * 8 + 2]), __float_as_uint(v[g * 8 + 3]), __float_as_uint(v[g * 8 + 4]),
                               __float_as_uint(v[g * 8 + 5]), __float_as_uint(v[g * 8 + 6]), __float_as_uint(v[g * 8 + 7]));
            }
          } else {  // EPI_RED_F32: C += acc.  The warp's 32 x 32 fp32 block goes through shared memory (128B-swizzled,
            // conflict-free 16-byte stores) and ONE TMA reduce-add: whole 128-byte lines are reduced at L2 instead
            // of 256 scattered 16-byte red.global per block, rows / columns out of range are clipped by the TMA
            // unit, and launches on other streams may accumulate into the same dW concurrently (atomic at L2).
            const uint32_t red_buf = tiles_addr + kStages * kStageBytes + quad * 4096;
            if (lane == 0) tma_store_wait_read<0>();            // the previous block has been read out of red_buf
            __syncwarp();
#pragma unroll
            for (int j = 0; j < 8; ++j)
              st_shared_v4_f32(red_buf + lane * 128 + ((j ^ (lane & 7)) << 4), v[4 * j], v[4 * j + 1], v[4 * j + 2],
                               v[4 * j + 3]);
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) {
              tma_reduce_add_2d(&tmC, red_buf, cbase, (m_tile * CG + static_cast<int>(cta_rank)) * BM + quad * 32, pol_c);
              tma_store_commit();
            }
          }
        }
        // all of this warp's TMEM reads of the accumulator are done: hand it back to the MMA warp
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          if constexpr (CG == 2) mbar_arrive_cluster(&bars->tmem_empty[acc], 0);   // the leader's barrier
          else mbar_arrive(&bars->tmem_empty[acc]);
        }
        acc ^= 1;
        if (acc == 0) acc_phase ^= 1;
      }

      if constexpr (EPI == EPI_RED_F32) {
        if (lane == 0) tma_store_wait<0>();                     // this unit's reductions are complete
      }
      if constexpr (is_lse(EPI)) {
        if (row_ok) {
          const int split = un.part;
          p.part_m[split * p.part_stride + row_local] = run_m;     // partials are indexed by the launch's own rows
          p.part_s[split * p.part_stride + row_local] = run_s;
          if (p.part_u != nullptr) p.part_u[split * p.part_stride + row_local] = run_u;
        }
      }
    }
  }

  // pair teardown: no CTA may exit (or free TMEM) while its peer can still signal its barriers or
  // the leader's MMAs can still read its shared memory
  tc_fence_before();
  if constexpr (CG == 2) cluster_sync_all(); else __syncthreads();
  if (warp == kMmaWarp) {
    tc_fence_after();
    tmem_dealloc<CG>(tmem_base, kTmemCols);
  }
}

}  // namespace grpo
