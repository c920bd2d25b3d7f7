// C ABI (include/grpo.h) of the fused GRPO policy-loss step: context, workspace, launch logic, CGP FIFO.
// Every step of the path runs in the kernels of this directory; there is no CPU or library fallback.
#include "../../include/grpo.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <deque>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "cgp_queue.h"
#include "gemm_sm100.cuh"
#include "token_kernels.cuh"

using namespace grpo;

// ------------------------------------------------------------------------------------- errors
static thread_local char g_err[512] = "";
static int32_t fail(int32_t code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}
// for the other translation units of the library (stitched_memory.cpp)
int32_t grpo_internal_fail(int32_t code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}
#define CU_OK(expr)                                                                                   \
  do {                                                                                                \
    cudaError_t e__ = (expr);                                                                         \
    if (e__ != cudaSuccess)                                                                           \
      return fail(GRPO_ERR_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
  } while (0)
#define GRPO_TRY(expr)                  \
  do {                                  \
    int32_t s__ = (expr);               \
    if (s__ != GRPO_OK) return s__;     \
  } while (0)

// ------------------------------------------------------------------------------------- context
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static inline int64_t align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

struct SlotLayout {
  int64_t part_cap = 0;   // floats per partial array
  int64_t s_max = 0;
  int64_t chunk_rows = 0;
  int64_t v_pad = 0;
  int64_t off_part_u = 0, off_shift = 0;
  int64_t n_vtiles = 0;   // 256-column vocab tiles (pitch of the stash shift array)
  int64_t off_part_m = 0, off_part_s = 0, off_zy = 0, off_total = 0, off_seq_count = 0, off_dz = 0;
  int64_t off_hidden = 0, off_targets = 0, off_old = 0, off_ref = 0, off_mask = 0, off_rewards = 0, off_adv = 0,
          off_cu_seq = 0, off_cu_grp = 0, off_logp = 0, off_lse = 0, off_coeff = 0, off_dh = 0, off_sync = 0,
          off_dz2 = 0;
  // token-granular compaction + split-K of A5
  int64_t off_row_idx = 0, off_meta = 0, off_hc = 0, off_yc = 0, off_lsec = 0, off_coeffc = 0, off_dh_part = 0,
          off_row_stats = 0;
  int64_t n_chunks_max = 0;
  int64_t fwd_block_rows = 0;   // rows per A2 launch (bounds the LSE partials)
  int64_t off_loss_part = 0, off_loss_count = 0;                  // A3: per-block partial sums, arrival counter
  int64_t off_w8 = 0, off_h8 = 0, off_hscale = 0, off_wscale = 0;   // FP8 study (cfg.fp8_logits)
  int64_t bytes = 0;
};

struct PendingGroup {
  grpo_group_desc desc;
  std::vector<int32_t> seqlens;
  int64_t tokens;
};

struct grpo_ctx {
  grpo_config cfg;
  int device = 0;
  int num_sms = 0;
  int cg = 2;                    // CTAs per MMA: 1 (cta_group::1) or 2 (CTA pairs, cta_group::2)
  EncodeTiledFn encode = nullptr;
  int32_t* err_dev = nullptr;
  float* denom_ring = nullptr;   // device scalars for implicit per-update denominators
  int denom_next = 0;
  cudaEvent_t denom_event = nullptr;
  float* entropy_out = nullptr;         // grpo_set_entropy_out: per-token entropy of the direct forward calls
  int32_t seq_denom = 0;                // grpo_set_seq_denom: sequences of the whole logical update (loss_agg 1)
  cudaStream_t copy_stream = nullptr;   // grpo_step_host: H2D / D2H overlapped with the compute stream
  std::vector<cudaEvent_t> pipe_events; // grpo_step_host: fence + per-chunk in / out events, created once
  // pinned staging ring for the small host-built index arrays of run_launch (cu_seqlens, cu_groups)
  static const int kStageRing = 8;
  int32_t* stage_host = nullptr;
  int64_t stage_ints = 0;               // ints per ring entry
  cudaEvent_t stage_ev[kStageRing] = {nullptr};
  int stage_next = 0;
  std::vector<cudaEvent_t> event_pool;  // timing events of the profiler, reused across launches
  uint8_t* ws = nullptr;
  int64_t ws_max_T = 0;
  int n_slots = 0;
  SlotLayout lay;
  std::deque<PendingGroup> fifo;
  int64_t launches = 0;
  int32_t consumed = 0;
  bool update_broken = false;    // a launch failed after part of its update was enqueued (see drain_one_update)
  // kernel accounting (always) and per-launch CUDA-event timing (only while profiling is on)
  int64_t kernel_count[GRPO_NUM_KERNEL_KINDS] = {0};
  bool profiling = false;
  struct ProfRec { int kind; cudaEvent_t beg, end; };
  std::vector<ProfRec> prof;
};

// Brackets one kernel launch: counts it and, while profiling, records events on the launch stream.
struct LaunchScope {
  grpo_ctx* ctx; cudaStream_t st; cudaEvent_t end = nullptr;
  LaunchScope(grpo_ctx* c, int kind, cudaStream_t s) : ctx(c), st(s) {
    ctx->kernel_count[kind]++;
    if (ctx->profiling) {
      grpo_ctx::ProfRec r{kind, take_event(c), take_event(c)};
      if (r.beg && r.end) {
        cudaEventRecord(r.beg, st);
        end = r.end;
        ctx->prof.push_back(r);
      }
    }
  }
  ~LaunchScope() { if (end) cudaEventRecord(end, st); }
  static cudaEvent_t take_event(grpo_ctx* c) {     // from the context's pool; created only when the pool is empty
    cudaEvent_t e = nullptr;
    if (!c->event_pool.empty()) { e = c->event_pool.back(); c->event_pool.pop_back(); return e; }
    return cudaEventCreate(&e) == cudaSuccess ? e : nullptr;
  }
};
static const int kDenomRing = 64;
static void prof_clear(grpo_ctx* ctx) {             // records go back to the pool
  for (auto& r : ctx->prof) { ctx->event_pool.push_back(r.beg); ctx->event_pool.push_back(r.end); }
  ctx->prof.clear();
}


static const int kSyncCap = 1 << 15;   // drift-gate epoch counters per workspace slot
static int64_t chunk_tokens(const grpo_config& c) { return c.bwd_chunk_tokens > 0 ? c.bwd_chunk_tokens : 9472; }

// The vocab split of the A2 units and the K split of A5 are functions of V (and the tile shape) ALONE: a token's
// log-sum-exp and dHidden row are then summed in one fixed order whatever launch, chunk or batch the token is part
// of (batch invariance: CGP changes "only group dispatch timing and order - not samples, advantages, or gradient
// computation").  Load balance comes from the ORDER the units are walked in, never from re-cutting
// a reduction.
// L2 working-set bounds of the unit orders (gemm_sm100.cuh: n_group / m_block / lse_block; results never depend on
// them).  Chosen so that d = 2048 walks its units exactly as it always has and wider models keep a comparable L2
// footprint.  DRAM reads per launch at d = 4096, T = 16-19k: A2 68 GB without a bound, 28 GB with 80 MB blocks, 10 with
// 56 MB, 8 with 40 MB (algorithmic 1.4; step time best at 56 MB); A4 10 GB -> 4; A6 18 GB -> 12.
static const int64_t kA2AllBytes = 80ll << 20;     // A2: every pair its own token tile while their rows fit in this ...
static const int64_t kA2BlockBytes = 56ll << 20;   // ... else blocks of token tiles of this many bytes of hidden state
static const int64_t kA4BlockBytes = 40ll << 20;   // A4 blocks (A4 also streams the dZ chunk out through L2)
static const int kNGroupTiles = 8;                 // A5 / A6: d tiles (256 columns) walked together (2048 columns)
static const int kLseTilesPerSplit = 8;      // 256-column vocab tiles per A2 unit (2048 logits)
static const int kDhKSplit = 4;              // K ranges of A5 (K = V)
static void lse_split(int V, int* n_split, int* tiles_per_split) {
  const int n_tiles = (V + BN - 1) / BN;
  *n_split = (n_tiles + kLseTilesPerSplit - 1) / kLseTilesPerSplit;
  *tiles_per_split = (n_tiles + *n_split - 1) / *n_split;
  *n_split = (n_tiles + *tiles_per_split - 1) / *tiles_per_split;
}
static void dh_ksplit(int V, int* k_split, int* kb_per_split) {
  const int k_blocks = (V + BK - 1) / BK;
  const int want = std::min(kDhKSplit, k_blocks);
  *kb_per_split = (k_blocks + want - 1) / want;
  *k_split = (k_blocks + *kb_per_split - 1) / *kb_per_split;
}

static SlotLayout make_layout(const grpo_config& c, int64_t max_T) {
  SlotLayout L;
  int64_t off = 0;
  auto take = [&](int64_t bytes) {
    int64_t o = off;
    off = align_up(off + bytes, 256);
    return o;
  };
  int n_split, tps, k_split, kbps;
  lse_split(c.V, &n_split, &tps);
  dh_ksplit(c.V, &k_split, &kbps);
  L.s_max = std::min<int64_t>(max_T, 1 << 20);
  L.chunk_rows = std::min<int64_t>(align_up(chunk_tokens(c), 256), align_up(max_T, 256));
  L.fwd_block_rows = std::min<int64_t>(align_up(max_T, 256), 4 * 74 * 256);
  L.part_cap = n_split * L.fwd_block_rows;
  L.v_pad = align_up(c.V, 64);
  L.off_part_m = take(L.part_cap * 4);
  L.off_part_s = take(L.part_cap * 4);
  L.off_part_u = take(L.part_cap * 4);
  L.off_zy = take(max_T * 4);
  L.off_total = take(256);
  L.off_seq_count = take(L.s_max * 4);
  L.off_dz = take(L.chunk_rows * L.v_pad * 2);
  L.n_vtiles = (c.V + BN - 1) / BN;
  L.off_shift = take(L.chunk_rows * L.n_vtiles * 4);
  L.off_hidden = take(max_T * c.d * 2);
  L.off_targets = take(max_T * 4);
  L.off_old = take(max_T * 4);
  L.off_ref = take(max_T * 4);
  L.off_mask = take(max_T);
  L.off_rewards = take(L.s_max * 4);
  L.off_adv = take(L.s_max * 4);
  L.off_cu_seq = take((L.s_max + 1) * 4);
  L.off_cu_grp = take((L.s_max + 1) * 4);
  L.off_logp = take(max_T * 4);
  L.off_lse = take(max_T * 4);
  L.off_coeff = take(max_T * 4);
  L.off_dh = take(max_T * c.d * (c.dhidden_fp32 ? 4 : 2));
  L.off_sync = take(kSyncCap * 4);
  L.off_dz2 = take(L.chunk_rows * L.v_pad * 2);   // 3-contraction variant: compacted dZ rows of a chunk
  L.n_chunks_max = (max_T + L.chunk_rows - 1) / L.chunk_rows + 1;
  L.off_row_idx = take(max_T * 4);
  L.off_meta = take(4 * (L.n_chunks_max + 1) * 4);
  L.off_hc = take(L.chunk_rows * c.d * 2);
  L.off_yc = take(L.chunk_rows * 4);
  L.off_lsec = take(L.chunk_rows * 4);
  L.off_coeffc = take(L.chunk_rows * 4);
  L.off_dh_part = take(static_cast<int64_t>(k_split) * L.chunk_rows * c.d * 4);
  L.off_row_stats = take(16);
  L.off_loss_part = take(((max_T + 255) / 256 + 1) * 5 * 4);
  L.off_loss_count = take(16);
  if (c.fp8_logits) {
    L.off_w8 = take(static_cast<int64_t>(c.V) * c.d);
    L.off_h8 = take(std::max(L.fwd_block_rows, L.chunk_rows) * c.d);
    L.off_hscale = take(max_T * 4 + 1024);
    L.off_wscale = take(256);
  }
  L.bytes = off;
  return L;
}

template <typename T>
static T* slot_ptr(const grpo_ctx* ctx, int slot, int64_t off) {
  return reinterpret_cast<T*>(ctx->ws + static_cast<int64_t>(slot) * ctx->lay.bytes + off);
}

// ------------------------------------------------------------------------------------- TMA maps
// 2-D bf16 tensor, `inner` contiguous elements per row, `outer` rows, row pitch in bytes; 128B swizzle;
// out-of-bounds elements of a box read as zero (this is what makes ragged M/N/K tails work).
static int32_t make_tmap(const grpo_ctx* ctx, CUtensorMap* m, const void* base, uint64_t inner, uint64_t outer,
                         uint64_t pitch_bytes, uint32_t box_inner, uint32_t box_outer) {
  if ((reinterpret_cast<uintptr_t>(base) & 15) != 0 || (pitch_bytes & 15) != 0)
    return fail(GRPO_ERR_SHAPE, "tensor base/pitch not 16-byte aligned (base %p pitch %llu)", base,
                (unsigned long long)pitch_bytes);
  cuuint64_t dims[2] = {inner, outer};
  cuuint64_t strides[1] = {pitch_bytes};
  cuuint32_t box[2] = {box_inner, box_outer};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = ctx->encode(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(GRPO_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
  return GRPO_OK;
}

// e4m3 operand (FP8 study): 2-D byte tensor, 128-byte k blocks, 128B swizzle.
static int32_t make_tmap_u8(const grpo_ctx* ctx, CUtensorMap* m, const void* base, uint64_t inner, uint64_t outer,
                            uint64_t pitch_bytes, uint32_t box_outer) {
  if ((reinterpret_cast<uintptr_t>(base) & 15) != 0 || (pitch_bytes & 15) != 0)
    return fail(GRPO_ERR_SHAPE, "e4m3 tensor base/pitch not 16-byte aligned (need d %% 16 == 0)");
  cuuint64_t dims[2] = {inner, outer};
  cuuint64_t strides[1] = {pitch_bytes};
  cuuint32_t box[2] = {128, box_outer};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = ctx->encode(m, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(GRPO_ERR_CUDA, "cuTensorMapEncodeTiled (u8) failed with CUresult %d", (int)r);
  return GRPO_OK;
}

// fp32 C tensor [outer, inner] for the A6 epilogue's TMA reduce-add: 32 x 32 boxes (128-byte rows), 128B swizzle.
static int32_t make_tmap_c_f32(const grpo_ctx* ctx, CUtensorMap* m, const void* base, uint64_t inner, uint64_t outer,
                               uint64_t pitch_bytes) {
  if ((reinterpret_cast<uintptr_t>(base) & 15) != 0 || (pitch_bytes & 15) != 0)
    return fail(GRPO_ERR_SHAPE, "dW base/pitch not 16-byte aligned (base %p pitch %llu)", base,
                (unsigned long long)pitch_bytes);
  cuuint64_t dims[2] = {inner, outer};
  cuuint64_t strides[1] = {pitch_bytes};
  cuuint32_t box[2] = {32, 32};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = ctx->encode(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                           CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(GRPO_ERR_CUDA, "cuTensorMapEncodeTiled (fp32 C) failed with CUresult %d", (int)r);
  return GRPO_OK;
}


template <int CG, bool A_MN, bool B_MN, int EPI, int DT = 0>
static int32_t launch_gemm_cg(grpo_ctx* ctx, int kind, const CUtensorMap& tmA, const CUtensorMap& tmB,
                              const GemmParams& p, int n_units, cudaStream_t st, const CUtensorMap* tmC) {
  // the dynamic shared memory limit is a per-device attribute of the function: one flag bit per device and
  // template instantiation (setting it twice is harmless, so a relaxed atomic is enough)
  static std::atomic<uint64_t> attr_set{0};
  auto kern = grpo_gemm_kernel<CG, A_MN, B_MN, EPI, DT>;
  constexpr int smem = GemmShape<CG, EPI>::kSmemBytes;
  const uint64_t dev_bit = 1ull << (ctx->device & 63);
  if (ctx->device >= 64 || !(attr_set.load(std::memory_order_relaxed) & dev_bit)) {
    CU_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    if (ctx->device < 64) attr_set.fetch_or(dev_bit, std::memory_order_relaxed);
  }
  if (n_units <= 0) return GRPO_OK;
  // persistent: one CTA (CG = 1) or one CTA pair (CG = 2, a 2-CTA cluster) per SM / SM pair
  // (gemm_max_ctas leaves SMs to a concurrent kernel; the unit -> reduction-range map never depends on the grid)
  const int ctas = ctx->cfg.gemm_max_ctas > 0 ? std::min(ctx->cfg.gemm_max_ctas, ctx->num_sms) : ctx->num_sms;
  const int grid = CG * std::min(n_units, std::max(ctas / CG, 1));
  GemmParams pl = p;
  // A2 walks its units in blocks of lse_block token tiles whose hidden-state rows stay L2-resident while W streams:
  // every pair of the grid gets its own token tile as long as those rows fit (80 MB: 74 tiles at d = 2048)
  const int64_t m_tile_bytes = static_cast<int64_t>(BM) * CG * ctx->cfg.d * 2;
  pl.lse_block = grid / CG;
  if (pl.lse_block * m_tile_bytes > kA2AllBytes)
    pl.lse_block = static_cast<int>(std::max<int64_t>(1, kA2BlockBytes / m_tile_bytes));
  // drift gate (gemm_sm100.cuh): epoch counters live in the launch's workspace slot, zeroed on the stream
  const int xsync = ctx->cfg.gemm_drift_epoch_kb == 0 ? 32 : ctx->cfg.gemm_drift_epoch_kb;
  pl.sync_lag = 1;   // epochs a pair may lead the slowest pair by (2-8 measured: no different from 1)
  if (pl.sync != nullptr && xsync > 0 && grid / CG > 1) {
    const int64_t n_pairs = grid / CG;
    const int64_t kb_unit = is_lse(EPI) ? static_cast<int64_t>(p.k_blocks) * p.tiles_per_split
                                        : (p.k_split > 1 ? p.kb_per_split : p.k_blocks);
    const int64_t max_kb = (n_units + n_pairs - 1) / n_pairs * kb_unit;
    int64_t E = xsync;
    while ((max_kb + E - 1) / E + 1 > kSyncCap) E *= 2;
    pl.sync_epoch_kb = static_cast<int>(E);
    pl.sync_epochs = static_cast<int>((max_kb + E - 1) / E + 1);
    CU_OK(cudaMemsetAsync(pl.sync, 0, static_cast<size_t>(pl.sync_epochs) * 4, st));
  } else {
    pl.sync = nullptr;
  }
  cudaLaunchConfig_t lc;
  std::memset(&lc, 0, sizeof(lc));
  lc.gridDim = dim3(grid);
  lc.blockDim = dim3(kGemmThreads);
  lc.dynamicSmemBytes = smem;
  lc.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = CG;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  lc.attrs = attr;
  lc.numAttrs = 1;
  {
    LaunchScope ls(ctx, kind, st);
    CU_OK(cudaLaunchKernelEx(&lc, kern, tmA, tmB, tmC ? *tmC : tmA, pl, n_units));
  }
  CU_OK(cudaGetLastError());
  return GRPO_OK;
}

template <bool A_MN, bool B_MN, int EPI, int DT = 0>
static int32_t launch_gemm(grpo_ctx* ctx, int kind, const CUtensorMap& tmA, const CUtensorMap& tmB, const GemmParams& p,
                           int n_units, cudaStream_t st, const CUtensorMap* tmC = nullptr) {
  if (EPI == EPI_RED_F32 && tmC == nullptr) return fail(GRPO_ERR_INVALID_ARG, "EPI_RED_F32 needs the C tensor map");
  if (ctx->cg == 2) return launch_gemm_cg<2, A_MN, B_MN, EPI, DT>(ctx, kind, tmA, tmB, p, n_units, st, tmC);
  return launch_gemm_cg<1, A_MN, B_MN, EPI, DT>(ctx, kind, tmA, tmB, p, n_units, st, tmC);
}

// FP8 study: quantise `rows` bf16 rows of width d to e4m3 (per-row scales, or the tensor's scale `fixed`).
static int32_t quantize_rows(grpo_ctx* ctx, const void* x, int64_t rows, void* q, float* scales, const float* fixed,
                             cudaStream_t st) {
  if (rows <= 0) return GRPO_OK;
  const int64_t blocks = std::min<int64_t>((rows + 7) / 8, 32LL * ctx->num_sms);
  {
    LaunchScope ls(ctx, GRPO_KERNEL_QUANTIZE, st);
    quantize_rows_e4m3_kernel<<<static_cast<unsigned>(blocks), 256, 0, st>>>(
        static_cast<const uint2*>(x), rows, ctx->cfg.d / 4, static_cast<uint32_t*>(q), scales, fixed);
  }
  CU_OK(cudaGetLastError());
  return GRPO_OK;
}
// ... and the vocab matrix with ONE scale (amax / 448) into the slot's W8 buffer.
static int32_t quantize_weights(grpo_ctx* ctx, int slot, const void* W, cudaStream_t st) {
  const grpo_config& c = ctx->cfg;
  float* wscale = slot_ptr<float>(ctx, slot, ctx->lay.off_wscale);
  unsigned int* amax = reinterpret_cast<unsigned int*>(wscale) + 1;
  CU_OK(cudaMemsetAsync(amax, 0, 4, st));
  {
    LaunchScope ls(ctx, GRPO_KERNEL_QUANTIZE, st);
    amax_kernel<<<8 * ctx->num_sms, 256, 0, st>>>(static_cast<const uint2*>(W), static_cast<int64_t>(c.V) * c.d / 4, amax);
  }
  {
    LaunchScope ls(ctx, GRPO_KERNEL_QUANTIZE, st);
    scale_from_amax_kernel<<<1, 1, 0, st>>>(amax, wscale);
  }
  CU_OK(cudaGetLastError());
  return quantize_rows(ctx, W, c.V, slot_ptr<uint8_t>(ctx, slot, ctx->lay.off_w8), nullptr, wscale, st);
}

// ------------------------------------------------------------------------------------- API: misc
extern "C" const char* grpo_last_error(void) { return g_err; }

extern "C" int32_t grpo_default_config(grpo_config* cfg) {
  if (!cfg) return fail(GRPO_ERR_INVALID_ARG, "cfg is NULL");
  std::memset(cfg, 0, sizeof(*cfg));
  cfg->eps_std = 1e-6f;
  cfg->clip_lo = 0.2f;
  cfg->clip_hi = 0.28f;
  cfg->logit_scale = 1.0f;
  cfg->groups_per_update = 1;
  cfg->bwd_chunk_tokens = 9472;
  cfg->max_pending_groups = 4096;
  return GRPO_OK;
}

extern "C" int32_t grpo_create(const grpo_config* cfg, grpo_ctx** out) {
  if (!cfg || !out) return fail(GRPO_ERR_INVALID_ARG, "cfg/out is NULL");
  if (cfg->d <= 0 || cfg->V <= 0 || cfg->d % 8 != 0)
    return fail(GRPO_ERR_SHAPE, "need d > 0, d %% 8 == 0, V > 0 (got d=%d V=%d)", cfg->d, cfg->V);
  if (cfg->gemm_cta_group < 0 || cfg->gemm_cta_group > 2)
    return fail(GRPO_ERR_INVALID_ARG, "gemm_cta_group must be 0 (default), 1 or 2");
  if (cfg->groups_per_update < 1 || cfg->std_ddof < 0 || cfg->std_ddof > 1 || cfg->loss_agg < 0 || cfg->loss_agg > 1)
    return fail(GRPO_ERR_INVALID_ARG, "bad groups_per_update / std_ddof / loss_agg");
  if (cfg->fp8_logits != 0 && (cfg->stash_logits != 0 || cfg->d % 16 != 0))
    return fail(GRPO_ERR_INVALID_ARG, "fp8_logits needs d %% 16 == 0 and is not available with stash_logits");
  if (!(cfg->logit_scale > 0.f))
    return fail(GRPO_ERR_INVALID_ARG, "logit_scale (1 / temperature) must be > 0 (got %g)", (double)cfg->logit_scale);
  if (cfg->gemm_max_ctas < 0) return fail(GRPO_ERR_INVALID_ARG, "gemm_max_ctas must be >= 0");
  if (cfg->kl_type < 0 || cfg->kl_type > 2 || (cfg->dual_clip != 0.f && !(cfg->dual_clip > 1.f)))
    return fail(GRPO_ERR_INVALID_ARG, "kl_type must be 0, 1 or 2 and dual_clip 0 or > 1");
  int dev = 0;
  CU_OK(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  CU_OK(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10)
    return fail(GRPO_ERR_ARCH, "device %d is sm_%d%d; this library is built for sm_100a only", dev, prop.major,
                prop.minor);
  grpo_ctx* ctx = new (std::nothrow) grpo_ctx();
  if (!ctx) return fail(GRPO_ERR_INVALID_ARG, "out of host memory");
  ctx->cfg = *cfg;
  if (ctx->cfg.max_pending_groups <= 0) ctx->cfg.max_pending_groups = 4096;
  ctx->device = dev;
  ctx->num_sms = prop.multiProcessorCount;
  ctx->cg = cfg->gemm_cta_group == 1 ? 1 : 2;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
    delete ctx;
    return fail(GRPO_ERR_CUDA, "cuTensorMapEncodeTiled entry point not available");
  }
  ctx->encode = reinterpret_cast<EncodeTiledFn>(fn);
  if (cudaMalloc(&ctx->err_dev, 256) != cudaSuccess || cudaMalloc(&ctx->denom_ring, kDenomRing * 4) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->denom_event, cudaEventDisableTiming) != cudaSuccess ||
      cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking) != cudaSuccess) {
    delete ctx;
    return fail(GRPO_ERR_CUDA, "context allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
  }
  CU_OK(cudaMemset(ctx->err_dev, 0, 256));
  *out = ctx;
  return GRPO_OK;
}

extern "C" int32_t grpo_destroy(grpo_ctx* ctx) {
  if (!ctx) return GRPO_OK;
  cudaFree(ctx->err_dev);
  cudaFree(ctx->denom_ring);
  prof_clear(ctx);
  for (auto e : ctx->event_pool) cudaEventDestroy(e);
  for (auto e : ctx->pipe_events) cudaEventDestroy(e);
  for (auto e : ctx->stage_ev) if (e) cudaEventDestroy(e);
  if (ctx->stage_host) cudaFreeHost(ctx->stage_host);
  if (ctx->denom_event) cudaEventDestroy(ctx->denom_event);
  if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
  delete ctx;
  return GRPO_OK;
}

extern "C" int32_t grpo_workspace_bytes(const grpo_ctx* ctx, int64_t max_T, int64_t* bytes_out) {
  if (!ctx || !bytes_out || max_T <= 0) return fail(GRPO_ERR_INVALID_ARG, "bad ctx / max_T / bytes_out");
  *bytes_out = make_layout(ctx->cfg, max_T).bytes;
  return GRPO_OK;
}

extern "C" int32_t grpo_set_workspace(grpo_ctx* ctx, void* dev_ptr, int64_t bytes, int64_t max_T, int32_t n_slots) {
  if (!ctx || !dev_ptr || max_T <= 0 || n_slots < 1) return fail(GRPO_ERR_INVALID_ARG, "bad workspace arguments");
  if (reinterpret_cast<uintptr_t>(dev_ptr) & 255) return fail(GRPO_ERR_WORKSPACE, "workspace must be 256-byte aligned");
  SlotLayout L = make_layout(ctx->cfg, max_T);
  if (bytes < L.bytes * n_slots)
    return fail(GRPO_ERR_WORKSPACE, "workspace too small: %lld < %d x %lld", (long long)bytes, n_slots,
                (long long)L.bytes);
  ctx->ws = static_cast<uint8_t*>(dev_ptr);
  ctx->ws_max_T = max_T;
  ctx->n_slots = n_slots;
  ctx->lay = L;
  for (int i = 0; i < n_slots; ++i) {
    CU_OK(cudaMemset(slot_ptr<int>(ctx, i, L.off_row_stats), 0, 16));
    CU_OK(cudaMemset(slot_ptr<int>(ctx, i, L.off_loss_count), 0, 16));
  }
  // pinned ring for run_launch's index arrays: cu_seqlens [S+1] + cu_groups [S+1] per entry
  const int64_t need = 2 * (L.s_max + 1);
  if (need > ctx->stage_ints) {
    CU_OK(cudaDeviceSynchronize());
    if (ctx->stage_host) cudaFreeHost(ctx->stage_host);
    ctx->stage_host = nullptr;
    CU_OK(cudaMallocHost(&ctx->stage_host, static_cast<size_t>(need) * grpo_ctx::kStageRing * 4));
    ctx->stage_ints = need;
    for (auto& e : ctx->stage_ev)
      if (!e) CU_OK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  }
  return GRPO_OK;
}

extern "C" int32_t grpo_check_errors_sync(grpo_ctx* ctx, int32_t* flags_out) {
  if (!ctx || !flags_out) return fail(GRPO_ERR_INVALID_ARG, "ctx/flags_out is NULL");
  CU_OK(cudaDeviceSynchronize());
  CU_OK(cudaMemcpy(flags_out, ctx->err_dev, 4, cudaMemcpyDeviceToHost));
  CU_OK(cudaMemset(ctx->err_dev, 0, 4));
  return GRPO_OK;
}

// ------------------------------------------------------------------------------------- accounting / profiling
extern "C" int32_t grpo_kernel_launches(const grpo_ctx* ctx, int64_t* counts_out) {
  if (!ctx || !counts_out) return fail(GRPO_ERR_INVALID_ARG, "ctx/counts_out is NULL");
  for (int i = 0; i < GRPO_NUM_KERNEL_KINDS; ++i) counts_out[i] = ctx->kernel_count[i];
  return GRPO_OK;
}

extern "C" int32_t grpo_profile_enable(grpo_ctx* ctx, int32_t on) {
  if (!ctx) return fail(GRPO_ERR_INVALID_ARG, "ctx is NULL");
  ctx->profiling = on != 0;
  if (!on) prof_clear(ctx);
  return GRPO_OK;
}

extern "C" int32_t grpo_profile_read_sync(grpo_ctx* ctx, double* ms_out, int64_t* launches_out) {
  if (!ctx || !ms_out || !launches_out) return fail(GRPO_ERR_INVALID_ARG, "NULL pointer");
  CU_OK(cudaDeviceSynchronize());
  for (int i = 0; i < GRPO_NUM_KERNEL_KINDS; ++i) { ms_out[i] = 0.0; launches_out[i] = 0; }
  for (auto& r : ctx->prof) {
    float ms = 0.f;
    CU_OK(cudaEventElapsedTime(&ms, r.beg, r.end));
    ms_out[r.kind] += ms;
    launches_out[r.kind]++;
  }
  prof_clear(ctx);
  return GRPO_OK;
}

extern "C" int32_t grpo_bwd_row_stats_sync(grpo_ctx* ctx, int64_t* active_out, int64_t* total_out) {
  if (!ctx || !active_out || !total_out) return fail(GRPO_ERR_INVALID_ARG, "NULL pointer");
  *active_out = *total_out = 0;
  if (!ctx->ws) return GRPO_OK;
  CU_OK(cudaDeviceSynchronize());
  for (int i = 0; i < ctx->n_slots; ++i) {
    long long h[2] = {0, 0};
    long long* stats = slot_ptr<long long>(ctx, i, ctx->lay.off_row_stats);
    CU_OK(cudaMemcpy(h, stats, 16, cudaMemcpyDeviceToHost));
    CU_OK(cudaMemset(stats, 0, 16));
    *active_out += h[0];
    *total_out += h[1];
  }
  return GRPO_OK;
}

// ------------------------------------------------------------------------------------- A1
extern "C" int32_t grpo_group_advantage(grpo_ctx* ctx, const float* rewards, const int32_t* cu_groups,
                                        int32_t n_groups, int32_t G, float* adv_out, uint8_t* zero_var_out,
                                        void* stream) {
  if (!ctx || !rewards || !adv_out) return fail(GRPO_ERR_INVALID_ARG, "ctx/rewards/adv_out is NULL");
  if (n_groups < 0 || (!cu_groups && G <= 0)) return fail(GRPO_ERR_INVALID_ARG, "need n_groups >= 0 and G > 0 or cu_groups");
  if (n_groups == 0) return GRPO_OK;
  const int threads = 128;
  const int blocks = (n_groups * 32 + threads - 1) / threads;
  {
    LaunchScope ls(ctx, GRPO_KERNEL_ADVANTAGE, static_cast<cudaStream_t>(stream));
    group_advantage_kernel<<<blocks, threads, 0, static_cast<cudaStream_t>(stream)>>>(
        rewards, cu_groups, n_groups, G, ctx->cfg.eps_std, ctx->cfg.std_ddof, adv_out, zero_var_out);
  }
  CU_OK(cudaGetLastError());
  return GRPO_OK;
}

// ------------------------------------------------------------------------------------- A2 + A3
// Per-token inputs / outputs of the forward, all indexed by the packed row of the whole call.
struct FwdArgs {
  const int32_t* cu_seqlens; int32_t S;
  const float* adv; const float* old_logp; const float* ref_logp; const uint8_t* mask;
  double loss_denom; const float* denom_dev;
  float* logp_out; float* lse_out; float* coeff_out; float* loss_accum; float* metrics_accum;
  float* entropy_out = nullptr;   // nullable (grpo_set_entropy_out)
  int32_t S_norm = 0;             // loss_agg 1: sequences of the WHOLE logical update (0: this call's S)
  int64_t T_call = 0;             // packed tokens of the call (bounds the fp32 token count of an implicit denominator)
};

// The loss-bearing token count behind an IMPLICIT token-mean denominator is accumulated in fp32 on the device, which
// is exact up to 2^24 tokens; larger calls must state loss_denom (include/grpo.h).
static const int64_t kMaxCountedTokens = int64_t(1) << 24;

static int32_t fwd_check(grpo_ctx* ctx, int32_t S, int64_t T) {
  if (!ctx->ws) return fail(GRPO_ERR_WORKSPACE, "no workspace set (grpo_set_workspace)");
  if (T > ctx->ws_max_T) return fail(GRPO_ERR_WORKSPACE, "T=%lld exceeds workspace max_T=%lld", (long long)T, (long long)ctx->ws_max_T);
  if (S > ctx->lay.s_max) return fail(GRPO_ERR_WORKSPACE, "S=%d exceeds workspace capacity", S);
  if (T > INT32_MAX - 256) return fail(GRPO_ERR_SHAPE, "T too large");
  return GRPO_OK;
}

// Loss-bearing token counts that define the mean (whole call, before any row is processed).
static int32_t fwd_counts(grpo_ctx* ctx, int slot, const int32_t* targets, const FwdArgs& a, cudaStream_t st,
                          int V = 0) {
  const grpo_config& c = ctx->cfg;
  if (V <= 0) V = c.V;
  const SlotLayout& L = ctx->lay;
  float* total = slot_ptr<float>(ctx, slot, L.off_total);
  float* seq_count = slot_ptr<float>(ctx, slot, L.off_seq_count);
  const bool implicit_denom = c.loss_agg == 0 && !(a.loss_denom > 0.0) && a.denom_dev == nullptr;
  if (implicit_denom && a.T_call > kMaxCountedTokens)
    return fail(GRPO_ERR_SHAPE, "T=%lld: the token-mean denominator is counted in fp32, exact only up to 2^24 tokens; "
                "pass loss_denom > 0 for a call this large", (long long)a.T_call);
  if (c.loss_agg == 1 || implicit_denom) {
    CU_OK(cudaMemsetAsync(total, 0, 4, st));
    const int threads = 128;
    const int blocks = (a.S * 32 + threads - 1) / threads;
    {
      LaunchScope ls(ctx, GRPO_KERNEL_TOKEN_COUNT, st);
      token_count_kernel<<<blocks, threads, 0, st>>>(a.mask, targets, V, a.cu_seqlens, a.S, seq_count, total);
    }
    CU_OK(cudaGetLastError());
  }
  return GRPO_OK;
}

// A2 alone over packed rows [t0, t0 + rows): the per-split (max, sum-exp) partials land in the slot's partial
// buffers ([n_split, rows], log2 domain), the target logit in zy[t] (rows whose target is not a column of W are
// left untouched).
static int32_t a2_rows(grpo_ctx* ctx, int slot, const void* hidden, const void* W, const int32_t* targets, float* zy,
                       bool entropy, int64_t t0, int64_t rows, __nv_bfloat16* stash, cudaStream_t st, int* n_split_out) {
  const grpo_config& c = ctx->cfg;
  const SlotLayout& L = ctx->lay;
  float* part_m = slot_ptr<float>(ctx, slot, L.off_part_m);
  float* part_s = slot_ptr<float>(ctx, slot, L.off_part_s);

  CUtensorMap tmH, tmW;
  const void* Hc = static_cast<const uint8_t*>(hidden) + t0 * c.d * 2;
  GRPO_TRY(make_tmap(ctx, &tmH, Hc, c.d, rows, static_cast<uint64_t>(c.d) * 2, BK, BM));
  const int TM = BM * ctx->cg;                      // rows of C per scheduling unit (CTA or CTA pair)
  GRPO_TRY(make_tmap(ctx, &tmW, W, c.d, c.V, static_cast<uint64_t>(c.d) * 2, BK, BN / ctx->cg));
  GemmParams p;
  std::memset(&p, 0, sizeof(p));
  p.m_total = static_cast<int>(rows);
  p.n_total = c.V;
  p.m_tiles = static_cast<int>((rows + TM - 1) / TM);
  p.n_tiles = (c.V + BN - 1) / BN;
  p.k_blocks = (c.d + BK - 1) / BK;
  lse_split(c.V, &p.n_split, &p.tiles_per_split);          // a function of V alone (batch invariance)
  if (static_cast<int64_t>(p.n_split) * rows > L.part_cap)
    return fail(GRPO_ERR_WORKSPACE, "forward launch of %lld rows exceeds the LSE partial buffers", (long long)rows);
  p.row_offset = t0;
  p.targets = targets;
  p.scale_log2e = c.logit_scale * kLog2e;
  p.logit_scale = c.logit_scale;
  p.part_m = part_m;
  p.part_s = part_s;
  p.part_u = entropy ? slot_ptr<float>(ctx, slot, L.off_part_u) : nullptr;
  p.part_stride = rows;
  p.zy = zy;
  p.dz = stash; p.dz_pitch = L.v_pad;
  p.stash_shift = slot_ptr<float>(ctx, slot, L.off_shift); p.shift_pitch = L.n_vtiles;
  p.sync = slot_ptr<unsigned int>(ctx, slot, L.off_sync);
  if (c.fp8_logits && !stash) {   // FP8 study: e4m3 operands, per-token and per-tensor scales folded into the epilogue
    if (t0 == 0) GRPO_TRY(quantize_weights(ctx, slot, W, st));        // once per call (the first row block)
    uint8_t* h8 = slot_ptr<uint8_t>(ctx, slot, L.off_h8);
    float* hscale = slot_ptr<float>(ctx, slot, L.off_hscale);
    GRPO_TRY(quantize_rows(ctx, Hc, rows, h8, hscale + t0, nullptr, st));
    CUtensorMap tmH8, tmW8;
    GRPO_TRY(make_tmap_u8(ctx, &tmH8, h8, c.d, rows, c.d, BM));
    GRPO_TRY(make_tmap_u8(ctx, &tmW8, slot_ptr<uint8_t>(ctx, slot, L.off_w8), c.d, c.V, c.d, BN / ctx->cg));
    p.k_blocks = (c.d + 2 * BK - 1) / (2 * BK);
    p.row_scale = hscale;
    p.w_scale = slot_ptr<float>(ctx, slot, L.off_wscale);
    GRPO_TRY((launch_gemm<false, false, EPI_LSE, 1>(ctx, GRPO_KERNEL_GEMM_LSE, tmH8, tmW8, p, p.m_tiles * p.n_split, st)));
  } else if (stash) {
    GRPO_TRY((launch_gemm<false, false, EPI_LSE_STASH>(ctx, GRPO_KERNEL_GEMM_LSE, tmH, tmW, p, p.m_tiles * p.n_split, st)));
  } else {
    GRPO_TRY((launch_gemm<false, false, EPI_LSE>(ctx, GRPO_KERNEL_GEMM_LSE, tmH, tmW, p, p.m_tiles * p.n_split, st)));
  }
  *n_split_out = p.n_split;
  return GRPO_OK;
}

// A3 over packed rows [t0, t0 + rows): combines `n_parts` (max, sum-exp) partials per token (part arrays
// [n_parts, part_stride], indexed by the launch's own row) and n_zy target-logit arrays (summed; stride zy_stride,
// indexed by the packed row), then the loss / coefficient arithmetic.  V = the GLOBAL vocabulary size.
static int32_t loss_rows(grpo_ctx* ctx, int slot, const float* part_m, const float* part_s, const float* part_u,
                         int n_parts, int64_t part_stride, const float* zy, int n_zy, int64_t zy_stride, int V,
                         const int32_t* targets, const FwdArgs& a, int64_t t0, int64_t rows, cudaStream_t st) {
  const grpo_config& c = ctx->cfg;
  const SlotLayout& L = ctx->lay;
  LossParams lp;
  std::memset(&lp, 0, sizeof(lp));
  lp.T = rows; lp.t_begin = t0; lp.S = a.S; lp.S_norm = a.S_norm > 0 ? a.S_norm : a.S; lp.V = V;
  lp.n_split = n_parts; lp.part_stride = part_stride;
  lp.part_m = part_m; lp.part_s = part_s; lp.part_u = part_u; lp.entropy = a.entropy_out; lp.zy = zy;
  lp.n_zy = n_zy; lp.zy_stride = zy_stride; lp.targets = targets; lp.cu_seqlens = a.cu_seqlens;
  lp.adv = a.adv; lp.old_logp = a.old_logp; lp.ref_logp = a.ref_logp; lp.mask = a.mask;
  lp.seq_count = slot_ptr<float>(ctx, slot, L.off_seq_count);
  lp.total_count = a.denom_dev ? a.denom_dev : slot_ptr<float>(ctx, slot, L.off_total);
  lp.denom_host = a.loss_denom > 0.0 ? static_cast<float>(a.loss_denom) : 0.f;
  lp.loss_agg = c.loss_agg; lp.clip_lo = c.clip_lo; lp.clip_hi = c.clip_hi; lp.kl_beta = c.kl_beta;
  lp.kl_type = c.kl_type; lp.dual_clip = c.dual_clip;
  lp.logp = a.logp_out; lp.lse = a.lse_out; lp.coeff = a.coeff_out; lp.loss_accum = a.loss_accum;
  lp.metrics_accum = a.metrics_accum; lp.err_flag = ctx->err_dev;
  lp.block_part = slot_ptr<float>(ctx, slot, L.off_loss_part);
  lp.block_count = slot_ptr<unsigned int>(ctx, slot, L.off_loss_count);
  const int threads = 256;
  const int blocks = static_cast<int>((rows + threads - 1) / threads);
  {
    LaunchScope ls(ctx, GRPO_KERNEL_LOSS, st);
    loss_epilogue_kernel<<<blocks, threads, 0, st>>>(lp);
  }
  CU_OK(cudaGetLastError());
  return GRPO_OK;
}

// A2 + A3 over packed rows [t0, t0 + rows) of a call of T tokens.  stash != nullptr: the 3-contraction
// variant's forward, which also writes the chunk's softmax numerators (fp16) to `stash`.
static int32_t fwd_rows(grpo_ctx* ctx, int slot, const void* hidden, const void* W, const int32_t* targets,
                        const FwdArgs& a, int64_t T, int64_t t0, int64_t rows, __nv_bfloat16* stash, cudaStream_t st) {
  const SlotLayout& L = ctx->lay;
  (void)T;
  float* zy = slot_ptr<float>(ctx, slot, L.off_zy);
  int n_split = 1;
  GRPO_TRY(a2_rows(ctx, slot, hidden, W, targets, zy, a.entropy_out != nullptr, t0, rows, stash, st, &n_split));
  return loss_rows(ctx, slot, slot_ptr<float>(ctx, slot, L.off_part_m), slot_ptr<float>(ctx, slot, L.off_part_s),
                   a.entropy_out ? slot_ptr<float>(ctx, slot, L.off_part_u) : nullptr, n_split, rows, zy, 1, 0,
                   ctx->cfg.V, targets, a, t0, rows, st);
}

static int32_t fwd_impl(grpo_ctx* ctx, int slot, const void* hidden, const void* W, const int32_t* targets,
                        const int32_t* cu_seqlens, int32_t S, int64_t T, const float* adv, const float* old_logp,
                        const float* ref_logp, const uint8_t* mask, double loss_denom, const float* denom_dev,
                        float* logp_out, float* lse_out, float* coeff_out, float* loss_accum, float* metrics_accum,
                        cudaStream_t st, float* entropy_out = nullptr, int32_t S_norm = 0) {
  GRPO_TRY(fwd_check(ctx, S, T));
  FwdArgs a{cu_seqlens, S, adv, old_logp, ref_logp, mask, loss_denom, denom_dev,
            logp_out, lse_out, coeff_out, loss_accum, metrics_accum};
  a.entropy_out = entropy_out;
  a.S_norm = S_norm;
  a.T_call = T;
  GRPO_TRY(fwd_counts(ctx, slot, targets, a, st));
  // A2 + A3 in launches of at most fwd_block_rows rows: bounds the LSE partial buffers; a row's result does not
  // depend on how the call is cut (fixed vocab split)
  for (int64_t t0 = 0; t0 < T; t0 += ctx->lay.fwd_block_rows)
    GRPO_TRY(fwd_rows(ctx, slot, hidden, W, targets, a, T, t0, std::min<int64_t>(ctx->lay.fwd_block_rows, T - t0),
                      nullptr, st));
  return GRPO_OK;
}

extern "C" int32_t grpo_fused_logprob_loss_fwd(grpo_ctx* ctx, const void* hidden, const void* W,
                                               const int32_t* targets, const int32_t* cu_seqlens, int32_t S,
                                               int64_t T, const float* adv, const float* old_logp,
                                               const float* ref_logp, const uint8_t* mask, double loss_denom,
                                               float* logp_out, float* lse_out, float* coeff_out, float* loss_accum,
                                               float* metrics_accum, void* stream) {
  if (!ctx || !hidden || !W || !targets || !cu_seqlens || !adv || !old_logp || !logp_out || !lse_out || !coeff_out ||
      !loss_accum)
    return fail(GRPO_ERR_INVALID_ARG, "a required pointer is NULL");
  if (T <= 0 || S <= 0) return fail(GRPO_ERR_SHAPE, "need T > 0 and S > 0 (got T=%lld S=%d)", (long long)T, S);
  return fwd_impl(ctx, 0, hidden, W, targets, cu_seqlens, S, T, adv, old_logp, ref_logp, mask, loss_denom, nullptr,
                  logp_out, lse_out, coeff_out, loss_accum, metrics_accum, static_cast<cudaStream_t>(stream),
                  ctx->entropy_out, ctx->seq_denom);
}

// ------------------------------------------------------------------------------------- NEXT-3(b): vocab-parallel LSE
// (max, sum-exp) of one token over the splits of a launch, in split order (log2 domain).
__global__ void combine_partials_kernel(const float* __restrict__ part_m, const float* __restrict__ part_s, int n_split,
                                        int64_t stride, int64_t rows, float* __restrict__ m2_out,
                                        float* __restrict__ s2_out) {
  const int64_t r = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (r >= rows) return;
  float M = -INFINITY;
  for (int i = 0; i < n_split; ++i) M = fmaxf(M, part_m[i * stride + r]);
  float sum = 0.f;
  for (int i = 0; i < n_split; ++i) sum += part_s[i * stride + r] * exp2f(part_m[i * stride + r] - M);
  m2_out[r] = M;
  s2_out[r] = sum;
}

extern "C" int32_t grpo_vocab_shard_partials(grpo_ctx* ctx, const void* hidden, const void* W_shard,
                                             const int32_t* targets_local, int64_t T, float* m2_out, float* s2_out,
                                             float* zy_out, void* stream) {
  if (!ctx || !hidden || !W_shard || !targets_local || !m2_out || !s2_out || !zy_out)
    return fail(GRPO_ERR_INVALID_ARG, "a required pointer is NULL");
  if (T <= 0) return fail(GRPO_ERR_SHAPE, "need T > 0");
  GRPO_TRY(fwd_check(ctx, 1, T));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const SlotLayout& L = ctx->lay;
  CU_OK(cudaMemsetAsync(zy_out, 0, static_cast<size_t>(T) * 4, st));   // rows whose target lives in another shard
  for (int64_t t0 = 0; t0 < T; t0 += L.fwd_block_rows) {
    const int64_t rows = std::min<int64_t>(L.fwd_block_rows, T - t0);
    int n_split = 1;
    GRPO_TRY(a2_rows(ctx, 0, hidden, W_shard, targets_local, zy_out, false, t0, rows, nullptr, st, &n_split));
    {
      LaunchScope ls(ctx, GRPO_KERNEL_LOSS, st);
      combine_partials_kernel<<<static_cast<unsigned>((rows + 255) / 256), 256, 0, st>>>(
          slot_ptr<float>(ctx, 0, L.off_part_m), slot_ptr<float>(ctx, 0, L.off_part_s), n_split, rows, rows, m2_out + t0,
          s2_out + t0);
    }
    CU_OK(cudaGetLastError());
  }
  return GRPO_OK;
}

extern "C" int32_t grpo_loss_from_partials(grpo_ctx* ctx, int32_t n_shards, const float* m2, const float* s2,
                                           const float* zy, const int32_t* targets, int32_t V_global,
                                           const int32_t* cu_seqlens, int32_t S, int64_t T, const float* adv,
                                           const float* old_logp, const float* ref_logp, const uint8_t* mask,
                                           double loss_denom, float* logp_out, float* lse_out, float* coeff_out,
                                           float* loss_accum, float* metrics_accum, void* stream) {
  if (!ctx || !m2 || !s2 || !zy || !targets || !cu_seqlens || !adv || !old_logp || !logp_out || !lse_out || !coeff_out ||
      !loss_accum)
    return fail(GRPO_ERR_INVALID_ARG, "a required pointer is NULL");
  if (n_shards < 1 || V_global < 1 || T <= 0 || S <= 0) return fail(GRPO_ERR_SHAPE, "need n_shards, V_global, T, S > 0");
  GRPO_TRY(fwd_check(ctx, S, T));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  FwdArgs a{cu_seqlens, S, adv, old_logp, ref_logp, mask, loss_denom, nullptr,
            logp_out, lse_out, coeff_out, loss_accum, metrics_accum};
  a.S_norm = ctx->seq_denom;
  a.T_call = T;
  GRPO_TRY(fwd_counts(ctx, 0, targets, a, st, V_global));
  return loss_rows(ctx, 0, m2, s2, nullptr, n_shards, T, zy, n_shards, T, V_global, targets, a, 0, T, st);
}

extern "C" int32_t grpo_set_seq_denom(grpo_ctx* ctx, int32_t n_sequences) {
  if (!ctx || n_sequences < 0) return fail(GRPO_ERR_INVALID_ARG, "ctx is NULL or n_sequences < 0");
  ctx->seq_denom = n_sequences;
  return GRPO_OK;
}

extern "C" int32_t grpo_set_entropy_out(grpo_ctx* ctx, float* entropy_out) {
  if (!ctx) return fail(GRPO_ERR_INVALID_ARG, "ctx is NULL");
  ctx->entropy_out = entropy_out;
  return GRPO_OK;
}

// ------------------------------------------------------------------------------------- A4 - A6
// Token rows per backward chunk: whole pair tiles, equalised so that the last chunk is not a sliver.
static int64_t rows_per_chunk_for(const grpo_ctx* ctx, int64_t T) {
  const int64_t Tc = ctx->lay.chunk_rows;
  const int64_t n_chunks = (T + Tc - 1) / Tc;
  return std::min<int64_t>(Tc, align_up((T + n_chunks - 1) / n_chunks, 256));
}

// grpo_step_host's copy pipeline: chunk i of the hidden states arrives on the copy stream (in[i]), and the
// dHidden rows of chunk i leave on it as soon as A5 has written them, under the next chunk's contractions.
struct HostPipe {
  cudaStream_t cs;
  std::vector<cudaEvent_t> in, out;   // owned by the context (grpo_ctx::pipe_events)
  uint8_t* dh_host;
};

// fused == nullptr: the backward of north_star (A4 recomputes the logits).  fused != nullptr: the
// 3-contraction variant: per chunk, the forward runs first and stashes the chunk's
// logits, which are then converted to dZ in place instead of being recomputed; lse / coeff are fused's.
//
// Zero-coefficient work is skipped (cfg.bwd_skip_zero_tiles >= 0):
//   north_star path: token-granular.  The call's rows with coeff != 0 are compacted on the device
//     (compact_rows_kernel), each backward chunk gathers its active hidden rows into a dense panel, A4 - A6 run
//     on that panel with the row count read from device memory, and the split-K reduction of A5 scatters the
//     dHidden rows back; rows with coeff == 0 are written as zeros.  Nothing is decided on the host.
//   3-contraction variant: the same per chunk (a chunk's logits are stashed before its coefficients exist): the
//     conversion pass writes the dZ rows of the chunk's active tokens, compacted, into a second chunk buffer.
// RMSNorm in front of the path: when given, the A5 reduction turns each dHidden row into
// dx (written to `dhidden_out`, which is then the dx buffer) and adds its share of dgamma.
struct PrenormArgs { const void* x; const void* gamma; const float* rstd; float* dgamma; };

static int32_t launch_prenorm_bwd(grpo_ctx* ctx, bool in_bf16, const void* parts, int k_split, int64_t split_stride_vec,
                                  int rows, const int* dyn_rows, const int* row_idx, int64_t row0, const PrenormArgs& pn,
                                  void* dx_out, cudaStream_t st) {
  const grpo_config& c = ctx->cfg;
  const int row_vec = c.d / 4;
  const int J = (row_vec + 255) / 256;
  if (J > 8) return fail(GRPO_ERR_SHAPE, "RMSNorm backward supports d <= 8192 (got %d)", c.d);
  const int grid = std::min(rows, 4 * ctx->num_sms);
  if (grid <= 0) return GRPO_OK;
  LaunchScope ls(ctx, GRPO_KERNEL_DH_REDUCE, st);
#define GRPO_PN(JJ)                                                                                                   \
  do {                                                                                                                \
    if (in_bf16)                                                                                                      \
      prenorm_bwd_kernel<JJ, true><<<grid, 256, 0, st>>>(parts, k_split, split_stride_vec, row_vec, rows, dyn_rows,   \
          row_idx, row0, static_cast<const uint2*>(pn.x), static_cast<const uint2*>(pn.gamma), pn.rstd, 1.f / c.d,    \
          dx_out, c.dhidden_fp32, pn.dgamma);                                                                         \
    else                                                                                                              \
      prenorm_bwd_kernel<JJ, false><<<grid, 256, 0, st>>>(parts, k_split, split_stride_vec, row_vec, rows, dyn_rows,  \
          row_idx, row0, static_cast<const uint2*>(pn.x), static_cast<const uint2*>(pn.gamma), pn.rstd, 1.f / c.d,    \
          dx_out, c.dhidden_fp32, pn.dgamma);                                                                         \
  } while (0)
  if (J <= 1) GRPO_PN(1); else if (J <= 2) GRPO_PN(2); else if (J <= 4) GRPO_PN(4); else GRPO_PN(8);
#undef GRPO_PN
  return GRPO_OK;
}

static int32_t bwd_impl(grpo_ctx* ctx, int slot, const void* hidden, const void* W, const int32_t* targets,
                        const float* lse, const float* coeff, int64_t T, float grad_scale, void* dhidden_out,
                        float* dW_accum, cudaStream_t st, const FwdArgs* fused = nullptr, HostPipe* pipe = nullptr,
                        const PrenormArgs* pn = nullptr) {
  const grpo_config& c = ctx->cfg;
  if (!ctx->ws) return fail(GRPO_ERR_WORKSPACE, "no workspace set (grpo_set_workspace)");
  if (T > ctx->ws_max_T) return fail(GRPO_ERR_WORKSPACE, "T=%lld exceeds workspace max_T=%lld", (long long)T, (long long)ctx->ws_max_T);
  if (!dhidden_out && !dW_accum && !fused) return GRPO_OK;
  if (pn && fused) return fail(GRPO_ERR_INVALID_ARG, "the pre-norm backward is not available for the stash variant");
  const SlotLayout& L = ctx->lay;
  __nv_bfloat16* dz = slot_ptr<__nv_bfloat16>(ctx, slot, L.off_dz);
  const int64_t rows_per_chunk = rows_per_chunk_for(ctx, T);
  const int n_chunks = static_cast<int>((T + rows_per_chunk - 1) / rows_per_chunk);
  const uint8_t* Hb = static_cast<const uint8_t*>(hidden);
  const int dh_elem = c.dhidden_fp32 ? 4 : 2;
  const bool compact = c.bwd_skip_zero_tiles >= 0;
  const int TM = BM * ctx->cg;
  int k_split, kb_per_split;
  dh_ksplit(c.V, &k_split, &kb_per_split);
  float* dh_part = slot_ptr<float>(ctx, slot, L.off_dh_part);

  CUtensorMap tmW_k, tmW_mn;
  GRPO_TRY(make_tmap(ctx, &tmW_k, W, c.d, c.V, static_cast<uint64_t>(c.d) * 2, BK, BN / ctx->cg));
  GRPO_TRY(make_tmap(ctx, &tmW_mn, W, c.d, c.V, static_cast<uint64_t>(c.d) * 2, 64, BK));

  int* row_idx = slot_ptr<int>(ctx, slot, L.off_row_idx);
  int* meta = slot_ptr<int>(ctx, slot, L.off_meta);
  long long* row_stats = slot_ptr<long long>(ctx, slot, L.off_row_stats);
  if (compact && n_chunks > L.n_chunks_max) return fail(GRPO_ERR_WORKSPACE, "too many backward chunks for the workspace");
  // Row compaction.  north_star path: once for the call (the forward has produced every coefficient), so that every
  // chunk but the last is full.  3-contraction variant: per chunk, after the chunk's forward.
  auto compact_rows = [&](const float* cf, int64_t n_rows, int64_t chunk_rows, int chunks, int* idx, int* m,
                          uint8_t* dh_rows) -> int32_t {
    {
      LaunchScope ls(ctx, GRPO_KERNEL_COMPACT, st);
      compact_rows_kernel<<<1, 1024, 0, st>>>(cf, static_cast<int>(n_rows), static_cast<int>(chunk_rows), chunks, idx, m,
                                              row_stats);
    }
    CU_OK(cudaGetLastError());
    if (dh_rows) {
      LaunchScope ls(ctx, GRPO_KERNEL_COMPACT, st);
      zero_coeff_rows_kernel<<<static_cast<unsigned>(n_rows), 128, 0, st>>>(cf, static_cast<int>(n_rows), dh_rows,
                                                                           static_cast<int64_t>(c.d) * dh_elem);
      CU_OK(cudaGetLastError());
    }
    return GRPO_OK;
  };
  if (compact && !fused)
    GRPO_TRY(compact_rows(coeff, T, rows_per_chunk, n_chunks, row_idx, meta, static_cast<uint8_t*>(dhidden_out)));

  for (int64_t t0 = 0; t0 < T; t0 += rows_per_chunk) {
    const int64_t rows = std::min<int64_t>(rows_per_chunk, T - t0);       // static upper bound of the chunk's rows
    const size_t chunk_idx = static_cast<size_t>(t0 / rows_per_chunk);
    const int m_tiles = static_cast<int>((rows + TM - 1) / TM);
    // compact: the chunk's operands live in dense panels of the workspace whose tails are zero-filled explicitly
    // (the row count is only known on the device); otherwise the tensor maps end at `rows` and TMA zero-fills.
    const int64_t map_rows = compact ? align_up(rows, 256) : rows;
    // row_idx entries of this chunk: absolute packed rows (north_star) or chunk-local rows (3-contraction variant)
    int* idx_c = row_idx + t0;
    const int* dyn_rows = !compact ? nullptr : (fused ? meta + 4 * chunk_idx + 2 : meta + 2 + chunk_idx);
    const void* Hc = compact ? static_cast<const void*>(slot_ptr<uint8_t>(ctx, slot, L.off_hc))
                             : static_cast<const void*>(Hb + t0 * c.d * 2);
    const int32_t* y_c = compact ? slot_ptr<int32_t>(ctx, slot, L.off_yc) : targets;
    const float* lse_c = compact ? slot_ptr<float>(ctx, slot, L.off_lsec) : lse;
    const float* coeff_c = compact ? slot_ptr<float>(ctx, slot, L.off_coeffc) : coeff;
    const int64_t row_off = compact ? 0 : t0;
    // where the dZ rows A5 / A6 contract live: the chunk buffer, or (compacted 3-contraction variant) the second one
    __nv_bfloat16* dz_rows = (fused && compact) ? slot_ptr<__nv_bfloat16>(ctx, slot, L.off_dz2) : dz;
    uint8_t* dh_chunk = dhidden_out ? static_cast<uint8_t*>(dhidden_out) + t0 * c.d * dh_elem : nullptr;

    if (fused) {
      if (pipe && chunk_idx < pipe->in.size()) CU_OK(cudaStreamWaitEvent(st, pipe->in[chunk_idx], 0));
      GRPO_TRY(fwd_rows(ctx, slot, hidden, W, targets, *fused, T, t0, rows, dz, st));
    }
    if (!dhidden_out && !dW_accum) continue;
    if (fused && compact)
      GRPO_TRY(compact_rows(coeff + t0, rows, rows, 1, idx_c, meta + 4 * chunk_idx, dh_chunk));

    if (compact) {
      LaunchScope ls(ctx, GRPO_KERNEL_COMPACT, st);
      gather_rows_kernel<<<static_cast<unsigned>(map_rows), 128, 0, st>>>(
          reinterpret_cast<const uint4*>(fused ? Hb + t0 * c.d * 2 : Hb), c.d / 8, idx_c, dyn_rows, 256,
          static_cast<int>(L.chunk_rows), fused ? targets + t0 : targets, fused ? lse + t0 : lse, fused ? coeff + t0 : coeff,
          slot_ptr<uint4>(ctx, slot, L.off_hc), slot_ptr<int32_t>(ctx, slot, L.off_yc),
          slot_ptr<float>(ctx, slot, L.off_lsec), slot_ptr<float>(ctx, slot, L.off_coeffc));
      CU_OK(cudaGetLastError());
    }

    CUtensorMap tmH_k, tmH_mn, tmDZ_k, tmDZ_mn;
    GRPO_TRY(make_tmap(ctx, &tmDZ_k, dz_rows, c.V, map_rows, static_cast<uint64_t>(L.v_pad) * 2, BK, BM));
    if (fused) {  // stashed softmax numerators -> dZ (HBM-bound elementwise pass instead of the A4 contraction)
      LaunchScope ls(ctx, GRPO_KERNEL_STASH_DZ, st);
      stash_to_dz_kernel<<<static_cast<unsigned>(map_rows), 256, 0, st>>>(
          reinterpret_cast<const uint16_t*>(dz), reinterpret_cast<uint16_t*>(dz_rows), static_cast<int>(rows), c.V, L.v_pad,
          slot_ptr<float>(ctx, slot, L.off_shift), L.n_vtiles, BN, targets + t0, lse + t0, coeff + t0,
          c.logit_scale * grad_scale, compact ? idx_c : nullptr, dyn_rows, 256, static_cast<int>(L.chunk_rows));
      CU_OK(cudaGetLastError());
    } else {  // A4: recompute logits, dZ = coeff (1[v=y] - p) * logit_scale * grad_scale  -> bf16 chunk
      GRPO_TRY(make_tmap(ctx, &tmH_k, Hc, c.d, map_rows, static_cast<uint64_t>(c.d) * 2, BK, BM));
      GemmParams p;
      std::memset(&p, 0, sizeof(p));
      p.m_total = static_cast<int>(rows); p.n_total = c.V;
      p.m_tiles = m_tiles; p.n_tiles = (c.V + BN - 1) / BN; p.k_blocks = (c.d + BK - 1) / BK;
      p.n_fastest = 0;
      p.m_block = static_cast<int>(std::max<int64_t>(1, kA4BlockBytes / (static_cast<int64_t>(TM) * c.d * 2)));
      p.row_offset = row_off; p.targets = y_c;
      p.scale_log2e = c.logit_scale * kLog2e; p.logit_scale = c.logit_scale;
      p.lse = lse_c; p.coeff = coeff_c; p.coeff_mul = c.logit_scale * grad_scale;
      p.dz = dz; p.dz_pitch = L.v_pad; p.dyn_rows = dyn_rows;
      p.m_alloc = compact ? static_cast<int>(L.chunk_rows) : 0;
      p.sync = slot_ptr<unsigned int>(ctx, slot, L.off_sync);
      if (c.fp8_logits) {   // FP8 study: the logits are recomputed from the same e4m3 operands the forward used
        if (t0 == 0) GRPO_TRY(quantize_weights(ctx, slot, W, st));
        uint8_t* h8 = slot_ptr<uint8_t>(ctx, slot, L.off_h8);
        float* hscale = slot_ptr<float>(ctx, slot, L.off_hscale);
        GRPO_TRY(quantize_rows(ctx, Hc, map_rows, h8, hscale + row_off, nullptr, st));
        CUtensorMap tmH8, tmW8;
        GRPO_TRY(make_tmap_u8(ctx, &tmH8, h8, c.d, map_rows, c.d, BM));
        GRPO_TRY(make_tmap_u8(ctx, &tmW8, slot_ptr<uint8_t>(ctx, slot, L.off_w8), c.d, c.V, c.d, BN / ctx->cg));
        p.k_blocks = (c.d + 2 * BK - 1) / (2 * BK);
        p.row_scale = hscale;
        p.w_scale = slot_ptr<float>(ctx, slot, L.off_wscale);
        GRPO_TRY((launch_gemm<false, false, EPI_DZ, 1>(ctx, GRPO_KERNEL_GEMM_DZ, tmH8, tmW8, p, p.m_tiles * p.n_tiles, st)));
      } else {
        GRPO_TRY((launch_gemm<false, false, EPI_DZ>(ctx, GRPO_KERNEL_GEMM_DZ, tmH_k, tmW_k, p, p.m_tiles * p.n_tiles, st)));
      }
    }
    if (dhidden_out) {  // A5: dH[rows, d] = dZ[rows, V] W[V, d], K cut into k_split fixed ranges, fp32 partials
      GemmParams p;
      std::memset(&p, 0, sizeof(p));
      p.m_total = static_cast<int>(rows); p.n_total = c.d;
      p.m_tiles = m_tiles; p.n_tiles = (c.d + BN - 1) / BN; p.k_blocks = (c.V + BK - 1) / BK;
      p.n_fastest = 1; p.n_group = kNGroupTiles;
      p.k_split = k_split; p.kb_per_split = kb_per_split; p.c_split_stride = L.chunk_rows * c.d;
      p.c_out = dh_part; p.c_pitch = c.d;
      p.dyn_rows = dyn_rows;
      p.sync = slot_ptr<unsigned int>(ctx, slot, L.off_sync);
      GRPO_TRY((launch_gemm<false, true, EPI_STORE>(ctx, GRPO_KERNEL_GEMM_DH, tmDZ_k, tmW_mn, p,
                                                    p.m_tiles * p.n_tiles * k_split, st)));
      // the reduction scatters compacted row r to packed row idx_c[r]: absolute for the north_star path (base = the
      // call's dHidden), chunk-local for the 3-contraction variant (base = the chunk's rows)
      void* scatter_base = (compact && !fused) ? dhidden_out : static_cast<void*>(dh_chunk);
      if (pn) {  // ... -> dx, dgamma (RMSNorm backward fused behind the reduction; dHidden is never written)
        GRPO_TRY(launch_prenorm_bwd(ctx, false, dh_part, k_split, L.chunk_rows * c.d / 4, static_cast<int>(rows), dyn_rows,
                                    compact ? idx_c : nullptr, t0, *pn, dhidden_out, st));
      } else {  // fixed-order sum of the partials (+ scatter of compacted rows) -> dHidden
        LaunchScope ls(ctx, GRPO_KERNEL_DH_REDUCE, st);
        splitk_reduce_kernel<<<static_cast<unsigned>(rows), 128, 0, st>>>(
            reinterpret_cast<const float4*>(dh_part), k_split, L.chunk_rows * c.d / 4, c.d / 4, static_cast<int>(rows),
            dyn_rows, compact ? idx_c : nullptr, scatter_base, c.dhidden_fp32);
      }
      CU_OK(cudaGetLastError());
      if (pipe && pipe->dh_host && chunk_idx < pipe->out.size()) {
        // packed rows [t0, t0 + rows) are final: compaction preserves order, so every active packed row below
        // t0 + rows has a compact index below it as well, and rows with a zero coefficient were written first
        CU_OK(cudaEventRecord(pipe->out[chunk_idx], st));
        CU_OK(cudaStreamWaitEvent(pipe->cs, pipe->out[chunk_idx], 0));
        CU_OK(cudaMemcpyAsync(pipe->dh_host + t0 * c.d * dh_elem, dh_chunk, rows * c.d * dh_elem, cudaMemcpyDeviceToHost,
                              pipe->cs));
      }
    }
    if (dW_accum) {  // A6: dW[V, d] += dZ^T[V, rows] H[rows, d]
      GRPO_TRY(make_tmap(ctx, &tmDZ_mn, dz_rows, c.V, map_rows, static_cast<uint64_t>(L.v_pad) * 2, 64, BK));
      GRPO_TRY(make_tmap(ctx, &tmH_mn, Hc, c.d, map_rows, static_cast<uint64_t>(c.d) * 2, 64, BK));
      GemmParams p;
      std::memset(&p, 0, sizeof(p));
      p.m_total = c.V; p.n_total = c.d;
      p.m_tiles = (c.V + TM - 1) / TM; p.n_tiles = (c.d + BN - 1) / BN;
      p.k_blocks = static_cast<int>((rows + BK - 1) / BK);
      p.n_fastest = 1; p.n_group = kNGroupTiles;
      p.c_out = dW_accum; p.c_pitch = c.d; p.dyn_rows = dyn_rows;
      p.sync = slot_ptr<unsigned int>(ctx, slot, L.off_sync);
      CUtensorMap tmDW;
      GRPO_TRY(make_tmap_c_f32(ctx, &tmDW, dW_accum, c.d, c.V, static_cast<uint64_t>(c.d) * 4));
      GRPO_TRY((launch_gemm<true, true, EPI_RED_F32>(ctx, GRPO_KERNEL_GEMM_DW, tmDZ_mn, tmH_mn, p, p.m_tiles * p.n_tiles, st, &tmDW)));
    }
  }
  return GRPO_OK;
}

extern "C" int32_t grpo_fused_logprob_loss_bwd(grpo_ctx* ctx, const void* hidden, const void* W,
                                               const int32_t* targets, const float* lse, const float* coeff,
                                               int64_t T, float grad_scale, void* dhidden_out, float* dW_accum,
                                               void* stream) {
  if (!ctx || !hidden || !W || !targets || !lse || !coeff) return fail(GRPO_ERR_INVALID_ARG, "a required pointer is NULL");
  if (T <= 0) return fail(GRPO_ERR_SHAPE, "need T > 0");
  return bwd_impl(ctx, 0, hidden, W, targets, lse, coeff, T, grad_scale, dhidden_out, dW_accum,
                  static_cast<cudaStream_t>(stream));
}

// ------------------------------------------------------------------------------------- NEXT-4: final RMSNorm
extern "C" int32_t grpo_rmsnorm_fwd(grpo_ctx* ctx, const void* x, const void* gamma, float eps_rms, int64_t T,
                                    void* hidden_out, float* rstd_out, void* stream) {
  if (!ctx || !x || !gamma || !hidden_out || !rstd_out) return fail(GRPO_ERR_INVALID_ARG, "a required pointer is NULL");
  if (T <= 0) return fail(GRPO_ERR_SHAPE, "need T > 0");
  if (!(eps_rms >= 0.f)) return fail(GRPO_ERR_INVALID_ARG, "eps_rms must be >= 0");
  if ((reinterpret_cast<uintptr_t>(x) | reinterpret_cast<uintptr_t>(gamma) | reinterpret_cast<uintptr_t>(hidden_out)) & 7)
    return fail(GRPO_ERR_SHAPE, "x / gamma / hidden_out must be 8-byte aligned");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int warps_per_block = 8;
  const int64_t blocks = std::min<int64_t>((T + warps_per_block - 1) / warps_per_block, 32LL * ctx->num_sms);
  {
    LaunchScope ls(ctx, GRPO_KERNEL_RMSNORM, st);
    rmsnorm_fwd_kernel<<<static_cast<unsigned>(blocks), 256, 0, st>>>(
        static_cast<const uint2*>(x), static_cast<const uint2*>(gamma), T, ctx->cfg.d / 4, 1.f / ctx->cfg.d, eps_rms,
        static_cast<uint2*>(hidden_out), rstd_out);
  }
  CU_OK(cudaGetLastError());
  return GRPO_OK;
}

extern "C" int32_t grpo_rmsnorm_bwd(grpo_ctx* ctx, const void* x, const void* gamma, const float* rstd,
                                    const void* dhidden, int32_t dhidden_is_fp32, int64_t T, void* dx_out,
                                    float* dgamma_accum, void* stream) {
  if (!ctx || !x || !gamma || !rstd || !dhidden || !dx_out || !dgamma_accum)
    return fail(GRPO_ERR_INVALID_ARG, "a required pointer is NULL");
  if (T <= 0 || T > INT32_MAX - 256) return fail(GRPO_ERR_SHAPE, "need 0 < T < 2^31");
  const PrenormArgs pn{x, gamma, rstd, dgamma_accum};
  GRPO_TRY(launch_prenorm_bwd(ctx, dhidden_is_fp32 == 0, dhidden, 1, 0, static_cast<int>(T), nullptr, nullptr, 0, pn,
                              dx_out, static_cast<cudaStream_t>(stream)));
  CU_OK(cudaGetLastError());
  return GRPO_OK;
}

extern "C" int32_t grpo_fused_logprob_loss_bwd_prenorm(grpo_ctx* ctx, const void* x, const void* gamma,
                                                       const float* rstd, const void* hidden, const void* W,
                                                       const int32_t* targets, const float* lse, const float* coeff,
                                                       int64_t T, float grad_scale, void* dx_out, float* dgamma_accum,
                                                       float* dW_accum, void* stream) {
  if (!ctx || !x || !gamma || !rstd || !hidden || !W || !targets || !lse || !coeff || !dx_out || !dgamma_accum)
    return fail(GRPO_ERR_INVALID_ARG, "a required pointer is NULL");
  if (T <= 0) return fail(GRPO_ERR_SHAPE, "need T > 0");
  const PrenormArgs pn{x, gamma, rstd, dgamma_accum};
  return bwd_impl(ctx, 0, hidden, W, targets, lse, coeff, T, grad_scale, dx_out, dW_accum,
                  static_cast<cudaStream_t>(stream), nullptr, nullptr, &pn);
}

extern "C" int32_t grpo_fused_logprob_loss_fwd_bwd(grpo_ctx* ctx, const void* hidden, const void* W,
                                                   const int32_t* targets, const int32_t* cu_seqlens, int32_t S,
                                                   int64_t T, const float* adv, const float* old_logp,
                                                   const float* ref_logp, const uint8_t* mask, double loss_denom,
                                                   float grad_scale, float* logp_out, float* lse_out, float* coeff_out,
                                                   float* loss_accum, float* metrics_accum, void* dhidden_out,
                                                   float* dW_accum, void* stream) {
  if (!ctx || !hidden || !W || !targets || !cu_seqlens || !adv || !old_logp || !logp_out || !lse_out || !coeff_out ||
      !loss_accum)
    return fail(GRPO_ERR_INVALID_ARG, "a required pointer is NULL");
  if (T <= 0 || S <= 0) return fail(GRPO_ERR_SHAPE, "need T > 0 and S > 0 (got T=%lld S=%d)", (long long)T, S);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  GRPO_TRY(fwd_check(ctx, S, T));
  FwdArgs a{cu_seqlens, S, adv, old_logp, ref_logp, mask, loss_denom, nullptr,
            logp_out, lse_out, coeff_out, loss_accum, metrics_accum};
  a.entropy_out = ctx->entropy_out;
  a.S_norm = ctx->seq_denom;
  a.T_call = T;
  GRPO_TRY(fwd_counts(ctx, 0, targets, a, st));
  return bwd_impl(ctx, 0, hidden, W, targets, lse_out, coeff_out, T, grad_scale, dhidden_out, dW_accum, st, &a);
}

// ------------------------------------------------------------------------------------- A0 / A7: CGP FIFO
extern "C" int32_t grpo_cgp_plan(const int64_t* group_tokens, int32_t n_pending, int32_t U, int64_t token_budget,
                                 int32_t flush, int32_t* launch_sizes_out, int32_t cap, int32_t* n_launches_out) {
  if (!n_launches_out || n_pending < 0 || (n_pending > 0 && !group_tokens))
    return fail(GRPO_ERR_INVALID_ARG, "bad arguments");
  std::vector<int> sizes;
  plan_update(group_tokens, n_pending, U, token_budget, flush != 0, sizes);
  if (static_cast<int>(sizes.size()) > cap) return fail(GRPO_ERR_INVALID_ARG, "launch_sizes_out too small");
  for (size_t i = 0; i < sizes.size(); ++i) launch_sizes_out[i] = sizes[i];
  *n_launches_out = static_cast<int32_t>(sizes.size());
  return GRPO_OK;
}

extern "C" int32_t grpo_queue_state(const grpo_ctx* ctx, int32_t* pending_groups, int64_t* pending_tokens,
                                    int32_t* consumed_groups, int32_t* round_complete) {
  if (!ctx) return fail(GRPO_ERR_INVALID_ARG, "ctx is NULL");
  if (pending_groups) *pending_groups = static_cast<int32_t>(ctx->fifo.size());
  if (pending_tokens) {
    int64_t s = 0;
    for (const auto& g : ctx->fifo) s += g.tokens;
    *pending_tokens = s;
  }
  if (consumed_groups) *consumed_groups = ctx->consumed;
  if (round_complete) *round_complete = (ctx->cfg.groups_per_round > 0 && ctx->consumed >= ctx->cfg.groups_per_round) ? 1 : 0;
  return GRPO_OK;
}

extern "C" int32_t grpo_reset_round(grpo_ctx* ctx) {
  if (!ctx) return fail(GRPO_ERR_INVALID_ARG, "ctx is NULL");
  ctx->fifo.clear();
  ctx->consumed = 0;
  ctx->update_broken = false;
  return GRPO_OK;
}

__global__ void token_count_flat_kernel(const uint8_t* __restrict__ mask, const int32_t* __restrict__ targets, int V,
                                        int64_t T, float* __restrict__ total) {
  int c = 0;
  for (int64_t t = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; t < T;
       t += static_cast<int64_t>(gridDim.x) * blockDim.x) {
    const int y = targets[t];
    c += ((mask == nullptr || mask[t] != 0) && y >= 0 && y < V) ? 1 : 0;
  }
  const float cf = warp_sum(static_cast<float>(c));
  if ((threadIdx.x & 31) == 0 && cf != 0.f) atomicAdd(total, cf);
}
__global__ void fill_u8_kernel(uint8_t* p, int64_t n, uint8_t v) {
  for (int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < n;
       i += static_cast<int64_t>(gridDim.x) * blockDim.x)
    p[i] = v;
}

static int32_t validate_group(const grpo_ctx* ctx, const grpo_group_desc& g) {
  if (g.G <= 0 || (ctx->cfg.group_size > 0 && g.G != ctx->cfg.group_size))
    return fail(GRPO_ERR_INCOMPLETE_GROUP, "group %lld has G=%d, expected %d complete responses", (long long)g.group_order,
                g.G, ctx->cfg.group_size);
  if (!g.seqlens_host || !g.hidden || !g.targets || !g.old_logp || !g.rewards)
    return fail(GRPO_ERR_INCOMPLETE_GROUP, "group %lld is missing hidden/targets/old_logp/rewards/seqlens",
                (long long)g.group_order);
  for (int i = 0; i < g.G; ++i)
    if (g.seqlens_host[i] <= 0)
      return fail(GRPO_ERR_INCOMPLETE_GROUP, "group %lld response %d has no tokens", (long long)g.group_order, i);
  return GRPO_OK;
}

// Everything about a launch of `k` whole groups that can be rejected WITHOUT touching the device: checked for
// every launch of a logical update before its first kernel is enqueued, so that a bad update leaves the
// accumulators and the FIFO untouched (drain_one_update).
static int32_t validate_launch(const grpo_ctx* ctx, const PendingGroup* groups, int k) {
  int64_t T = 0;
  int64_t S = 0;
  bool any_ref = false, all_ref = true;
  for (int i = 0; i < k; ++i) {
    T += groups[i].tokens;
    S += groups[i].desc.G;
    any_ref |= groups[i].desc.ref_logp != nullptr;
    all_ref &= groups[i].desc.ref_logp != nullptr;
  }
  if (!ctx->ws) return fail(GRPO_ERR_WORKSPACE, "no workspace set (grpo_set_workspace)");
  if (T > ctx->ws_max_T) return fail(GRPO_ERR_WORKSPACE, "launch of %lld tokens exceeds workspace max_T=%lld", (long long)T, (long long)ctx->ws_max_T);
  if (S > ctx->lay.s_max) return fail(GRPO_ERR_WORKSPACE, "too many sequences in one launch");
  if (T > INT32_MAX - 256) return fail(GRPO_ERR_SHAPE, "T too large");
  if (any_ref && !all_ref) return fail(GRPO_ERR_INVALID_ARG, "ref_logp must be given for all groups of a launch or none");
  return GRPO_OK;
}

// One launch = A1 -> A2/A3 -> A4-A6 over `k` whole groups packed into one token stream.  S_update: sequences
// of the whole logical update (the per-sequence mean of loss_agg 1 averages over all of them, R10).
static int32_t run_launch(grpo_ctx* ctx, const PendingGroup* groups, int k, const void* W, float* dW_accum,
                          float* loss_accum, float* metrics_accum, double loss_denom, const float* denom_dev,
                          int32_t S_update, int slot, cudaStream_t st) {
  const grpo_config& c = ctx->cfg;
  const SlotLayout& L = ctx->lay;
  GRPO_TRY(validate_launch(ctx, groups, k));
  int64_t T = 0;
  int S = 0;
  bool any_ref = false, any_mask = false, any_dh = false;
  for (int i = 0; i < k; ++i) {
    T += groups[i].tokens;
    S += groups[i].desc.G;
    any_ref |= groups[i].desc.ref_logp != nullptr;
    any_mask |= groups[i].desc.mask != nullptr;
    any_dh |= groups[i].desc.dhidden_out != nullptr;
  }

  // small host-built index arrays, staged in the context's pinned ring (a pageable source would make the copy
  // synchronise the stream with the host and serialise multi-stream dispatch)
  const int ring = ctx->stage_next++ % grpo_ctx::kStageRing;
  CU_OK(cudaEventSynchronize(ctx->stage_ev[ring]));          // the copies that last used this entry have run
  int32_t* cu_seq = ctx->stage_host + static_cast<int64_t>(ring) * ctx->stage_ints;
  int32_t* cu_grp = cu_seq + (L.s_max + 1);
  cu_seq[0] = 0;
  cu_grp[0] = 0;
  int s = 0;
  for (int i = 0; i < k; ++i) {
    for (int j = 0; j < groups[i].desc.G; ++j, ++s) cu_seq[s + 1] = cu_seq[s] + groups[i].seqlens[j];
    cu_grp[i + 1] = s;
  }
  int32_t* d_cu_seq = slot_ptr<int32_t>(ctx, slot, L.off_cu_seq);
  int32_t* d_cu_grp = slot_ptr<int32_t>(ctx, slot, L.off_cu_grp);
  float* d_rewards = slot_ptr<float>(ctx, slot, L.off_rewards);
  float* d_adv = slot_ptr<float>(ctx, slot, L.off_adv);
  CU_OK(cudaMemcpyAsync(d_cu_seq, cu_seq, (S + 1) * 4, cudaMemcpyHostToDevice, st));
  CU_OK(cudaMemcpyAsync(d_cu_grp, cu_grp, (k + 1) * 4, cudaMemcpyHostToDevice, st));
  CU_OK(cudaEventRecord(ctx->stage_ev[ring], st));
  for (int i = 0; i < k; ++i)
    CU_OK(cudaMemcpyAsync(d_rewards + cu_grp[i], groups[i].desc.rewards, groups[i].desc.G * 4, cudaMemcpyDeviceToDevice, st));

  // pack the token stream (a single group is used in place)
  const void* hidden;
  const int32_t* targets;
  const float *old_logp, *ref_logp;
  const uint8_t* mask;
  const int dh_elem = c.dhidden_fp32 ? 4 : 2;
  if (k == 1) {
    hidden = groups[0].desc.hidden; targets = groups[0].desc.targets; old_logp = groups[0].desc.old_logp;
    ref_logp = groups[0].desc.ref_logp; mask = groups[0].desc.mask;
  } else {
    uint8_t* sh = slot_ptr<uint8_t>(ctx, slot, L.off_hidden);
    int32_t* stg = slot_ptr<int32_t>(ctx, slot, L.off_targets);
    float* so = slot_ptr<float>(ctx, slot, L.off_old);
    float* sr = slot_ptr<float>(ctx, slot, L.off_ref);
    uint8_t* sm = slot_ptr<uint8_t>(ctx, slot, L.off_mask);
    int64_t off = 0;
    for (int i = 0; i < k; ++i) {
      const grpo_group_desc& g = groups[i].desc;
      const int64_t n = groups[i].tokens;
      CU_OK(cudaMemcpyAsync(sh + off * c.d * 2, g.hidden, n * c.d * 2, cudaMemcpyDeviceToDevice, st));
      CU_OK(cudaMemcpyAsync(stg + off, g.targets, n * 4, cudaMemcpyDeviceToDevice, st));
      CU_OK(cudaMemcpyAsync(so + off, g.old_logp, n * 4, cudaMemcpyDeviceToDevice, st));
      if (any_ref) CU_OK(cudaMemcpyAsync(sr + off, g.ref_logp, n * 4, cudaMemcpyDeviceToDevice, st));
      if (any_mask) {
        if (g.mask) CU_OK(cudaMemcpyAsync(sm + off, g.mask, n, cudaMemcpyDeviceToDevice, st));
        else {
          { LaunchScope ls(ctx, GRPO_KERNEL_TOKEN_COUNT, st); fill_u8_kernel<<<64, 256, 0, st>>>(sm + off, n, 1); }
          CU_OK(cudaGetLastError());
        }
      }
      off += n;
    }
    hidden = sh; targets = stg; old_logp = so; ref_logp = any_ref ? sr : nullptr; mask = any_mask ? sm : nullptr;
  }

  GRPO_TRY(grpo_group_advantage(ctx, d_rewards, d_cu_grp, k, 0, d_adv, nullptr, st));

  float* logp = (k == 1 && groups[0].desc.logp_out) ? groups[0].desc.logp_out : slot_ptr<float>(ctx, slot, L.off_logp);
  float* lse = slot_ptr<float>(ctx, slot, L.off_lse);
  float* coeff = slot_ptr<float>(ctx, slot, L.off_coeff);
  void* dh = nullptr;
  if (any_dh) dh = (k == 1) ? groups[0].desc.dhidden_out : static_cast<void*>(slot_ptr<uint8_t>(ctx, slot, L.off_dh));
  if (c.stash_logits) {
    GRPO_TRY(fwd_check(ctx, S, T));
    FwdArgs a{d_cu_seq, S, d_adv, old_logp, ref_logp, mask, loss_denom, denom_dev,
              logp, lse, coeff, loss_accum, metrics_accum};
    a.S_norm = S_update;
    a.T_call = T;
    GRPO_TRY(fwd_counts(ctx, slot, targets, a, st));
    GRPO_TRY(bwd_impl(ctx, slot, hidden, W, targets, lse, coeff, T, 1.0f, dh, dW_accum, st, &a));
  } else {
    GRPO_TRY(fwd_impl(ctx, slot, hidden, W, targets, d_cu_seq, S, T, d_adv, old_logp, ref_logp, mask, loss_denom,
                      denom_dev, logp, lse, coeff, loss_accum, metrics_accum, st, nullptr, S_update));
    GRPO_TRY(bwd_impl(ctx, slot, hidden, W, targets, lse, coeff, T, 1.0f, dh, dW_accum, st));
  }
  if (k > 1) {
    int64_t off = 0;
    for (int i = 0; i < k; ++i) {
      const grpo_group_desc& g = groups[i].desc;
      const int64_t n = groups[i].tokens;
      if (g.dhidden_out)
        CU_OK(cudaMemcpyAsync(g.dhidden_out, static_cast<uint8_t*>(dh) + off * c.d * dh_elem, n * c.d * dh_elem,
                              cudaMemcpyDeviceToDevice, st));
      if (g.logp_out) CU_OK(cudaMemcpyAsync(g.logp_out, logp + off, n * 4, cudaMemcpyDeviceToDevice, st));
      off += n;
    }
  }
  return GRPO_OK;
}

static int32_t drain_one_update(grpo_ctx* ctx, bool flush, const void* W, float* dW_accum, float* loss_accum,
                                float* metrics_accum, double loss_denom, void* const* streams, int32_t n_streams,
                                int32_t* boundary) {
  *boundary = 0;
  if (ctx->update_broken)
    return fail(GRPO_ERR_CUDA, "an earlier launch failed in the middle of a logical update: its partial sums are in the "
                "accumulators and were scaled by that update's denominator; discard the update (zero dW / loss / "
                "metrics), then call grpo_reset_round and resubmit the round's remaining groups");
  if (ctx->fifo.empty()) return GRPO_OK;
  std::vector<int64_t> tokens;
  tokens.reserve(ctx->fifo.size());
  for (const auto& g : ctx->fifo) tokens.push_back(g.tokens);
  std::vector<int> sizes;
  const int take = plan_update(tokens.data(), static_cast<int>(tokens.size()), ctx->cfg.groups_per_update,
                               ctx->cfg.token_budget, flush, sizes);
  if (take == 0) return GRPO_OK;
  if (!W || !loss_accum) return fail(GRPO_ERR_INVALID_ARG, "W / loss_accum is NULL");
  if (n_streams < 1 || n_streams > ctx->n_slots)
    return fail(GRPO_ERR_WORKSPACE, "n_streams=%d but workspace has %d slots", n_streams, ctx->n_slots);
  std::vector<PendingGroup> upd(ctx->fifo.begin(), ctx->fifo.begin() + take);
  // reject the whole update before anything is accumulated: every launch is checked first
  int32_t S_update = 0;
  {
    int pos = 0;
    for (int k : sizes) {
      GRPO_TRY(validate_launch(ctx, upd.data() + pos, k));
      pos += k;
    }
    for (const auto& g : upd) S_update += g.desc.G;
    // data parallelism (loss_agg 1): this rank holds only its share of the update's groups; the per-sequence mean
    // still averages over the sequences of the WHOLE update, which the caller states with grpo_set_seq_denom
    if (ctx->cfg.loss_agg == 1 && ctx->seq_denom > 0) {
      if (ctx->seq_denom < S_update)
        return fail(GRPO_ERR_INVALID_ARG, "grpo_set_seq_denom(%d) is smaller than the %d sequences of this update",
                    ctx->seq_denom, S_update);
      S_update = ctx->seq_denom;
    }
  }

  // implicit denominator of the whole update: count loss-bearing tokens of all its groups first
  const float* denom_dev = nullptr;
  if (ctx->cfg.loss_agg == 0 && !(loss_denom > 0.0)) {   // fp32 count on the device: exact up to 2^24 tokens
    int64_t T_update = 0;
    for (const auto& g : upd) T_update += g.tokens;
    if (T_update > kMaxCountedTokens)
      return fail(GRPO_ERR_SHAPE, "update of %lld tokens: the token-mean denominator is counted in fp32, exact only "
                  "up to 2^24 tokens; pass loss_denom > 0 for an update this large", (long long)T_update);
  }
  if (ctx->cfg.loss_agg == 0 && !(loss_denom > 0.0) && sizes.size() > 1) {
    float* dd = ctx->denom_ring + (ctx->denom_next++ % kDenomRing);
    cudaStream_t s0 = static_cast<cudaStream_t>(streams ? streams[ctx->launches % n_streams] : nullptr);
    CU_OK(cudaMemsetAsync(dd, 0, 4, s0));
    for (const auto& g : upd) {
      {
        LaunchScope ls(ctx, GRPO_KERNEL_TOKEN_COUNT, s0);
        token_count_flat_kernel<<<64, 256, 0, s0>>>(g.desc.mask, g.desc.targets, ctx->cfg.V, g.tokens, dd);
      }
      CU_OK(cudaGetLastError());
    }
    CU_OK(cudaEventRecord(ctx->denom_event, s0));
    for (int i = 0; i < n_streams; ++i)
      if (streams && streams[i] != s0) CU_OK(cudaStreamWaitEvent(static_cast<cudaStream_t>(streams[i]), ctx->denom_event, 0));
    denom_dev = dd;
  }
  int pos = 0;
  for (int k : sizes) {
    const int slot = static_cast<int>(ctx->launches % n_streams);
    cudaStream_t st = static_cast<cudaStream_t>(streams ? streams[slot] : nullptr);
    const int32_t rc = run_launch(ctx, upd.data() + pos, k, W, dW_accum, loss_accum, metrics_accum, loss_denom,
                                  denom_dev, S_update, slot, st);
    if (rc != GRPO_OK) {
      // a device-side failure in the middle of an update (everything checkable was checked above): the groups
      // of the launches that did run are consumed - their gradients are in the accumulators - so that a retry
      // cannot add them twice; the failed launch and the rest of the update stay at the head of the FIFO
      ctx->fifo.erase(ctx->fifo.begin(), ctx->fifo.begin() + pos);
      ctx->consumed += pos;
      // the rest of the update cannot simply be re-planned: it would get a new boundary, denominator and sequence
      // count, and kernels of the failed launch may already have added to the accumulators.  Refuse further
      // dispatch until the caller has discarded the update (grpo_reset_round).
      if (rc == GRPO_ERR_CUDA || pos > 0) ctx->update_broken = true;
      return rc;
    }
    ctx->launches++;
    pos += k;
  }
  ctx->fifo.erase(ctx->fifo.begin(), ctx->fifo.begin() + take);
  ctx->consumed += take;
  *boundary = 1;
  return GRPO_OK;
}

extern "C" int32_t grpo_enqueue_groups(grpo_ctx* ctx, const grpo_group_desc* groups, int32_t n, const void* W,
                                       float* dW_accum, float* loss_accum, float* metrics_accum, double loss_denom,
                                       void* const* streams, int32_t n_streams, int32_t* groups_consumed_out,
                                       int32_t* update_boundary_out) {
  if (!ctx || n < 0 || (n > 0 && !groups)) return fail(GRPO_ERR_INVALID_ARG, "bad ctx / groups / n");
  for (int i = 0; i < n; ++i) GRPO_TRY(validate_group(ctx, groups[i]));
  if (static_cast<int64_t>(ctx->fifo.size()) + n > ctx->cfg.max_pending_groups)
    return fail(GRPO_ERR_QUEUE_FULL, "FIFO holds %zu groups, capacity %d", ctx->fifo.size(), ctx->cfg.max_pending_groups);
  for (int i = 0; i < n; ++i) {
    PendingGroup pg;
    pg.desc = groups[i];
    pg.seqlens.assign(groups[i].seqlens_host, groups[i].seqlens_host + groups[i].G);
    pg.desc.seqlens_host = nullptr;
    pg.tokens = 0;
    for (int32_t l : pg.seqlens) pg.tokens += l;
    ctx->fifo.push_back(std::move(pg));
  }
  int32_t boundary = 0;
  int32_t st = drain_one_update(ctx, false, W, dW_accum, loss_accum, metrics_accum, loss_denom, streams, n_streams, &boundary);
  if (groups_consumed_out) *groups_consumed_out = ctx->consumed;
  if (update_boundary_out) *update_boundary_out = boundary;
  return st;
}

extern "C" int32_t grpo_flush(grpo_ctx* ctx, const void* W, float* dW_accum, float* loss_accum, float* metrics_accum,
                              double loss_denom, void* const* streams, int32_t n_streams, int32_t* groups_consumed_out,
                              int32_t* update_boundary_out) {
  if (!ctx) return fail(GRPO_ERR_INVALID_ARG, "ctx is NULL");
  int32_t boundary = 0;
  int32_t st = drain_one_update(ctx, true, W, dW_accum, loss_accum, metrics_accum, loss_denom, streams, n_streams, &boundary);
  if (groups_consumed_out) *groups_consumed_out = ctx->consumed;
  if (update_boundary_out) *update_boundary_out = boundary;
  return st;
}

// ------------------------------------------------------------------------------------- end to end over host buffers
extern "C" int32_t grpo_step_host(grpo_ctx* ctx, const void* hidden_host, const int32_t* targets_host,
                                  const int32_t* cu_seqlens_host, const float* rewards_host,
                                  const float* old_logp_host, const float* ref_logp_host, const uint8_t* mask_host,
                                  int32_t n_groups, int32_t G, int64_t T, const void* W, float* dW_accum,
                                  double loss_denom, float* loss_host, float* logp_host, void* dhidden_host,
                                  void* stream) {
  if (!ctx || !hidden_host || !targets_host || !cu_seqlens_host || !rewards_host || !old_logp_host || !W || !loss_host)
    return fail(GRPO_ERR_INVALID_ARG, "a required pointer is NULL");
  if (n_groups <= 0 || G <= 0 || T <= 0) return fail(GRPO_ERR_SHAPE, "need n_groups, G, T > 0");
  if (!ctx->ws) return fail(GRPO_ERR_WORKSPACE, "no workspace set (grpo_set_workspace)");
  if (T > ctx->ws_max_T) return fail(GRPO_ERR_WORKSPACE, "T exceeds workspace max_T");
  const grpo_config& c = ctx->cfg;
  const SlotLayout& L = ctx->lay;
  const int S = n_groups * G;
  if (S > L.s_max) return fail(GRPO_ERR_WORKSPACE, "too many sequences");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  uint8_t* sh = slot_ptr<uint8_t>(ctx, 0, L.off_hidden);
  int32_t* stg = slot_ptr<int32_t>(ctx, 0, L.off_targets);
  float* so = slot_ptr<float>(ctx, 0, L.off_old);
  float* sr = slot_ptr<float>(ctx, 0, L.off_ref);
  uint8_t* sm = slot_ptr<uint8_t>(ctx, 0, L.off_mask);
  int32_t* d_cu = slot_ptr<int32_t>(ctx, 0, L.off_cu_seq);
  float* d_rw = slot_ptr<float>(ctx, 0, L.off_rewards);
  float* d_adv = slot_ptr<float>(ctx, 0, L.off_adv);
  float* logp = slot_ptr<float>(ctx, 0, L.off_logp);
  float* lse = slot_ptr<float>(ctx, 0, L.off_lse);
  float* coeff = slot_ptr<float>(ctx, 0, L.off_coeff);
  uint8_t* dh = slot_ptr<uint8_t>(ctx, 0, L.off_dh);
  float* loss_dev = slot_ptr<float>(ctx, 0, L.off_total) + 8;   // scratch scalar inside the 256-byte cell
  // copy pipeline: the hidden states arrive in pieces on the copy stream while the compute stream works.  Pieces:
  // a short first one (so that A2 starts after ~0.15 ms of transfer instead of a whole chunk's 0.7 ms: with the
  // V-only vocab split a launch of a few token tiles still fills the SMs), the rest of backward chunk 0, then one
  // piece per backward chunk.  piece_of_chunk[i] = the last piece backward chunk i needs.
  const int64_t rpc = rows_per_chunk_for(ctx, T);
  const size_t n_chunks = static_cast<size_t>((T + rpc - 1) / rpc);
  const int64_t first_rows = std::min<int64_t>(2048, std::min<int64_t>(rpc, T));
  std::vector<std::pair<int64_t, int64_t>> pieces;             // [begin, end) packed rows
  std::vector<size_t> piece_of_chunk(n_chunks);
  pieces.emplace_back(0, first_rows);
  if (first_rows < std::min<int64_t>(rpc, T)) pieces.emplace_back(first_rows, std::min<int64_t>(rpc, T));
  piece_of_chunk[0] = pieces.size() - 1;
  for (size_t i = 1; i < n_chunks; ++i) {
    pieces.emplace_back(static_cast<int64_t>(i) * rpc, std::min<int64_t>(T, static_cast<int64_t>(i + 1) * rpc));
    piece_of_chunk[i] = pieces.size() - 1;
  }
  HostPipe pipe;
  pipe.cs = ctx->copy_stream;
  pipe.dh_host = static_cast<uint8_t*>(dhidden_host);
  // events live in the context and are created once (1 fence + one per piece + one per chunk of dHidden)
  while (ctx->pipe_events.size() < 1 + pieces.size() + n_chunks) {
    cudaEvent_t e = nullptr;
    CU_OK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    ctx->pipe_events.push_back(e);
  }
  const cudaEvent_t fence = ctx->pipe_events[0];
  const cudaEvent_t* piece_ev = ctx->pipe_events.data() + 1;
  for (size_t i = 0; i < n_chunks; ++i) pipe.in.push_back(piece_ev[piece_of_chunk[i]]);
  if (dhidden_host)
    pipe.out.assign(ctx->pipe_events.begin() + 1 + pieces.size(), ctx->pipe_events.begin() + 1 + pieces.size() + n_chunks);
  // the small per-token arrays go first: they must not queue behind the hidden states on the copy engine
  CU_OK(cudaMemcpyAsync(stg, targets_host, T * 4, cudaMemcpyHostToDevice, st));
  CU_OK(cudaMemcpyAsync(so, old_logp_host, T * 4, cudaMemcpyHostToDevice, st));
  if (ref_logp_host) CU_OK(cudaMemcpyAsync(sr, ref_logp_host, T * 4, cudaMemcpyHostToDevice, st));
  if (mask_host) CU_OK(cudaMemcpyAsync(sm, mask_host, T, cudaMemcpyHostToDevice, st));
  CU_OK(cudaMemcpyAsync(d_cu, cu_seqlens_host, (S + 1) * 4, cudaMemcpyHostToDevice, st));
  CU_OK(cudaMemcpyAsync(d_rw, rewards_host, S * 4, cudaMemcpyHostToDevice, st));
  CU_OK(cudaEventRecord(fence, st));                         // staging buffers are free once st reaches here
  CU_OK(cudaStreamWaitEvent(pipe.cs, fence, 0));
  for (size_t i = 0; i < pieces.size(); ++i) {
    const int64_t t0 = pieces[i].first, rows = pieces[i].second - pieces[i].first;
    CU_OK(cudaMemcpyAsync(sh + t0 * c.d * 2, static_cast<const uint8_t*>(hidden_host) + t0 * c.d * 2, rows * c.d * 2,
                          cudaMemcpyHostToDevice, pipe.cs));
    CU_OK(cudaEventRecord(piece_ev[i], pipe.cs));
  }
  CU_OK(cudaMemsetAsync(loss_dev, 0, 4, st));
  GRPO_TRY(grpo_group_advantage(ctx, d_rw, nullptr, n_groups, G, d_adv, nullptr, st));
  GRPO_TRY(fwd_check(ctx, S, T));
  FwdArgs a{d_cu, S, d_adv, so, ref_logp_host ? sr : nullptr, mask_host ? sm : nullptr, loss_denom, nullptr,
            logp, lse, coeff, loss_dev, nullptr};
  a.T_call = T;
  GRPO_TRY(fwd_counts(ctx, 0, stg, a, st));
  if (c.stash_logits) {
    GRPO_TRY(bwd_impl(ctx, 0, sh, W, stg, lse, coeff, T, 1.0f, dhidden_host ? dh : nullptr, dW_accum, st, &a, &pipe));
  } else {
    for (size_t i = 0; i < pieces.size(); ++i) {             // A2 + A3 piece by piece, as the rows arrive
      CU_OK(cudaStreamWaitEvent(st, piece_ev[i], 0));
      GRPO_TRY(fwd_rows(ctx, 0, sh, W, stg, a, T, pieces[i].first, pieces[i].second - pieces[i].first, nullptr, st));
    }
    GRPO_TRY(bwd_impl(ctx, 0, sh, W, stg, lse, coeff, T, 1.0f, dhidden_host ? dh : nullptr, dW_accum, st, nullptr, &pipe));
  }
  CU_OK(cudaMemcpyAsync(loss_host, loss_dev, 4, cudaMemcpyDeviceToHost, st));
  if (logp_host) CU_OK(cudaMemcpyAsync(logp_host, logp, T * 4, cudaMemcpyDeviceToHost, st));
  CU_OK(cudaStreamSynchronize(pipe.cs));
  CU_OK(cudaStreamSynchronize(st));
  return GRPO_OK;
}

// ------------------------------------------------------------------------------------- diagnostics
extern "C" int32_t grpo_debug_max_active_clusters(grpo_ctx* ctx, int32_t cluster_size, int32_t* clusters_out) {
  if (!ctx || !clusters_out || cluster_size < 1 || cluster_size > 16 || (cluster_size & 1 && cluster_size != 1))
    return fail(GRPO_ERR_INVALID_ARG, "need ctx, clusters_out and cluster_size in {1, 2, 4, ..., 16}");
  auto kern = grpo_gemm_kernel<2, false, false, EPI_LSE>;
  constexpr int smem = GemmShape<2, EPI_RED_F32>::kSmemBytes;
  CU_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  if (cluster_size > 8) CU_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  cudaLaunchConfig_t lc;
  std::memset(&lc, 0, sizeof(lc));
  lc.gridDim = dim3(static_cast<unsigned>(ctx->num_sms / cluster_size * cluster_size * 4));
  lc.blockDim = dim3(kGemmThreads);
  lc.dynamicSmemBytes = smem;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = static_cast<unsigned>(cluster_size);
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  lc.attrs = attr;
  lc.numAttrs = 1;
  int n = 0;
  CU_OK(cudaOccupancyMaxActiveClusters(&n, kern, &lc));
  *clusters_out = n;
  return GRPO_OK;
}

// ------------------------------------------------------------------------------------- test hook
extern "C" int32_t grpo_debug_gemm(grpo_ctx* ctx, int32_t layout, const void* A, const void* B, float* C, int32_t M,
                                   int32_t N, int32_t K, int32_t accumulate, void* stream) {
  if (!ctx || !A || !B || !C) return fail(GRPO_ERR_INVALID_ARG, "NULL pointer");
  if (M <= 0 || N <= 0 || K <= 0 || (M % 8) || (N % 8) || (K % 8)) return fail(GRPO_ERR_SHAPE, "M, N, K must be positive multiples of 8");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  CUtensorMap tmA, tmB;
  GemmParams p;
  std::memset(&p, 0, sizeof(p));
  p.m_total = M; p.n_total = N;
  const int TM = BM * ctx->cg;
  p.m_tiles = (M + TM - 1) / TM; p.n_tiles = (N + BN - 1) / BN; p.k_blocks = (K + BK - 1) / BK;
  p.n_fastest = 1;
  p.c_out = C; p.c_pitch = N;
  if (ctx->ws) p.sync = slot_ptr<unsigned int>(ctx, 0, ctx->lay.off_sync);
  const int units = p.m_tiles * p.n_tiles;
  const bool a_mn = layout == 2, b_mn = layout >= 1;
  if (!a_mn) GRPO_TRY(make_tmap(ctx, &tmA, A, K, M, static_cast<uint64_t>(K) * 2, BK, BM));
  else GRPO_TRY(make_tmap(ctx, &tmA, A, M, K, static_cast<uint64_t>(M) * 2, 64, BK));
  if (!b_mn) GRPO_TRY(make_tmap(ctx, &tmB, B, K, N, static_cast<uint64_t>(K) * 2, BK, BN / ctx->cg));
  else GRPO_TRY(make_tmap(ctx, &tmB, B, N, K, static_cast<uint64_t>(N) * 2, 64, BK));
  CUtensorMap tmCm;
  if (accumulate) GRPO_TRY(make_tmap_c_f32(ctx, &tmCm, C, N, M, static_cast<uint64_t>(N) * 4));
  const CUtensorMap* tmC = accumulate ? &tmCm : nullptr;
  if (layout == 0) {
    if (accumulate) return launch_gemm<false, false, EPI_RED_F32>(ctx, GRPO_KERNEL_DEBUG, tmA, tmB, p, units, st, tmC);
    return launch_gemm<false, false, EPI_STORE>(ctx, GRPO_KERNEL_DEBUG, tmA, tmB, p, units, st);
  } else if (layout == 1) {
    if (accumulate) return launch_gemm<false, true, EPI_RED_F32>(ctx, GRPO_KERNEL_DEBUG, tmA, tmB, p, units, st, tmC);
    return launch_gemm<false, true, EPI_STORE>(ctx, GRPO_KERNEL_DEBUG, tmA, tmB, p, units, st);
  } else if (layout == 2) {
    if (accumulate) return launch_gemm<true, true, EPI_RED_F32>(ctx, GRPO_KERNEL_DEBUG, tmA, tmB, p, units, st, tmC);
    return launch_gemm<true, true, EPI_STORE>(ctx, GRPO_KERNEL_DEBUG, tmA, tmB, p, units, st);
  }
  return fail(GRPO_ERR_INVALID_ARG, "layout must be 0, 1 or 2");
}

// ------------------------------------------------------------------------------------- A3 without any allocation
// grpo_loss_from_partials_static (include/grpo.h): the A3 launch of grpo_loss_from_partials with its scratch - the
// per-block partial sums and arrival counter of the fixed-order loss reduction, the loss-bearing token counts that
// define the mean - in an array that is part of the library image instead of a context's workspace slot.
// Layout of the array (bytes): [0, 256) header {u32 arrival counter, f32 total token count, i32 unread error word};
// then 5 floats per 256-token block; then one float per sequence.
namespace {
constexpr int64_t kStaticMaxBlocks = (GRPO_STATIC_MAX_TOKENS + 255) / 256;
constexpr int64_t kStaticOffPart = 256;
constexpr int64_t kStaticOffSeq = kStaticOffPart + kStaticMaxBlocks * 5 * 4;
constexpr int64_t kStaticBytes = kStaticOffSeq + static_cast<int64_t>(GRPO_STATIC_MAX_SEQUENCES) * 4;
constexpr int kStaticMaxDevices = 64;
}  // namespace

// Every GPU that loads the library carries one copy of this array until the process exits.
static __device__ __align__(256) unsigned char g_static_loss_scratch[kStaticBytes];

// In host code `g_static_loss_scratch` is only a handle for the runtime's symbol table, never a device address: the
// address on the CURRENT device comes from cudaGetSymbolAddress, asked once per device and remembered here.
static void* g_static_scratch_addr[kStaticMaxDevices] = {nullptr};
static std::mutex g_static_scratch_mutex;

static int32_t static_scratch_for_current_device(uint8_t** out) {
  int dev = 0;
  CU_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kStaticMaxDevices) return fail(GRPO_ERR_INVALID_ARG, "device ordinal %d not supported", dev);
  std::lock_guard<std::mutex> guard(g_static_scratch_mutex);
  void* p = g_static_scratch_addr[dev];
  int32_t status = GRPO_OK;
  if (p == nullptr) {   // first call on this device: set-up (do it before any stream capture)
    int major = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) status = fail(GRPO_ERR_CUDA, "cudaDeviceGetAttribute failed: %s", cudaGetErrorString(e));
    else if (major != 10) status = fail(GRPO_ERR_ARCH, "device %d is sm_%dx; this library is built for sm_100a only", dev, major);
    else {
      e = cudaGetSymbolAddress(&p, g_static_loss_scratch);
      if (e != cudaSuccess || p == nullptr)
        status = fail(GRPO_ERR_CUDA, "cudaGetSymbolAddress(g_static_loss_scratch) failed on device %d: %s", dev,
                      cudaGetErrorString(e));
      else g_static_scratch_addr[dev] = p;
    }
  }
  if (status != GRPO_OK) return status;
  *out = static_cast<uint8_t*>(p);
  return GRPO_OK;
}

extern "C" int32_t grpo_loss_from_partials_static(const grpo_config* cfg, int32_t n_shards, const float* m2,
                                                  const float* s2, const float* zy, const int32_t* targets,
                                                  int32_t V_global, const int32_t* cu_seqlens, int32_t S,
                                                  int32_t S_norm, int64_t T, const float* adv, const float* old_logp,
                                                  const float* ref_logp, const uint8_t* mask, double loss_denom,
                                                  float* logp_out, float* lse_out, float* coeff_out, float* loss_accum,
                                                  float* metrics_accum, int32_t* err_flags, void* stream) {
  if (!cfg || !m2 || !s2 || !zy || !targets || !cu_seqlens || !adv || !old_logp || !logp_out || !lse_out || !coeff_out ||
      !loss_accum)
    return fail(GRPO_ERR_INVALID_ARG, "a required pointer is NULL");
  if (n_shards < 1 || V_global < 1 || T <= 0 || S <= 0) return fail(GRPO_ERR_SHAPE, "need n_shards, V_global, T, S > 0");
  if (T > GRPO_STATIC_MAX_TOKENS)
    return fail(GRPO_ERR_WORKSPACE, "T=%lld exceeds GRPO_STATIC_MAX_TOKENS=%d: the built-in scratch array holds no more; "
                "cut the call or use grpo_loss_from_partials with a workspace", (long long)T, GRPO_STATIC_MAX_TOKENS);
  if (S > GRPO_STATIC_MAX_SEQUENCES)
    return fail(GRPO_ERR_WORKSPACE, "S=%d exceeds GRPO_STATIC_MAX_SEQUENCES=%d: the built-in scratch array holds no more; "
                "cut the call or use grpo_loss_from_partials with a workspace", S, GRPO_STATIC_MAX_SEQUENCES);
  if (S_norm != 0 && S_norm < S) return fail(GRPO_ERR_INVALID_ARG, "S_norm=%d is smaller than this call's S=%d", S_norm, S);
  if (cfg->loss_agg != 0 && cfg->loss_agg != 1) return fail(GRPO_ERR_INVALID_ARG, "loss_agg must be 0 or 1");
  if (cfg->kl_type < 0 || cfg->kl_type > 2 || (cfg->dual_clip != 0.f && !(cfg->dual_clip > 1.f)))
    return fail(GRPO_ERR_INVALID_ARG, "kl_type must be 0, 1 or 2 and dual_clip 0 or > 1");
  uint8_t* scratch = nullptr;
  GRPO_TRY(static_scratch_for_current_device(&scratch));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  unsigned int* block_count = reinterpret_cast<unsigned int*>(scratch);
  float* total = reinterpret_cast<float*>(scratch + 4);
  int32_t* err_word = err_flags ? err_flags : reinterpret_cast<int32_t*>(scratch + 8);
  float* block_part = reinterpret_cast<float*>(scratch + kStaticOffPart);
  float* seq_count = reinterpret_cast<float*>(scratch + kStaticOffSeq);
  // the array keeps what the previous call left: the arrival counter and the token total must start at zero (the
  // block sums and per-sequence counts are written before they are read)
  CU_OK(cudaMemsetAsync(scratch, 0, 16, st));
  const bool implicit_denom = cfg->loss_agg == 0 && !(loss_denom > 0.0);
  if (cfg->loss_agg == 1 || implicit_denom) {
    const int threads = 128;
    const int blocks = static_cast<int>((static_cast<int64_t>(S) * 32 + threads - 1) / threads);
    token_count_kernel<<<blocks, threads, 0, st>>>(mask, targets, V_global, cu_seqlens, S, seq_count, total);
    CU_OK(cudaGetLastError());
  }
  LossParams lp;
  std::memset(&lp, 0, sizeof(lp));
  lp.T = T; lp.t_begin = 0; lp.S = S; lp.S_norm = S_norm > 0 ? S_norm : S; lp.V = V_global;
  lp.n_split = n_shards; lp.part_stride = T;
  lp.part_m = m2; lp.part_s = s2; lp.zy = zy; lp.n_zy = n_shards; lp.zy_stride = T;
  lp.targets = targets; lp.cu_seqlens = cu_seqlens; lp.adv = adv; lp.old_logp = old_logp; lp.ref_logp = ref_logp;
  lp.mask = mask; lp.seq_count = seq_count; lp.total_count = total;
  lp.denom_host = loss_denom > 0.0 ? static_cast<float>(loss_denom) : 0.f;
  lp.loss_agg = cfg->loss_agg; lp.clip_lo = cfg->clip_lo; lp.clip_hi = cfg->clip_hi; lp.kl_beta = cfg->kl_beta;
  lp.kl_type = cfg->kl_type; lp.dual_clip = cfg->dual_clip;
  lp.logp = logp_out; lp.lse = lse_out; lp.coeff = coeff_out; lp.loss_accum = loss_accum;
  lp.metrics_accum = metrics_accum; lp.err_flag = err_word;
  lp.block_part = block_part; lp.block_count = block_count;
  const int blocks = static_cast<int>((T + 255) / 256);
  loss_epilogue_kernel<<<blocks, 256, 0, st>>>(lp);
  CU_OK(cudaGetLastError());
  return GRPO_OK;
}
