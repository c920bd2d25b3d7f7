// HBM-bound per-group / per-token kernels of the GRPO step: A1 (group advantage), the mask counts that
// define the mean, and A3 (partial-LSE combine + clipped surrogate + k3 + coefficient for the backward).
#pragma once
#include <cuda_fp16.h>

#include "ptx_sm100.cuh"

namespace grpo {

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float warp_min(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// A1 — Eq. 1: one warp per group; two-pass mean / variance in fp32.
// A group whose rewards are all equal gets advantages that are exactly 0 (max == min test), so the
// zero-advantage path does not depend on the rounding of the mean.
__global__ void group_advantage_kernel(const float* __restrict__ rewards, const int32_t* __restrict__ cu_groups,
                                       int n_groups, int G, float eps_std, int ddof, float* __restrict__ adv,
                                       uint8_t* __restrict__ zero_var) {
  const int g = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (g >= n_groups) return;
  const int beg = cu_groups ? cu_groups[g] : g * G;
  const int end = cu_groups ? cu_groups[g + 1] : beg + G;
  const int n = end - beg;
  float s = 0.f, mx = -INFINITY, mn = INFINITY;
  for (int i = beg + lane; i < end; i += 32) {
    const float r = rewards[i];
    s += r;
    mx = fmaxf(mx, r);
    mn = fminf(mn, r);
  }
  s = warp_sum(s);
  mx = warp_max(mx);
  mn = warp_min(mn);
  const float mu = n > 0 ? s / static_cast<float>(n) : 0.f;
  float ss = 0.f;
  for (int i = beg + lane; i < end; i += 32) {
    const float dlt = rewards[i] - mu;
    ss += dlt * dlt;
  }
  ss = warp_sum(ss);
  const int div = n - ddof;
  const bool flat = !(mx > mn) || div <= 0;
  const float sigma = flat ? 0.f : sqrtf(ss / static_cast<float>(div));
  const float inv = 1.f / (sigma + eps_std);
  for (int i = beg + lane; i < end; i += 32) adv[i] = flat ? 0.f : (rewards[i] - mu) * inv;
  if (zero_var && lane == 0) zero_var[g] = flat ? 1 : 0;
}

// Loss-bearing token counts: per sequence (loss_agg 1) and total (loss_agg 0 with implicit denominator).
// One warp per sequence.  A token counts iff mask != 0 and 0 <= target < V.
__global__ void token_count_kernel(const uint8_t* __restrict__ mask, const int32_t* __restrict__ targets, int V,
                                   const int32_t* __restrict__ cu_seqlens, int S, float* __restrict__ seq_count,
                                   float* __restrict__ total) {
  const int s = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (s >= S) return;
  int c = 0;
  for (int t = cu_seqlens[s] + lane; t < cu_seqlens[s + 1]; t += 32) {
    const int y = targets[t];
    c += ((mask == nullptr || mask[t] != 0) && y >= 0 && y < V) ? 1 : 0;
  }
  const float cf = warp_sum(static_cast<float>(c));
  if (lane == 0) {
    if (seq_count) seq_count[s] = cf;
    if (total) atomicAdd(total, cf);
  }
}

struct LossParams {
  int64_t T;                 // tokens handled by this launch: packed rows [t_begin, t_begin + T)
  int64_t t_begin;
  int S, V;
  int S_norm;                 // loss_agg 1: sequences of the whole logical update (>= S)
  int n_split;
  int64_t part_stride;
  const float* part_m;
  const float* part_s;
  const float* part_u;       // nullable (entropy output)
  const float* zy;           // target logit s z_t[y_t]: n_zy arrays of stride zy_stride are summed (vocab shards:
  int n_zy;                  // exactly one shard holds the target column, the others hold 0)
  int64_t zy_stride;
  const int32_t* targets;
  const int32_t* cu_seqlens;
  const float* adv;
  const float* old_logp;
  const float* ref_logp;     // nullable
  const uint8_t* mask;       // nullable
  const float* seq_count;    // loss_agg 1
  const float* total_count;  // loss_agg 0, implicit denominator (device scalar)
  float denom_host;          // > 0: explicit
  int loss_agg;
  float clip_lo, clip_hi, kl_beta;
  int kl_type;               // 0 = k3, 1 = k1, 2 = k2 (R26)
  float dual_clip;           // 0 = off (R27)
  float* logp;
  float* lse;
  float* coeff;
  float* entropy;            // nullable: per-token policy entropy in nats (R28), every row of the launch
  float* loss_accum;
  float* metrics_accum;      // nullable, [4]
  int32_t* err_flag;
  // fixed-order reduction over the launch's blocks: [gridDim.x][5] partial sums + an arrival counter (self-resetting)
  float* block_part;
  unsigned int* block_count;
};

// A3.  One thread per packed token; block-level reduction; the block sums go to a workspace array and the block
// that arrives last adds them up in block order, so that a launch contributes ONE add per quantity and the scalar
// loss / metrics are bit-reproducible run to run (like every per-token output and, on one stream, dW).
__global__ void __launch_bounds__(256) loss_epilogue_kernel(const LossParams p) {
  const int64_t t = p.t_begin + static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  float loss_t = 0.f, m_cnt = 0.f, m_rho = 0.f, m_k3 = 0.f, m_clip = 0.f;
  if (t < p.t_begin + p.T) {
    // combine the per-split (max, sum 2^(z2 - max)) pairs -> natural-log lse
    const int64_t tl = t - p.t_begin;                 // the A2 launch's own row
    float M = -INFINITY;
    for (int i = 0; i < p.n_split; ++i) M = fmaxf(M, p.part_m[i * p.part_stride + tl]);
    float sum = 0.f;
    for (int i = 0; i < p.n_split; ++i)
      sum += p.part_s[i * p.part_stride + tl] * exp2f(p.part_m[i * p.part_stride + tl] - M);
    const float lse = (M + log2f(sum)) * kLn2;
    if (p.entropy != nullptr && p.part_u != nullptr) {          // entropy = lse - sum_v p_v z_v   (log2 domain, then nats)
      float usum = 0.f;
      for (int i = 0; i < p.n_split; ++i)
        usum += p.part_u[i * p.part_stride + tl] * exp2f(p.part_m[i * p.part_stride + tl] - M);
      p.entropy[t] = ((M + log2f(sum)) - usum / sum) * kLn2;
    }
    const int y = p.targets[t];
    const bool valid = y >= 0 && y < p.V;
    if (y >= p.V) atomicOr(p.err_flag, 1);
    float zy = 0.f;
    if (valid) {
      zy = p.zy[t];
      for (int i = 1; i < p.n_zy; ++i) zy += p.zy[i * p.zy_stride + t];
    }
    const float logp = valid ? zy - lse : 0.f;
    // sequence of this token: largest s with cu_seqlens[s] <= t
    int lo = 0, hi = p.S;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (static_cast<int64_t>(p.cu_seqlens[mid]) <= t) lo = mid; else hi = mid;
    }
    const float A = p.adv[lo];
    const float m = (valid && (p.mask == nullptr || p.mask[t] != 0)) ? 1.f : 0.f;
    float w;
    if (p.loss_agg == 0) {
      const float denom = p.denom_host > 0.f ? p.denom_host : fmaxf(*p.total_count, 1.f);
      w = m / denom;
    } else {
      w = m / (fmaxf(p.seq_count[lo], 1.f) * static_cast<float>(p.S_norm));
    }
    float coeff = 0.f;
    if (m != 0.f) {
      const float rho = expf(logp - p.old_logp[t]);
      const float lo_b = 1.f - p.clip_lo, hi_b = 1.f + p.clip_hi;
      float surr = fminf(rho * A, fminf(fmaxf(rho, lo_b), hi_b) * A);
      bool clipped = (A > 0.f && rho > hi_b) || (A < 0.f && rho < lo_b);
      if (p.dual_clip > 0.f && A < 0.f) {
        surr = fmaxf(surr, p.dual_clip * A);
        clipped = clipped || rho > p.dual_clip;
      }
      float k3 = 0.f, dk3 = 0.f;
      if (p.kl_beta != 0.f && p.ref_logp != nullptr) {
        const float delta = p.ref_logp[t] - logp;
        if (p.kl_type == 1) {
          k3 = -delta;
          dk3 = 1.f;
        } else if (p.kl_type == 2) {
          k3 = 0.5f * delta * delta;
          dk3 = -delta;
        } else {
          const float e = expf(delta);
          k3 = e - delta - 1.f;
          dk3 = 1.f - e;
        }
      }
      loss_t = w * (-surr + p.kl_beta * k3);
      coeff = w * ((clipped ? 0.f : -A * rho) + p.kl_beta * dk3);
      m_cnt = 1.f;
      m_rho = rho;
      m_k3 = k3;
      m_clip = clipped ? 1.f : 0.f;
    }
    p.logp[t] = logp;
    p.lse[t] = lse;
    p.coeff[t] = coeff;
  }
  __shared__ float red[5][8];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float vals[5] = {loss_t, m_cnt, m_rho, m_k3, m_clip};
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const float r = warp_sum(vals[q]);
    if (lane == 0) red[q][warp] = r;
  }
  __syncthreads();
  __shared__ int is_last;
  if (warp == 0) {
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      float r = lane < 8 ? red[q][lane] : 0.f;
      r = warp_sum(r);
      if (lane == 0) p.block_part[blockIdx.x * 5 + q] = r;
    }
    if (lane == 0) {
      __threadfence();
      is_last = atomicAdd(p.block_count, 1u) == gridDim.x - 1 ? 1 : 0;
    }
  }
  __syncthreads();
  if (is_last && warp == 0) {
    __threadfence();
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      float r = 0.f;
      for (unsigned int b = lane; b < gridDim.x; b += 32) r += __ldcg(p.block_part + b * 5 + q);   // fixed order
      r = warp_sum(r);
      if (lane == 0 && r != 0.f) {
        if (q == 0) atomicAdd(p.loss_accum, r);
        else if (p.metrics_accum) atomicAdd(p.metrics_accum + (q - 1), r);
      }
    }
    if (lane == 0) *p.block_count = 0u;           // ready for the slot's next launch (stream-ordered)
  }
}

// Token-granular zero-coefficient compaction.  coeff_t = dloss/dlogp_t is exactly zero for
// masked / ignored tokens, for clipped tokens at kl_beta = 0 (the clipped surrogate has no gradient
// there) and for every token of a zero-variance group at kl_beta = 0; their dZ rows are zero, so the backward
// contractions run only over the other rows.  One block: an order-preserving stream compaction of the call's T
// rows.  row_idx[0 .. n_active) = packed rows with coeff != 0, ascending.  meta[0] = n_active, meta[1] = T,
// meta[2 + c] = rows of backward chunk c = clamp(n_active - c * chunk_rows, 0, chunk_rows) for c < n_chunks.
// stats (nullable): [0] += n_active, [1] += T.
__global__ void __launch_bounds__(1024) compact_rows_kernel(const float* __restrict__ coeff, int T, int chunk_rows,
                                                            int n_chunks, int* __restrict__ row_idx,
                                                            int* __restrict__ meta, long long* __restrict__ stats) {
  __shared__ int warp_cnt[32];
  __shared__ int base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) base_s = 0;
  __syncthreads();
  for (int t0 = 0; t0 < T; t0 += 1024) {
    const int t = t0 + threadIdx.x;
    const bool act = t < T && coeff[t] != 0.f;
    const unsigned bal = __ballot_sync(0xffffffffu, act);
    if (lane == 0) warp_cnt[warp] = __popc(bal);
    __syncthreads();
    int before = 0, total = 0;
#pragma unroll
    for (int w = 0; w < 32; ++w) {
      const int c = warp_cnt[w];
      before += w < warp ? c : 0;
      total += c;
    }
    const int base = base_s;
    if (act) row_idx[base + before + __popc(bal & ((1u << lane) - 1u))] = t;
    __syncthreads();
    if (threadIdx.x == 0) base_s = base + total;
  }
  __syncthreads();
  const int n_active = base_s;
  if (threadIdx.x == 0) {
    meta[0] = n_active;
    meta[1] = T;
    if (stats) { atomicAdd(reinterpret_cast<unsigned long long*>(stats), static_cast<unsigned long long>(n_active));
                 atomicAdd(reinterpret_cast<unsigned long long*>(stats + 1), static_cast<unsigned long long>(T)); }
  }
  for (int c = threadIdx.x; c < n_chunks; c += blockDim.x)
    meta[2 + c] = max(0, min(chunk_rows, n_active - c * chunk_rows));
}

// Gather one backward chunk of active rows: Hc[r,:] = H[row_idx[r],:] and the per-row inputs of the dZ epilogue
// (target, lse, coeff) for r < rows = *dyn_rows; rows [rows, round_up(rows, tile_rows)) are zero-filled (zero
// hidden state, coeff 0, target -1): they are the tail of the last token tile A4 walks and of the last k block
// A6 reduces over.  One block per destination row; 16-byte accesses (d % 8 == 0).
__global__ void __launch_bounds__(128) gather_rows_kernel(const uint4* __restrict__ H, int64_t row_vec /* d / 8 */,
                                                          const int* __restrict__ row_idx,
                                                          const int* __restrict__ dyn_rows, int tile_rows,
                                                          int rows_alloc, const int32_t* __restrict__ targets,
                                                          const float* __restrict__ lse, const float* __restrict__ coeff,
                                                          uint4* __restrict__ Hc, int32_t* __restrict__ yc,
                                                          float* __restrict__ lsec, float* __restrict__ coeffc) {
  const int r = blockIdx.x;
  const int rows = *dyn_rows;
  const int rows_pad = min(rows_alloc, (rows + tile_rows - 1) / tile_rows * tile_rows);
  if (r >= rows_pad) return;
  uint4* dst = Hc + static_cast<int64_t>(r) * row_vec;
  if (r < rows) {
    const int t = row_idx[r];
    const uint4* src = H + static_cast<int64_t>(t) * row_vec;
    for (int64_t i = threadIdx.x; i < row_vec; i += blockDim.x) dst[i] = src[i];
    if (threadIdx.x == 0) { yc[r] = targets[t]; lsec[r] = lse[t]; coeffc[r] = coeff[t]; }
  } else {
    for (int64_t i = threadIdx.x; i < row_vec; i += blockDim.x) dst[i] = make_uint4(0u, 0u, 0u, 0u);
    if (threadIdx.x == 0) { yc[r] = -1; lsec[r] = 0.f; coeffc[r] = 0.f; }
  }
}

// Split-K reduction of A5 (and the scatter of compacted rows back to their packed positions):
// out[dst(r), :] = ((part_0[r,:] + part_1[r,:]) + part_2[r,:]) + ...   in that fixed order, r < rows.
// dst(r) = row_idx[r] if row_idx != nullptr, else r.  One block per row; 16-byte accesses.
__global__ void __launch_bounds__(128) splitk_reduce_kernel(const float4* __restrict__ parts, int k_split,
                                                            int64_t split_stride_vec, int64_t row_vec /* d / 4 */,
                                                            int rows_static, const int* __restrict__ dyn_rows,
                                                            const int* __restrict__ row_idx,
                                                            void* __restrict__ out, int out_fp32) {
  const int r = blockIdx.x;
  const int rows = dyn_rows ? min(rows_static, *dyn_rows) : rows_static;
  if (r >= rows) return;
  const int64_t dst_row = row_idx ? row_idx[r] : r;
  const float4* src = parts + static_cast<int64_t>(r) * row_vec;
  for (int64_t i = threadIdx.x; i < row_vec; i += blockDim.x) {
    float4 a = src[i];
    for (int k = 1; k < k_split; ++k) {
      const float4 b = src[k * split_stride_vec + i];
      a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w;
    }
    if (out_fp32) {
      reinterpret_cast<float4*>(out)[dst_row * row_vec + i] = a;
    } else {
      reinterpret_cast<uint2*>(out)[dst_row * row_vec + i] = make_uint2(pack_bf16x2(a.x, a.y), pack_bf16x2(a.z, a.w));
    }
  }
}

// dHidden rows of tokens with a zero coefficient are zeros (what the dense A5 gives for an all-zero dZ row).
// One block per packed row; 16-byte stores (row_bytes % 16 == 0).
__global__ void __launch_bounds__(128) zero_coeff_rows_kernel(const float* __restrict__ coeff, int T,
                                                              uint8_t* __restrict__ out, int64_t row_bytes) {
  const int t = blockIdx.x;
  if (t >= T || coeff[t] != 0.f) return;
  uint4* dst = reinterpret_cast<uint4*>(out + static_cast<int64_t>(t) * row_bytes);
  for (int64_t i = threadIdx.x; i < row_bytes / 16; i += blockDim.x) dst[i] = make_uint4(0u, 0u, 0u, 0u);
}

// ------------------------------------------------------------------------------------------------------------
// NEXT-4 (R29-R31): the final RMSNorm in front of the path.
__device__ __forceinline__ float4 bf16x4_to_float4(uint2 v) {
  float4 f;
  f.x = __uint_as_float(v.x << 16);
  f.y = __uint_as_float(v.x & 0xffff0000u);
  f.z = __uint_as_float(v.y << 16);
  f.w = __uint_as_float(v.y & 0xffff0000u);
  return f;
}

// H[t,:] = bf16(gamma * x[t,:] * rstd_t),  rstd_t = 1 / sqrt(mean_k x_tk^2 + eps)   (fp32 arithmetic, one rounding).
// One warp per row, 8-byte loads (4 bf16); the second pass re-reads the row from L1.  HBM-bound: 2 d bytes read +
// 2 d bytes written per token.
__global__ void __launch_bounds__(256) rmsnorm_fwd_kernel(const uint2* __restrict__ x, const uint2* __restrict__ gamma,
                                                          int64_t T, int row_vec /* d / 4 */, float inv_d, float eps,
                                                          uint2* __restrict__ H, float* __restrict__ rstd_out) {
  const int lane = threadIdx.x & 31;
  const int64_t warps = static_cast<int64_t>(gridDim.x) * (blockDim.x >> 5);
  for (int64_t t = static_cast<int64_t>(blockIdx.x) * (blockDim.x >> 5) + (threadIdx.x >> 5); t < T; t += warps) {
    const uint2* row = x + t * row_vec;
    float ss = 0.f;
    for (int i = lane; i < row_vec; i += 32) {
      const float4 v = bf16x4_to_float4(row[i]);
      ss = fmaf(v.x, v.x, fmaf(v.y, v.y, fmaf(v.z, v.z, fmaf(v.w, v.w, ss))));
    }
    ss = warp_sum(ss);
    const float rstd = 1.f / sqrtf(ss * inv_d + eps);
    if (lane == 0) rstd_out[t] = rstd;
    uint2* dst = H + t * row_vec;
    for (int i = lane; i < row_vec; i += 32) {
      const float4 v = bf16x4_to_float4(row[i]);
      const float4 g = bf16x4_to_float4(gamma[i]);
      dst[i] = make_uint2(pack_bf16x2(g.x * (v.x * rstd), g.y * (v.y * rstd)),
                          pack_bf16x2(g.z * (v.z * rstd), g.w * (v.w * rstd)));
    }
  }
}

// RMSNorm backward, fused behind A5: the split-K reduction of the dHidden row (fixed order, fp32) is followed in
// registers by   g = gamma * dH,  xh = x rstd,  dx = rstd (g - xh mean_k(g xh)),  dgamma += dH * xh,
// so dHidden is never written: the row goes straight to dx (scattered to its packed position under compaction).
// IN_BF16: `parts` is a bf16 [rows, d] dHidden instead (the standalone grpo_rmsnorm_bwd; k_split = 1).
// Blocks loop over rows and keep their dgamma partial sums in registers (J float4 per thread: d <= 1024 J), then
// add them to dgamma_accum with one atomic per column and block.
template <int J, bool IN_BF16>
__global__ void __launch_bounds__(256) prenorm_bwd_kernel(const void* __restrict__ parts, int k_split,
                                                          int64_t split_stride_vec, int row_vec /* d / 4 */,
                                                          int rows_static, const int* __restrict__ dyn_rows,
                                                          const int* __restrict__ row_idx, int64_t row0,
                                                          const uint2* __restrict__ x, const uint2* __restrict__ gamma,
                                                          const float* __restrict__ rstd, float inv_d,
                                                          void* __restrict__ dx_out, int out_fp32,
                                                          float* __restrict__ dgamma_accum) {
  __shared__ float red[8];
  const int rows = dyn_rows ? min(rows_static, *dyn_rows) : rows_static;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float4 acc[J], gm[J];
#pragma unroll
  for (int j = 0; j < J; ++j) {
    acc[j] = make_float4(0.f, 0.f, 0.f, 0.f);
    const int i = threadIdx.x + j * 256;
    gm[j] = i < row_vec ? bf16x4_to_float4(gamma[i]) : make_float4(0.f, 0.f, 0.f, 0.f);
  }
  for (int r = blockIdx.x; r < rows; r += gridDim.x) {
    const int64_t t = row_idx ? row_idx[r] : row0 + r;           // packed row of the call
    const float rs = rstd[t];
    float4 dh[J], xh[J];
    float dot = 0.f;
#pragma unroll
    for (int j = 0; j < J; ++j) {
      const int i = threadIdx.x + j * 256;
      dh[j] = make_float4(0.f, 0.f, 0.f, 0.f);
      xh[j] = dh[j];
      if (i < row_vec) {
        if constexpr (IN_BF16) {
          dh[j] = bf16x4_to_float4(reinterpret_cast<const uint2*>(parts)[static_cast<int64_t>(r) * row_vec + i]);
        } else {
          const float4* src = reinterpret_cast<const float4*>(parts) + static_cast<int64_t>(r) * row_vec + i;
          dh[j] = src[0];
          for (int k = 1; k < k_split; ++k) {
            const float4 b = src[k * split_stride_vec];
            dh[j].x += b.x; dh[j].y += b.y; dh[j].z += b.z; dh[j].w += b.w;
          }
        }
        const float4 xv = bf16x4_to_float4(x[t * row_vec + i]);
        xh[j] = make_float4(xv.x * rs, xv.y * rs, xv.z * rs, xv.w * rs);
        dot += gm[j].x * dh[j].x * xh[j].x + gm[j].y * dh[j].y * xh[j].y + gm[j].z * dh[j].z * xh[j].z +
               gm[j].w * dh[j].w * xh[j].w;
      }
    }
    dot = warp_sum(dot);
    __syncthreads();                                             // red[] of the previous row has been read
    if (lane == 0) red[warp] = dot;
    __syncthreads();
    float mean = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) mean += red[w];
    mean *= inv_d;
#pragma unroll
    for (int j = 0; j < J; ++j) {
      const int i = threadIdx.x + j * 256;
      if (i < row_vec) {
        const float4 o = make_float4(rs * (gm[j].x * dh[j].x - xh[j].x * mean), rs * (gm[j].y * dh[j].y - xh[j].y * mean),
                                     rs * (gm[j].z * dh[j].z - xh[j].z * mean), rs * (gm[j].w * dh[j].w - xh[j].w * mean));
        if (out_fp32) reinterpret_cast<float4*>(dx_out)[t * row_vec + i] = o;
        else reinterpret_cast<uint2*>(dx_out)[t * row_vec + i] = make_uint2(pack_bf16x2(o.x, o.y), pack_bf16x2(o.z, o.w));
        acc[j].x = fmaf(dh[j].x, xh[j].x, acc[j].x);
        acc[j].y = fmaf(dh[j].y, xh[j].y, acc[j].y);
        acc[j].z = fmaf(dh[j].z, xh[j].z, acc[j].z);
        acc[j].w = fmaf(dh[j].w, xh[j].w, acc[j].w);
      }
    }
  }
#pragma unroll
  for (int j = 0; j < J; ++j) {
    const int i = threadIdx.x + j * 256;
    if (i < row_vec && static_cast<int>(blockIdx.x) < rows) {
      atomicAdd(dgamma_accum + 4 * i + 0, acc[j].x);
      atomicAdd(dgamma_accum + 4 * i + 1, acc[j].y);
      atomicAdd(dgamma_accum + 4 * i + 2, acc[j].z);
      atomicAdd(dgamma_accum + 4 * i + 3, acc[j].w);
    }
  }
}

// ------------------------------------------------------------------------------------------------------------
// FP8 precision study: e4m3 operands for the two logit
// contractions (A2, A4).  Hidden rows get one scale each (amax / 448), the vocab matrix one scale for the tensor.
__global__ void __launch_bounds__(256) amax_kernel(const uint2* __restrict__ x, int64_t n_vec,
                                                   unsigned int* __restrict__ amax_bits) {
  float m = 0.f;
  for (int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < n_vec;
       i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
    const float4 v = bf16x4_to_float4(x[i]);
    m = fmaxf(fmaxf(m, fmaxf(fabsf(v.x), fabsf(v.y))), fmaxf(fabsf(v.z), fabsf(v.w)));
  }
  m = warp_max(m);
  if ((threadIdx.x & 31) == 0) atomicMax(amax_bits, __float_as_uint(m));   // non-negative floats order like uints
}
__global__ void scale_from_amax_kernel(const unsigned int* __restrict__ amax_bits, float* __restrict__ scale) {
  const float a = __uint_as_float(*amax_bits);
  *scale = a > 0.f ? a * (1.f / 448.f) : 1.f;
}
// q[r,:] = e4m3(x[r,:] / s_r).  fixed_scale != nullptr: s_r = *fixed_scale for every row (per-tensor); else
// s_r = amax_r / 448 (1 for an all-zero row), written to scale_out[r].  One warp per row.
__global__ void __launch_bounds__(256) quantize_rows_e4m3_kernel(const uint2* __restrict__ x, int64_t R, int row_vec,
                                                                 uint32_t* __restrict__ q, float* __restrict__ scale_out,
                                                                 const float* __restrict__ fixed_scale) {
  const int lane = threadIdx.x & 31;
  const int64_t warps = static_cast<int64_t>(gridDim.x) * (blockDim.x >> 5);
  for (int64_t r = static_cast<int64_t>(blockIdx.x) * (blockDim.x >> 5) + (threadIdx.x >> 5); r < R; r += warps) {
    const uint2* row = x + r * row_vec;
    float s;
    if (fixed_scale != nullptr) {
      s = *fixed_scale;
    } else {
      float m = 0.f;
      for (int i = lane; i < row_vec; i += 32) {
        const float4 v = bf16x4_to_float4(row[i]);
        m = fmaxf(fmaxf(m, fmaxf(fabsf(v.x), fabsf(v.y))), fmaxf(fabsf(v.z), fabsf(v.w)));
      }
      m = warp_max(m);
      s = m > 0.f ? m * (1.f / 448.f) : 1.f;
      if (lane == 0) scale_out[r] = s;
    }
    const float inv = 1.f / s;
    uint32_t* dst = q + r * row_vec;
    for (int i = lane; i < row_vec; i += 32) {
      const float4 v = bf16x4_to_float4(row[i]);
      dst[i] = pack_e4m3x2(v.x * inv, v.y * inv) | (pack_e4m3x2(v.z * inv, v.w * inv) << 16);
    }
  }
}

// 3-contraction variant: turn the stashed exponentials e = 2^(z2 - m) (fp16, written by the
// EPI_LSE_STASH epilogue together with m per (row, 256-column tile) in `shift`) into
// dZ = k_t (1[v = y_t] - e 2^(m - lse2_t)) (bf16); k_t = coeff_t * coeff_mul.  HBM-bound: 2 B read + 2 B written
// per logit.  One block per row; 16-byte accesses; one ex2 per 8 logits.
// row_idx == nullptr: in place, every row of the chunk.  row_idx != nullptr (zero-coefficient compaction, DESIGN.md
// section 10): destination row r < *dyn_rows is built from stash row row_idx[r] (chunk-local) and written to `out`,
// a second chunk buffer; rows [*dyn_rows, round_up(*dyn_rows, tile_rows)) of `out` are zero-filled (the tail of the
// last token tile A5 walks and of the last k block A6 reduces over).
__global__ void __launch_bounds__(256) stash_to_dz_kernel(const uint16_t* stash, uint16_t* out /* may alias stash */,
                                                          int rows_static, int V, int64_t pitch,
                                                          const float* __restrict__ shift, int64_t shift_pitch,
                                                          int tile_cols, const int32_t* __restrict__ targets,
                                                          const float* __restrict__ lse, const float* __restrict__ coeff,
                                                          float coeff_mul, const int* __restrict__ row_idx,
                                                          const int* __restrict__ dyn_rows, int tile_rows, int rows_alloc) {
  const int r = blockIdx.x;
  const int n_vec = (V + 7) / 8;
  int src = r;
  if (row_idx != nullptr) {
    const int rows = *dyn_rows;
    if (r >= min(rows_alloc, (rows + tile_rows - 1) / tile_rows * tile_rows)) return;
    if (r >= rows) {
      uint4* z = reinterpret_cast<uint4*>(out + static_cast<int64_t>(r) * pitch);
      for (int i = threadIdx.x; i < n_vec; i += blockDim.x) z[i] = make_uint4(0u, 0u, 0u, 0u);
      return;
    }
    src = row_idx[r];
  } else if (r >= rows_static) {
    return;
  }
  const float lse2 = lse[src] * kLog2e;
  const float k = coeff[src] * coeff_mul;
  int y = targets[src];
  if (y >= V) y = -1;
  const uint4* line = reinterpret_cast<const uint4*>(stash + static_cast<int64_t>(src) * pitch);
  uint4* dst = reinterpret_cast<uint4*>(out + static_cast<int64_t>(r) * pitch);
  const float* sh = shift + static_cast<int64_t>(src) * shift_pitch;
  for (int i = threadIdx.x; i < n_vec; i += blockDim.x) {
    const uint4 in = line[i];
    const float f = -k * ex2_approx(sh[i * 8 / tile_cols] - lse2);      // - k 2^(m - lse2) <= k in magnitude
    const uint32_t w4[4] = {in.x, in.y, in.z, in.w};
    float dz[8];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const float2 e = __half22float2(*reinterpret_cast<const __half2*>(&w4[j]));
      dz[2 * j] = f * e.x;
      dz[2 * j + 1] = f * e.y;
    }
    if (static_cast<uint32_t>(y - i * 8) < 8u) {
#pragma unroll
      for (int j = 0; j < 8; ++j) dz[j] = (y - i * 8 == j) ? dz[j] + k : dz[j];
    }
    dst[i] = make_uint4(pack_bf16x2(dz[0], dz[1]), pack_bf16x2(dz[2], dz[3]), pack_bf16x2(dz[4], dz[5]),
                        pack_bf16x2(dz[6], dz[7]));
  }
}

}  // namespace grpo
