/*
 * grpo.h — C ABI of the B200 (sm_100a) fused GRPO policy-loss step.
 *
 * The trainer-side hot path that RolloutPipe's complete-group pipelining (CGP) feeds
 * (arxiv/paper_2606_26997; citations are PAPER.md line numbers):
 *
 *   A0  CGP handoff: FIFO of complete groups, feasible prefix under a token budget, dispatch in
 *       logical updates of U groups                       PAPER.md:92, 111, 187; Alg. 1 l.16-22
 *   A1  group-relative advantage  A_i = (r_i - mu_g)/(sigma_g + eps_std)      Eq. 1
 *   A2  LM-head contraction + online log-sum-exp + target gather  -> logp_t    ("Megatron executes
 *       forward"; definition: BASELINE.json north_star)
 *   A3  clipped importance-ratio surrogate + optional k3 KL + masked mean (loss mask,
 *       PAPER.md:40)
 *   A4-A6 backward: recompute logits chunk, dZ = c_t (1[v=y_t] - p_tv), dH = dZ W, dW += dZ^T H
 *   A7  gradients / loss only ever ACCUMULATE until the caller's optimizer boundary
 *
 * Conventions
 *   - Every function returns a grpo_status (int32).  No exception crosses the ABI.
 *     grpo_last_error() gives a thread-local message for the last non-OK status on this thread.
 *   - Unless a parameter says HOST, tensor pointers are DEVICE pointers owned by the caller and must
 *     stay valid until the stream reaches the work of the call.  The library owns only its context.
 *   - No function synchronises the host with the device unless its name ends in _sync or _host.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - Layouts: hidden bf16 [T, d] row-major; W bf16 [V, d] row-major; dW fp32 [V, d] row-major;
 *     per-token arrays are [T] over the PACKED token stream; cu_seqlens int32 [S+1] gives sequence
 *     boundaries in that stream.  Row t of `hidden` is the state that predicts targets[t]
 *     (caller pre-shifts; only loss-bearing positions are packed).
 *   - Requirements: d % 8 == 0, V >= 1, T >= 1, hidden/W/dW 16-byte aligned.  Otherwise GRPO_ERR_SHAPE.
 *   - Device arch must be sm_100; otherwise GRPO_ERR_ARCH.  There is no CPU or other-GPU fallback.
 */
#ifndef GRPO_B200_H_
#define GRPO_B200_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  GRPO_OK = 0,
  GRPO_ERR_INVALID_ARG = 1,
  GRPO_ERR_SHAPE = 2,
  GRPO_ERR_WORKSPACE = 3,
  GRPO_ERR_ARCH = 4,
  GRPO_ERR_CUDA = 5,
  GRPO_ERR_INCOMPLETE_GROUP = 6,
  GRPO_ERR_QUEUE_FULL = 7
} grpo_status;

typedef struct grpo_ctx grpo_ctx;

typedef struct {
  int32_t d;                 /* hidden width */
  int32_t V;                 /* vocabulary size */
  float   eps_std;           /* Eq. 1 stabiliser; 1e-6 */
  int32_t std_ddof;          /* 0: population sigma (default reading of PAPER.md:90), 1: sample sigma */
  float   clip_lo, clip_hi;  /* ratio clipped to [1-clip_lo, 1+clip_hi]; 0.2 / 0.28 */
  float   kl_beta;           /* weight of the k3 term; 0 disables it */
  int32_t loss_agg;          /* 0: token mean over the logical update; 1: per-sequence mean, then mean over sequences */
  float   logit_scale;       /* 1 / temperature; 1 */
  int32_t dhidden_fp32;      /* 0: dHidden written as bf16, 1: fp32 */
  int32_t group_size;        /* K: responses per complete group; 0 = do not check */
  int32_t groups_per_update; /* U = B/K; >= 1 */
  int32_t groups_per_round;  /* R; 0 = unknown (round-complete flag never raised) */
  int64_t token_budget;      /* feasible-batch token budget per launch; 0 = unlimited */
  int64_t bwd_chunk_tokens;  /* tokens per backward dZ chunk; 0 = default (9472) */
  int32_t max_pending_groups;/* FIFO capacity; 0 = default (4096) */
  int32_t gemm_cta_group;    /* CTAs cooperating on one tcgen05 MMA: 0 = default (2: CTA pairs, 256x256 pair
                                tiles), 1 = single-CTA 128x256 tiles (kept as an A/B reference) */
  int32_t gemm_drift_epoch_kb; /* drift gate of the contraction kernels: the CTA pairs of a launch stay within
                                one epoch of this many k blocks of each other so that the operand panels they
                                share are fetched from HBM once.  0 = default (32),
                                < 0 = off.  Performance only: results do not depend on it. */
  int32_t kl_type;           /* KL estimator weighted by kl_beta (R8, R26): 0 = k3 (default),
                                1 = k1 = logp - ref, 2 = k2 = (logp - ref)^2 / 2 */
  float   dual_clip;         /* 0 = off; c > 1: for A < 0 the surrogate is max(min(rho A, clip(rho) A), c A)
                                (R27) */
  int32_t bwd_skip_zero_tiles; /* 0 = default (on), < 0 = off.  The backward skips every token whose coefficient
                                dloss/dlogp is exactly zero (masked or ignored tokens; at kl_beta = 0 also clipped
                                tokens, and zero-variance groups): the remaining rows are compacted
                                on the device and A4-A6 run on the compact panel; skipped dHidden rows are
                                written as zeros and add nothing to dW, which is what the dense computation
                                gives.  Decided on the device; no host synchronisation. */
  int32_t stash_logits;      /* 0 = default: grpo_enqueue_groups / grpo_step_host run forward then backward with
                                the logits RECOMPUTED chunk by chunk (north_star, 4 contractions); 1 = they run
                                grpo_fused_logprob_loss_fwd_bwd instead (3 contractions) */
  int32_t fp8_logits;        /* 0 = default (bf16).  1 = FP8 PRECISION STUDY (DESIGN.md
                                section 13): the two logit contractions (A2 and the A4 recompute) run on e4m3 operands
                                (tcgen05 kind::f8f6f4, twice the bf16 tensor rate): every hidden row is quantised with
                                its own scale amax/448, the vocab matrix with one scale for the tensor, both folded
                                into the epilogue; dZ, A5 and A6 stay bf16 x bf16 -> fp32.  Log-probs then carry the
                                e4m3 rounding of the operands (2^-4 relative per element): this does NOT meet
                                north_star's 2e-3 log-prob tolerance and is never the default or the headline.
                                Needs d % 16 == 0; not with stash_logits. */
  int32_t gemm_max_ctas;     /* 0 = default: the persistent contraction kernels take every SM of the device.  n > 0:
                                at most n CTAs (rounded down to whole CTA pairs), which leaves the other SMs to a
                                kernel running concurrently on another stream — the all-reduce of the data-parallel
                                update boundary.  Results do not depend on it bit for bit
                                (every reduction is cut by the problem's shape alone). */
} grpo_config;

/* Fill *cfg with the defaults above (d, V must still be set). */
int32_t grpo_default_config(grpo_config* cfg);

/* Create / destroy a context on the CURRENT CUDA device.  HOST pointers. */
int32_t grpo_create(const grpo_config* cfg, grpo_ctx** out);
int32_t grpo_destroy(grpo_ctx* ctx);

/* Thread-local, never NULL; valid until the next failing call on this thread. */
const char* grpo_last_error(void);

/* Bytes of ONE workspace slot able to process launches of up to max_T packed tokens. */
int32_t grpo_workspace_bytes(const grpo_ctx* ctx, int64_t max_T, int64_t* bytes_out /*HOST*/);

/* Hand the library n_slots workspace slots (caller-allocated device memory, 256-byte aligned,
 * bytes >= n_slots * grpo_workspace_bytes(max_T)).  Direct fwd/bwd calls use slot 0 and must
 * not run concurrently with each other; grpo_enqueue_groups uses slot (stream index). */
int32_t grpo_set_workspace(grpo_ctx* ctx, void* dev_ptr, int64_t bytes, int64_t max_T, int32_t n_slots);

/* A1 — Eq. 1.  rewards fp32 [S]; groups are [cu_groups[g], cu_groups[g+1]) if
 * cu_groups (int32 [n_groups+1], device) is given, else uniform of size G.  adv_out fp32 [S];
 * zero_var_out u8 [n_groups] or NULL (1 where all rewards of the group are equal => advantages are
 * exactly 0).  One warp per group. */
int32_t grpo_group_advantage(grpo_ctx* ctx, const float* rewards, const int32_t* cu_groups, int32_t n_groups,
                             int32_t G, float* adv_out, uint8_t* zero_var_out, void* stream);

/* A2 + A3.  targets int32 [T] (<0: token ignored; >=V: ignored and an error bit is raised, see
 * grpo_check_errors_sync).  adv fp32 [S].  old_logp fp32 [T].  ref_logp fp32 [T] or NULL (no KL).
 * mask u8 [T] or NULL (all ones).  loss_denom > 0: explicit denominator of the whole logical update
 * (loss_agg 0); <= 0: max(sum of this call's mask, 1), counted on the device in fp32 - exact up to 2^24 tokens, so a
 * call (or a grpo_enqueue_groups update) of more than 16 777 216 tokens without an explicit loss_denom is
 * GRPO_ERR_SHAPE and nothing runs.
 * Outputs: logp_out, lse_out, coeff_out fp32 [T] (coeff_t = d loss / d logp_t, consumed by bwd);
 * loss_accum fp32 [1] is ADDED to; metrics_accum fp32 [4] or NULL is ADDED to:
 * {loss-bearing tokens, sum rho, sum k3, tokens whose policy gradient is clipped}. */
int32_t grpo_fused_logprob_loss_fwd(grpo_ctx* ctx, const void* hidden, const void* W, const int32_t* targets,
                                    const int32_t* cu_seqlens, int32_t S, int64_t T, const float* adv,
                                    const float* old_logp, const float* ref_logp, const uint8_t* mask,
                                    double loss_denom, float* logp_out, float* lse_out, float* coeff_out,
                                    float* loss_accum, float* metrics_accum, void* stream);

/* loss_agg = 1 only (per-sequence mean, then mean over sequences): the number of sequences of the WHOLE logical
 * update that later grpo_fused_logprob_loss_fwd / _fwd_bwd calls of this context divide by, for callers that cut
 * one update into several calls (micro-batches); 0 (default) = each call's own S.  grpo_enqueue_groups / grpo_flush
 * count the sequences of the update's groups themselves (R10) while this is 0; a data-parallel rank, which
 * holds only its share of the update's groups, sets the update's GLOBAL sequence count here before it enqueues
 * them (an update with more local sequences than the stated count is GRPO_ERR_INVALID_ARG and nothing runs). */
int32_t grpo_set_seq_denom(grpo_ctx* ctx, int32_t n_sequences);

/* ---- NEXT-3(b): vocab-parallel (tensor-parallel) forward -------------------------
 * The paper's trainer ran TP = 4, which shards W by rows.  Rank r holds W_shard = W[v0_r : v1_r, :]
 * and a context created with V = v1_r - v0_r.
 *
 * grpo_vocab_shard_partials: A2 on the shard.  targets_local[t] = y_t - v0_r (any value outside [0, V_shard) means
 * the target column lives in another shard).  Outputs, fp32 [T]: m2_out / s2_out = running maximum and sum of
 * 2^(z2 - m2) over the shard's columns in the log2 domain (z2 = s z log2 e), zy_out = s z_t[y_t] where this shard
 * holds the target column, else 0.  The three arrays are what the ranks exchange (one all-gather of [T] x 3 fp32).
 *
 * grpo_loss_from_partials: A3 on the gathered partials [n_shards, T] (shard-major): combines them in shard order into
 * lse / logp and runs the loss arithmetic of grpo_fused_logprob_loss_fwd (same arguments; targets are GLOBAL ids,
 * V_global the full vocabulary).  Every rank then calls grpo_fused_logprob_loss_bwd on its shard with targets_local,
 * the global lse and coeff: dW_accum is the shard's rows of dW, and dhidden_out the shard's PARTIAL dHidden, which
 * the ranks sum (all-reduce of [T, d]).  DESIGN.md section 7. */
int32_t grpo_vocab_shard_partials(grpo_ctx* ctx, const void* hidden, const void* W_shard, const int32_t* targets_local,
                                  int64_t T, float* m2_out, float* s2_out, float* zy_out, void* stream);
int32_t grpo_loss_from_partials(grpo_ctx* ctx, int32_t n_shards, const float* m2, const float* s2, const float* zy,
                                const int32_t* targets, int32_t V_global, const int32_t* cu_seqlens, int32_t S, int64_t T,
                                const float* adv, const float* old_logp, const float* ref_logp, const uint8_t* mask,
                                double loss_denom, float* logp_out, float* lse_out, float* coeff_out, float* loss_accum,
                                float* metrics_accum, void* stream);

/* ---- A3 for callers that must not allocate -----------------------------------------------------------------
 * Everything above needs a context (grpo_create calls cudaMalloc / cudaMallocHost) and a workspace the caller has to
 * allocate.  Some callers cannot do either at the point where they need the loss: a trainer whose framework has
 * already handed the whole of HBM to its own caching allocator (a raw cudaMalloc then fails, or takes memory the
 * framework counts on), a step running while the decode side of the same process overlaps rollouts on other streams
 * (cudaMalloc / cudaFree synchronise the device and stall them; PAPER.md:92-111 is about keeping exactly that
 * overlap), a loss-only rank of a vocab-parallel job that holds no vocab shard and would otherwise size a workspace
 * for contractions it never runs, or a plug-in that is only ever given input and output pointers.
 *
 * grpo_loss_from_partials_static is grpo_loss_from_partials (same kernels, same arithmetic, same argument meaning)
 * with NO context and NO workspace: the switches come from *cfg (HOST; read during the call: clip_lo, clip_hi,
 * kl_beta, kl_type, dual_clip, loss_agg), S_norm replaces grpo_set_seq_denom (loss_agg 1: sequences of the whole
 * logical update, 0 = this call's S), and the kernel's scratch - block sums and arrival counter of the fixed-order
 * loss reduction, the token counts that define the mean, 336 KiB in all - is an array compiled into the library.
 * Every GPU that loads the library holds that array until the process exits.  The call runs no cudaMalloc, cudaFree,
 * cudaMallocHost or any other allocating routine; inputs and outputs are the caller's, as everywhere else.
 *
 * Limits: T <= GRPO_STATIC_MAX_TOKENS and S <= GRPO_STATIC_MAX_SEQUENCES, otherwise GRPO_ERR_WORKSPACE and nothing
 * is launched (cut the update into several calls with an explicit loss_denom / S_norm, or use the workspace path).
 * First call on a device: looks the array's device address up once (with that device current) and checks the arch;
 * make that first call outside any stream capture.  Later calls on that device only enqueue work on `stream`.
 * Sharing: there is ONE array per GPU, shared by every caller and every stream in the process, and it keeps the last
 * call's contents (the call clears the words that must start at zero).  Two calls whose work overlaps on the same
 * GPU race on it and give wrong loss / metrics sums: order them on one stream or with events.
 * err_flags: device int32 [1] or NULL; bit 0 is OR-ed in when a target id >= V_global is seen (such tokens are
 * ignored, as in the forward); with NULL the condition is not reported.  The caller clears the word. */
#define GRPO_STATIC_MAX_TOKENS 1048576
#define GRPO_STATIC_MAX_SEQUENCES 65536
int32_t grpo_loss_from_partials_static(const grpo_config* cfg /*HOST*/, int32_t n_shards, const float* m2,
                                       const float* s2, const float* zy, const int32_t* targets, int32_t V_global,
                                       const int32_t* cu_seqlens, int32_t S, int32_t S_norm, int64_t T,
                                       const float* adv, const float* old_logp, const float* ref_logp,
                                       const uint8_t* mask, double loss_denom, float* logp_out, float* lse_out,
                                       float* coeff_out, float* loss_accum, float* metrics_accum, int32_t* err_flags,
                                       void* stream);

/* A4-A6.  lse, coeff from the forward.  grad_scale multiplies both gradients (upstream dLoss).
 * dhidden_out [T, d] (bf16, or fp32 if cfg.dhidden_fp32) is OVERWRITTEN; dW_accum fp32 [V, d] is
 * ADDED to with atomics (caller zeroes it at the optimizer boundary).  Either may be NULL to skip. */
int32_t grpo_fused_logprob_loss_bwd(grpo_ctx* ctx, const void* hidden, const void* W, const int32_t* targets,
                                    const float* lse, const float* coeff, int64_t T, float grad_scale,
                                    void* dhidden_out, float* dW_accum, void* stream);

/* Optional diagnostic output of the forward (R28): while a non-NULL
 * device pointer is set, every later grpo_fused_logprob_loss_fwd / _fwd_bwd call of this context also writes
 * entropy_out[t] = - sum_v p_tv log p_tv (nats) for each of its T packed rows (one more running sum in the A2
 * epilogue; no gradient flows through it).  The caller owns the buffer ([T] fp32 of the largest call) and
 * keeps it alive until the stream reaches the call's work.  NULL turns it off (default).  Not used by
 * grpo_enqueue_groups / grpo_step_host. */
int32_t grpo_set_entropy_out(grpo_ctx* ctx, float* entropy_out);

/* ---- NEXT-4: the step before the path, the final RMSNorm, and its backward ----------
 * BASELINE.json configs describe the path's input as "hidden ... after RMSNorm-like scaling"; these calls take the
 * PRE-norm activations x bf16 [T, d] and the norm weight gamma bf16 [d] instead (R29-R31).
 *
 * grpo_rmsnorm_fwd: rstd_t = 1 / sqrt(mean_k x_tk^2 + eps_rms);  hidden_out[t,:] = bf16(gamma * x[t,:] * rstd_t)
 * (fp32 arithmetic, rounded once: the contraction kernels consume H as bf16 tiles through TMA, so H is materialised
 * by this one-pass HBM-bound kernel - 4 d bytes of traffic per token against 8 V d FLOPs).  rstd_out fp32 [T] is kept
 * for the backward.  x, gamma, hidden_out 8-byte aligned.
 *
 * grpo_fused_logprob_loss_bwd_prenorm: grpo_fused_logprob_loss_bwd with the RMSNorm backward fused behind A5: the
 * fp32 dHidden row coming out of the split-K reduction is turned, in registers, into
 *     dx[t,:] = rstd_t (g - xh mean_k(g xh)),   g = gamma * dH[t,:],  xh = x[t,:] rstd_t,
 * and dgamma_accum fp32 [d] += sum_t dH[t,:] * xh (ADDED to, like dW).  dHidden itself is never written.
 * dx_out [T, d] (bf16, or fp32 if cfg.dhidden_fp32) is OVERWRITTEN.  d <= 8192.
 *
 * grpo_rmsnorm_bwd: the same backward as a stand-alone HBM-bound kernel for a dHidden that already exists
 * (e.g. the per-group dhidden_out of grpo_enqueue_groups): dhidden bf16 [T, d], or fp32 if dhidden_is_fp32. */
int32_t grpo_rmsnorm_fwd(grpo_ctx* ctx, const void* x, const void* gamma, float eps_rms, int64_t T, void* hidden_out,
                         float* rstd_out, void* stream);
int32_t grpo_rmsnorm_bwd(grpo_ctx* ctx, const void* x, const void* gamma, const float* rstd, const void* dhidden,
                         int32_t dhidden_is_fp32, int64_t T, void* dx_out, float* dgamma_accum, void* stream);
int32_t grpo_fused_logprob_loss_bwd_prenorm(grpo_ctx* ctx, const void* x, const void* gamma, const float* rstd,
                                            const void* hidden, const void* W, const int32_t* targets,
                                            const float* lse, const float* coeff, int64_t T, float grad_scale,
                                            void* dx_out, float* dgamma_accum, float* dW_accum, void* stream);

/* 3-contraction variant of forward + backward in ONE call.
 * Per chunk of bwd_chunk_tokens tokens: the forward contraction (A2) also writes the chunk's softmax numerators
 * as fp16 into the workspace chunk buffer, A3 runs on the chunk, an HBM-bound pass turns the stashed logits into
 * dZ in place, then A5 and A6 run as in the backward.  The [T, V] logits are still never materialised (one
 * [Tc, V] chunk lives in the workspace) but nothing is recomputed: 6 T V d FLOPs instead of 8 T V d.
 * Arguments and outputs are those of grpo_fused_logprob_loss_fwd followed by grpo_fused_logprob_loss_bwd
 * (dhidden_out / dW_accum may each be NULL); results agree with that pair within the parity tolerances (what
 * is stashed is each logit's exponential relative to its row's running maximum, rounded to fp16: a 2^-11
 * relative error per probability whatever the magnitude of the logits; the recomputed path has none).  The denominator of the mean must be
 * known before the first chunk: loss_denom > 0, or it is counted from mask / targets of this call first. */
int32_t grpo_fused_logprob_loss_fwd_bwd(grpo_ctx* ctx, const void* hidden, const void* W, const int32_t* targets,
                                        const int32_t* cu_seqlens, int32_t S, int64_t T, const float* adv,
                                        const float* old_logp, const float* ref_logp, const uint8_t* mask,
                                        double loss_denom, float grad_scale, float* logp_out, float* lse_out,
                                        float* coeff_out, float* loss_accum, float* metrics_accum, void* dhidden_out,
                                        float* dW_accum, void* stream);

/* One COMPLETE group (all K responses present, rewards verified). */
typedef struct {
  int64_t group_order;          /* submission order; informational, FIFO is by arrival */
  int32_t G;                    /* responses in the group */
  const int32_t* seqlens_host;  /* HOST int32 [G]: loss-bearing tokens per response (copied by the call) */
  const void* hidden;           /* bf16 [T_g, d], the group's packed tokens */
  const int32_t* targets;       /* [T_g] */
  const float* old_logp;        /* [T_g] */
  const float* ref_logp;        /* [T_g] or NULL */
  const uint8_t* mask;          /* [T_g] or NULL */
  const float* rewards;         /* device fp32 [G] */
  void* dhidden_out;            /* [T_g, d] or NULL */
  float* logp_out;              /* [T_g] or NULL */
} grpo_group_desc;

/* A0 + A7.  Append n complete groups to the FIFO in arrival order, then, if at least U
 * groups are pending, run ONE logical update over the earliest U: they are split into launches, each
 * the largest prefix of whole groups within cfg.token_budget (at least one group); launch
 * k of the context runs on streams[k % n_streams] with workspace slot k % n_streams; each launch is
 * A1 -> A2/A3 -> A4-A6 on its packed tokens.  dW_accum / loss_accum are only ADDED to.
 * loss_denom as in the forward but over the whole update (<= 0: derived from the update's masks).
 * A group with G != cfg.group_size (when set), G <= 0, a NULL pointer where one is required or a
 * non-positive sequence length is GRPO_ERR_INCOMPLETE_GROUP and nothing is appended.
 * HOST outputs: groups_consumed_out (total consumed so far), update_boundary_out (1 if an update was
 * run by this call: the caller may step the optimizer and zero dW once the streams reach this work).
 * n = 0 is allowed (continue draining the FIFO). */
/* Errors: everything that can be rejected without the device (workspace capacity, ref_logp given for some groups
 * of a launch only, an implicit denominator over more than 2^24 tokens) is checked for EVERY launch of the update
 * before the first kernel is enqueued - nothing is accumulated and the FIFO is unchanged.  If a launch fails later
 * (a CUDA error while enqueueing), the update is BROKEN: the launches already enqueued have added their share -
 * scaled by this update's denominator - to dW / loss / metrics, kernels of the failed launch may have too, and the
 * accumulators no longer hold a whole number of groups.  The context then refuses every further grpo_enqueue_groups
 * / grpo_flush (GRPO_ERR_CUDA) until the caller has discarded the update - zero dW_accum / loss_accum /
 * metrics_accum - and called grpo_reset_round, which empties the FIFO (groups_consumed_out says how many groups of
 * the round had been consumed); the caller resubmits what the round still needs. */
int32_t grpo_enqueue_groups(grpo_ctx* ctx, const grpo_group_desc* groups, int32_t n, const void* W,
                            float* dW_accum, float* loss_accum, float* metrics_accum, double loss_denom,
                            void* const* streams, int32_t n_streams, int32_t* groups_consumed_out,
                            int32_t* update_boundary_out);

/* End of round: run whatever is pending (< U groups) as a final, short update. */
int32_t grpo_flush(grpo_ctx* ctx, const void* W, float* dW_accum, float* loss_accum, float* metrics_accum,
                   double loss_denom, void* const* streams, int32_t n_streams, int32_t* groups_consumed_out,
                   int32_t* update_boundary_out);

/* FIFO state (HOST outputs, any may be NULL): groups / tokens pending, groups consumed,
 * round_complete = 1 once consumed >= cfg.groups_per_round > 0 (Alg. 1 l.22). */
int32_t grpo_queue_state(const grpo_ctx* ctx, int32_t* pending_groups, int64_t* pending_tokens,
                         int32_t* consumed_groups, int32_t* round_complete);
int32_t grpo_reset_round(grpo_ctx* ctx);

/* Pure host helper (no CUDA): how the next logical update is cut into launches.  group_tokens HOST
 * int64 [n_pending] in FIFO order.  Returns in launch_sizes_out[0..*n_launches_out) the number of
 * groups per launch; *n_launches_out = 0 if fewer than U groups are pending and flush == 0. */
int32_t grpo_cgp_plan(const int64_t* group_tokens, int32_t n_pending, int32_t U, int64_t token_budget,
                      int32_t flush, int32_t* launch_sizes_out, int32_t cap, int32_t* n_launches_out);

/* Reads the device error word (bit 0: a target id >= V was seen) and clears it.  Synchronises. */
int32_t grpo_check_errors_sync(grpo_ctx* ctx, int32_t* flags_out /*HOST*/);

/* End-to-end convenience over HOST buffers (pinned recommended): copies one packed batch to the
 * device (slot 0 staging), runs A1 -> A6 with W / dW_accum resident on the device, copies
 * loss, logp and dHidden back, and synchronises `stream`.  n_groups uniform groups of size G.
 * hidden_host bf16 [T,d]; dhidden_host [T,d] or NULL; logp_host [T] or NULL; loss_host fp32 [1]. */
int32_t grpo_step_host(grpo_ctx* ctx, const void* hidden_host, const int32_t* targets_host,
                       const int32_t* cu_seqlens_host, const float* rewards_host, const float* old_logp_host,
                       const float* ref_logp_host, const uint8_t* mask_host, int32_t n_groups, int32_t G,
                       int64_t T, const void* W, float* dW_accum, double loss_denom, float* loss_host,
                       float* logp_host, void* dhidden_host, void* stream);

/* Kernel accounting.  Every kernel this library launches belongs to one kind. */
enum {
  GRPO_KERNEL_ADVANTAGE = 0,   /* A1 */
  GRPO_KERNEL_TOKEN_COUNT = 1, /* mask counts / fills that define the mean */
  GRPO_KERNEL_GEMM_LSE = 2,    /* A2: z = H W^T with the online log-sum-exp epilogue */
  GRPO_KERNEL_LOSS = 3,        /* A3 */
  GRPO_KERNEL_GEMM_DZ = 4,     /* A4: recompute z, dZ epilogue */
  GRPO_KERNEL_GEMM_DH = 5,     /* A5: dH = dZ W */
  GRPO_KERNEL_GEMM_DW = 6,     /* A6: dW += dZ^T H */
  GRPO_KERNEL_DEBUG = 7,       /* grpo_debug_gemm */
  GRPO_KERNEL_RESERVED_8 = 8,  /* (round 1's per-tile zero scan; replaced by GRPO_KERNEL_COMPACT) */
  GRPO_KERNEL_STASH_DZ = 9,    /* 3-contraction variant: stashed logits -> dZ in place */
  GRPO_KERNEL_COMPACT = 10,    /* backward: zero-coefficient row compaction, gather of active rows, zero fill */
  GRPO_KERNEL_DH_REDUCE = 11,  /* A5: fixed-order sum of the split-K partials (+ scatter of compacted rows; + the
                                  RMSNorm backward of the pre-norm calls) */
  GRPO_KERNEL_RMSNORM = 12,    /* NEXT-4: final RMSNorm forward */
  GRPO_KERNEL_QUANTIZE = 13,   /* FP8 study: e4m3 quantisation of hidden rows / the vocab matrix */
  GRPO_NUM_KERNEL_KINDS = 14
};

/* Packed rows the backward calls of all workspace slots ran their contractions over (active: coeff != 0) and saw
 * (total) since the last call of this function; both 0 when bwd_skip_zero_tiles is off.  Synchronises. */
int32_t grpo_bwd_row_stats_sync(grpo_ctx* ctx, int64_t* active_out /*HOST*/, int64_t* total_out /*HOST*/);

/* counts_out HOST int64 [GRPO_NUM_KERNEL_KINDS]: kernels launched by this context since creation. */
int32_t grpo_kernel_launches(const grpo_ctx* ctx, int64_t* counts_out);

/* While enabled, every kernel launch is bracketed by CUDA events recorded on its launch stream.
 * grpo_profile_read_sync synchronises the device, sums the elapsed milliseconds per kind into
 * ms_out (HOST double [GRPO_NUM_KERNEL_KINDS]) with the number of timed launches in launches_out
 * (HOST int64 [GRPO_NUM_KERNEL_KINDS]), and clears the records.  Disabling discards records. */
int32_t grpo_profile_enable(grpo_ctx* ctx, int32_t on);
int32_t grpo_profile_read_sync(grpo_ctx* ctx, double* ms_out, int64_t* launches_out);

/* ---- NEXT-3: a dW accumulator stitched from per-rank shards --------------------
 * Data parallelism over complete groups needs the sum of the ranks' dW at the update boundary.
 * Instead of an all-reduce after the GEMM, the accumulator itself is laid out across the GPUs with CUDA virtual
 * memory management: every rank creates ONE physical chunk on its own GPU (grpo_shard_create; *fd_out is a POSIX
 * file descriptor to hand to the other ranks over a Unix socket, the caller closes it), imports the others'
 * (grpo_shard_import) and maps all chunks in rank order into one contiguous device range (grpo_stitch_map: shard i
 * at byte offset i * bytes).  That range is an ordinary `dW_accum` for grpo_fused_logprob_loss_bwd /
 * grpo_enqueue_groups: the A6 epilogue's fp32 reduce-adds (performed at the L2 of the memory's home GPU) are carried
 * by NVLink to the peers' shards, so the reduce-scatter happens INSIDE the contraction kernel, overlapped with its
 * MMAs tile by tile; after a barrier rank r holds the fully reduced rows [r R, (r+1) R), R = bytes / (4 d).
 * bytes must be a multiple of grpo_shard_granularity (2 MiB on B200: 256 rows at d = 2048) and of 4 d.
 * All pointers HOST except the mapped range.  grpo_stitch_unmap synchronises the device.  DESIGN.md section 7. */
typedef struct grpo_shard grpo_shard;
int32_t grpo_shard_granularity(grpo_ctx* ctx, int64_t* bytes_out);
int32_t grpo_shard_create(grpo_ctx* ctx, int64_t bytes, grpo_shard** shard_out, int32_t* fd_out);
int32_t grpo_shard_import(grpo_ctx* ctx, int32_t fd, int64_t bytes, grpo_shard** shard_out);
int32_t grpo_shard_release(grpo_ctx* ctx, grpo_shard* shard);
int32_t grpo_stitch_map(grpo_ctx* ctx, grpo_shard* const* shards, int32_t n, void** dev_ptr_out);
int32_t grpo_stitch_unmap(grpo_ctx* ctx, void* dev_ptr);

/* Diagnostic: how many thread-block clusters of `cluster_size` CTAs of the contraction kernel (224 threads, its
 * full shared-memory ring) the device can hold at once (cudaOccupancyMaxActiveClusters).  clusters_out HOST.
 * The kernels run as 74 CTA pairs; DESIGN.md section 5 records why larger multicast clusters are not used
 * (148 CTAs co-resident at cluster size 2, 132 at 4, 120 at 8 on B200). */
int32_t grpo_debug_max_active_clusters(grpo_ctx* ctx, int32_t cluster_size, int32_t* clusters_out);

/* Test hook: C[M,N] (fp32, row-major, pitch N) = A * B with the production tcgen05 kernel.
 * layout 0: A [M,K] K-major, B [N,K] K-major;  1: A [M,K] K-major, B [K,N] MN-major;
 * 2: A [K,M] MN-major, B [K,N] MN-major.  accumulate != 0: C += (atomic).  bf16 inputs.
 * M, N, K multiples of 8. */
int32_t grpo_debug_gemm(grpo_ctx* ctx, int32_t layout, const void* A, const void* B, float* C, int32_t M,
                        int32_t N, int32_t K, int32_t accumulate, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* GRPO_B200_H_ */
