/* rollout_pipe.h — C ABI of the host-side RolloutPipe scheduler model.
 *
 * The paper's two mechanisms, as an event-driven model of one rollout round:
 *   FGD  frontier-group dispatch at the serving-admission stage   (Eq. 5-6; Alg. 1 l.8-12)
 *   CGP  complete-group pipelining at the trainer boundary        (Eq. 2-4; Alg. 1 l.16-23)
 * All pointers are HOST pointers owned by the caller; nothing here touches the GPU.  Every function
 * returns 0 on success and a non-zero code on a bad argument (the same numbering as grpo_status:
 * 1 = invalid argument).  No function allocates memory that outlives the call.
 *
 * Readings where the paper is silent: RP1 service is egalitarian processor sharing of
 * `capacity` ("rollout capacity is evenly spread across all in-flight requests") with an
 * optional per-request rate cap; RP2 a freed frontier slot is refilled at the completion instant; RP3
 * materialization latency is a per-group constant; RP4 FIFO order = order of trainable times, ties by
 * submission order; RP5 a last partial update (U does not divide R) is dispatched when the round is
 * complete; RP6 the rollout starts at t = 0.
 */
#ifndef ROLLOUT_PIPE_H_
#define ROLLOUT_PIPE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { RP_MODE_SLIME = 0, RP_MODE_CGP = 1, RP_MODE_CGP_FGD = 2 };

/* Eq. 5: the F_w lowest-order groups among `n` unfinished groups.
 * orders [n] in, frontier_out [min(F_w, n)] out (ascending), *n_out = its length. */
int32_t rp_fgd_frontier(const int64_t* orders, int32_t n, int32_t F_w, int64_t* frontier_out, int32_t* n_out);

/* Rollout node: R groups x K requests arrive at t = 0 in submission order g = 0..R-1.
 *   work [R*K]        decode length of request (g, i) at work[g*K + i], >= 0 (tokens)
 *   capacity          engine throughput shared equally by the in-flight requests (tokens/s), > 0
 *   max_rate          per-request rate cap (tokens/s); <= 0: none
 *   F_w               <= 0: default request-level FIFO admission (everything in flight);
 *                     > 0: FGD, a request is in flight iff its group is in the frontier (Eq. 6)
 * Outputs (each may be NULL):
 *   request_done [R*K], group_done [R]   completion times (s)
 *   trace_time [trace_cap], trace_groups [trace_cap * max(F_w,1)] (-1 padded), *n_trace
 *                     the frontier after each change of F (only when F_w > 0; extra changes beyond
 *                     trace_cap are counted in *n_trace but not stored)
 */
int32_t rp_rollout(const double* work, int32_t R, int32_t K, double capacity, double max_rate, int32_t F_w,
                   double* request_done, double* group_done, double* trace_time, int64_t* trace_groups,
                   int32_t trace_cap, int32_t* n_trace);

typedef struct {
  double t_first_U;    /* time the first U groups are all trainable                         (Eq. 2) */
  double t_complete;   /* time the last group is trainable (rollout completion)                      */
  double dt_cgp;       /* t_complete - t_first_U                                             (Eq. 3) */
  double t_start;      /* trainer start of the first update in the simulated mode           (Eq. 2) */
  double t_train_end;
  double compute;      /* total active trainer time                                                  */
  double wait;         /* trainer idle time between rollout start and train end                      */
  double w_train_eq4;  /* (t_start - t_rollout_start) / (t_train_end - t_rollout_start)      (Eq. 4) */
  double w_train_alt;  /* wait / (wait + compute) */
  int32_t n_updates;
} rp_timeline;

/* Control + training node for given trainable times.
 *   trainable [R], train_s [R]  time group g became trainable; trainer compute time of group g
 *   U >= 1, mode in {RP_MODE_SLIME, RP_MODE_CGP, RP_MODE_CGP_FGD} (the last two behave alike here)
 * Outputs (each may be NULL): fifo_order [R]; ready / start / end [ceil(R/U)] per logical update. */
int32_t rp_cgp_timeline(const double* trainable, const double* train_s, int32_t R, int32_t U, int32_t mode,
                        rp_timeline* out, int32_t* fifo_order, double* ready, double* start, double* end);

/* One whole round (Alg. 1 l.1-7): rp_rollout (FGD only in RP_MODE_CGP_FGD), trainable = group_done +
 * materialize_s (RP3), then rp_cgp_timeline.  group_trainable_out [R] may be NULL. */
int32_t rp_simulate(const double* work, int32_t R, int32_t K, double capacity, double max_rate, int32_t F_w,
                    int32_t U, int32_t mode, const double* materialize_s, const double* train_s, rp_timeline* out,
                    double* group_trainable_out, int32_t* fifo_order, double* ready, double* start, double* end);

#ifdef __cplusplus
}
#endif
#endif /* ROLLOUT_PIPE_H_ */
