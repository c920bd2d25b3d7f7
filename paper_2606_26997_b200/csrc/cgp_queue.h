// Host-side complete-group pipelining (CGP) bookkeeping: the FIFO of trainable complete groups, the
// feasible-batch selector and the logical-update boundary.  Pure C++, no CUDA.
//
//   "CGP appends each group to a FIFO ... as soon as it finishes materialization, and once the FIFO
//    accumulates U trainable groups, the earliest U are dispatched to the trainer."
//   "The Feasible Batch Selector picks the largest prefix of groups (counted in whole groups, never
//    single requests) that fits the per-GPU token budget.  Even when a single group exceeds the budget,
//    it is still taken alone and adapted through dynamic micro-batching."
//   "the optimizer step triggers only when accumulation reaches U"
#pragma once
#include <cstdint>
#include <deque>
#include <vector>

namespace grpo {

// Largest prefix of whole groups of tokens[begin, end) whose token sum fits `budget`; at least one group.
// budget <= 0 means unlimited.
inline int feasible_prefix(const int64_t* tokens, int begin, int end, int64_t budget) {
  if (begin >= end) return 0;
  if (budget <= 0) return end - begin;
  int64_t sum = 0;
  int n = 0;
  for (int i = begin; i < end; ++i) {
    if (n > 0 && sum + tokens[i] > budget) break;
    sum += tokens[i];
    ++n;
  }
  return n;
}

// Cut the next logical update (earliest min(U, pending) groups; only if pending >= U or flush) into
// launches of whole groups.  Returns the number of groups in the update (0 = nothing to dispatch).
inline int plan_update(const int64_t* tokens, int n_pending, int U, int64_t budget, bool flush,
                       std::vector<int>& launch_sizes) {
  launch_sizes.clear();
  if (U < 1) U = 1;
  int take = 0;
  if (n_pending >= U) take = U;
  else if (flush) take = n_pending;
  int pos = 0;
  while (pos < take) {
    const int k = feasible_prefix(tokens, pos, take, budget);
    launch_sizes.push_back(k);
    pos += k;
  }
  return take;
}

}  // namespace grpo
