// Host-side RolloutPipe scheduler model (include/rollout_pipe.h).  Pure C++.
//
// Rollout node: egalitarian processor sharing is simulated in *virtual time*: every in-flight request
// receives service at the same rate min(max_rate, capacity / n), so with v(t) = service received per
// in-flight request since t = 0, a request admitted at virtual time v_a with `work` tokens completes when
// v = v_a + work.  A min-heap over those completion keys gives the next event in O(log RK); wall time
// advances by dv / rate between events.  FGD only changes WHICH requests are in the heap:
// those of the F_w lowest-order unfinished groups (Eq. 5-6); a finished group frees a slot that the next
// lowest-order deferred group takes at once (reading RP2).
//
// Control + training node: the ActorGroup FIFO is the list of groups sorted by trainable time;
// update j is ready when its U groups are in the FIFO (CGP) or when the round is complete (Slime), and the
// trainer serves updates back to back (Alg. 1 l.16-23).  Eq. 2-4 are then read off the timeline.
#include "../../include/rollout_pipe.h"

#include <algorithm>
#include <cmath>
#include <functional>
#include <numeric>
#include <queue>
#include <utility>
#include <vector>

namespace {

struct Ev {
  double key;     // virtual completion time
  int32_t g, i;
  bool operator>(const Ev& o) const { return key > o.key || (key == o.key && (g > o.g || (g == o.g && i > o.i))); }
};

}  // namespace

extern "C" int32_t rp_fgd_frontier(const int64_t* orders, int32_t n, int32_t F_w, int64_t* frontier_out,
                                   int32_t* n_out) {
  if (n < 0 || (n > 0 && !orders) || !n_out) return 1;
  const int32_t k = std::max(0, std::min(F_w, n));
  std::vector<int64_t> v(orders, orders + n);
  std::partial_sort(v.begin(), v.begin() + k, v.end());
  if (frontier_out) std::copy(v.begin(), v.begin() + k, frontier_out);
  *n_out = k;
  return 0;
}

extern "C" int32_t rp_rollout(const double* work, int32_t R, int32_t K, double capacity, double max_rate, int32_t F_w,
                              double* request_done, double* group_done, double* trace_time, int64_t* trace_groups,
                              int32_t trace_cap, int32_t* n_trace) {
  if (!work || R < 0 || K <= 0 || !(capacity > 0.0)) return 1;
  for (int64_t q = 0; q < static_cast<int64_t>(R) * K; ++q)
    if (!(work[q] >= 0.0)) return 1;
  const bool fgd = F_w > 0;
  const int32_t width = fgd ? std::min(F_w, R) : R;
  std::priority_queue<Ev, std::vector<Ev>, std::greater<Ev>> heap;
  std::vector<int32_t> left(R, K);          // unfinished requests per group
  std::vector<int32_t> frontier;            // groups in service, ascending order
  int32_t next_group = 0, traces = 0;
  double v = 0.0, t = 0.0;
  int64_t inflight = 0;

  auto record = [&]() {
    if (!fgd) return;
    if (traces < trace_cap && trace_time && trace_groups) {
      trace_time[traces] = t;
      for (int32_t s = 0; s < std::max(F_w, 1); ++s)
        trace_groups[static_cast<int64_t>(traces) * std::max(F_w, 1) + s] =
            s < static_cast<int32_t>(frontier.size()) ? frontier[s] : -1;
    }
    ++traces;
  };
  auto admit = [&]() {                       // "while |F| < F_w: admit the lowest-order deferred group"
    bool changed = false;
    while (static_cast<int32_t>(frontier.size()) < width && next_group < R) {
      const int32_t g = next_group++;
      frontier.push_back(g);
      for (int32_t i = 0; i < K; ++i) heap.push(Ev{v + work[static_cast<int64_t>(g) * K + i], g, i});
      inflight += K;
      changed = true;
    }
    return changed;
  };

  admit();
  record();
  while (!heap.empty()) {
    const Ev e = heap.top();
    heap.pop();
    if (e.key > v) {
      double rate = capacity / static_cast<double>(inflight);
      if (max_rate > 0.0) rate = std::min(rate, max_rate);
      t += (e.key - v) / rate;
      v = e.key;
    }
    --inflight;
    if (request_done) request_done[static_cast<int64_t>(e.g) * K + e.i] = t;
    if (--left[e.g] == 0) {                  // "When g completes K requests it leaves F"
      if (group_done) group_done[e.g] = t;
      frontier.erase(std::find(frontier.begin(), frontier.end(), e.g));
      admit();
      record();
    }
  }
  if (n_trace) *n_trace = traces;
  return 0;
}

extern "C" int32_t rp_cgp_timeline(const double* trainable, const double* train_s, int32_t R, int32_t U, int32_t mode,
                                   rp_timeline* out, int32_t* fifo_order, double* ready, double* start, double* end) {
  if (!trainable || !train_s || R < 0 || U < 1 || mode < 0 || mode > 2 || !out) return 1;
  std::vector<int32_t> order(R);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return trainable[a] < trainable[b]; });
  if (fifo_order) std::copy(order.begin(), order.end(), fifo_order);
  rp_timeline r{};
  for (int32_t g = 0; g < R; ++g) {
    r.t_complete = std::max(r.t_complete, trainable[g]);
    r.compute += train_s[g];
  }
  r.t_first_U = R > 0 ? trainable[order[std::min(U, R) - 1]] : 0.0;
  r.dt_cgp = r.t_complete - r.t_first_U;
  r.n_updates = (R + U - 1) / U;
  double prev_end = 0.0;
  for (int32_t j = 0; j < r.n_updates; ++j) {
    const int32_t b = j * U, e = std::min(R, b + U);
    double rdy = r.t_complete, work = 0.0;
    if (mode != RP_MODE_SLIME && e - b == U) rdy = trainable[order[e - 1]];   // FIFO holds these U groups
    for (int32_t k = b; k < e; ++k) work += train_s[order[k]];
    const double s = std::max(rdy, prev_end), f = s + work;
    if (ready) ready[j] = rdy;
    if (start) start[j] = s;
    if (end) end[j] = f;
    if (j == 0) r.t_start = s;
    prev_end = f;
  }
  r.t_train_end = prev_end;
  r.wait = r.t_train_end - r.compute;
  r.w_train_eq4 = r.t_train_end > 0.0 ? r.t_start / r.t_train_end : 0.0;
  r.w_train_alt = (r.wait + r.compute) > 0.0 ? r.wait / (r.wait + r.compute) : 0.0;
  *out = r;
  return 0;
}

extern "C" int32_t rp_simulate(const double* work, int32_t R, int32_t K, double capacity, double max_rate, int32_t F_w,
                               int32_t U, int32_t mode, const double* materialize_s, const double* train_s,
                               rp_timeline* out, double* group_trainable_out, int32_t* fifo_order, double* ready,
                               double* start, double* end) {
  if (!materialize_s || !train_s || R < 0) return 1;
  std::vector<double> done(std::max(R, 0));
  const int32_t st = rp_rollout(work, R, K, capacity, max_rate, mode == RP_MODE_CGP_FGD ? F_w : 0, nullptr,
                                done.data(), nullptr, nullptr, 0, nullptr);
  if (st != 0) return st;
  for (int32_t g = 0; g < R; ++g) done[g] += materialize_s[g];
  if (group_trainable_out) std::copy(done.begin(), done.end(), group_trainable_out);
  return rp_cgp_timeline(done.data(), train_s, R, U, mode, out, fifo_order, ready, start, end);
}
