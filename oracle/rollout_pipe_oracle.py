"""Oracle (TEST INFRASTRUCTURE, not product code) for SURVEY.md §8(f) NEXT-1: RolloutPipe's two scheduling
mechanisms as a plain event-by-event simulation in float64, written in the paper's order and notation.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module.  It shares no
code with the C++ implementation (paper_2606_26997_b200/csrc/rollout_pipe.cpp) and neither imports the other.

What the paper fixes, and where:
  * FGD admission (Eq. 5-6; Alg. 1 l.8-12): the frontier F holds the
    F_w lowest-order groups that arrived and are not yet serving-complete; a request is admitted iff its
    group is in F, otherwise it is deferred; when a group completes its K requests it leaves F and the next
    lowest-order deferred group is admitted.
  * Default admission: request-level FIFO, all R*K requests arrive together and are admitted.
  * "rollout capacity is evenly spread across all in-flight requests": egalitarian processor
    sharing of the engine's capacity.
  * Materialization makes a serving-complete group trainable; CGP appends it to the
    ActorGroup FIFO at that moment.
  * CGP dispatch (Alg. 1 l.16-19): once the FIFO holds U trainable groups the earliest U are
    dispatched; Slime hands all R groups over when the rollout completes.
  * Train (Alg. 1 l.20-23): forward/backward/accumulate over the U groups, optimizer step at U.
  * Eq. 2: t_start^Slime = t_complete, t_start^CGP = t_first^(U).  Eq. 3: dt_CGP = t_complete - t_first^(U).
    Eq. 4: w_train = (t_start - t_rollout_start) / (t_train_end - t_rollout_start).
    Second definition: trainer-side wait / (wait + compute).

Readings where the paper is silent (RP1-RP6):
  RP1  per-request service: rate = min(max_rate, capacity / n_inflight) work units per second (max_rate <= 0:
       no cap).  `work` is the request's decode length in tokens, capacity in tokens/s.
  RP2  the "scheduling cycle" has zero period: a freed frontier slot is refilled at the completion instant.
  RP3  materialization latency is a per-group constant added to the serving-complete time.
  RP4  FIFO order = order of trainable times, ties broken by submission order.
  RP5  if U does not divide R the last partial update is dispatched when all R groups are trainable.
  RP6  t_rollout_start = 0 (all requests arrive at time 0).

Parity pins (tests/test_rollout_pipe.py): the paper's three worked examples (
tests/golden/rollout_pipe_examples.txt), Eq. 2-4 evaluated by hand, the textbook closed form of
egalitarian processor sharing, F_w >= R reducing FGD to default admission, work conservation, and the
paper's invariant that the three modes do the same amount of trainer compute.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np

MODE_SLIME, MODE_CGP, MODE_CGP_FGD = 0, 1, 2


# ------------------------------------------------------------------------------- rollout node
def fgd_frontier(unfinished_orders: Sequence[int], F_w: int) -> List[int]:
    """Eq. 5: the F_w groups of lowest order among the groups not yet serving-complete."""
    return sorted(unfinished_orders)[:max(F_w, 0)]


def rollout(work: np.ndarray, capacity: float, max_rate: float = 0.0, F_w: int = 0):
    """Serve R groups x K requests, all arriving at t = 0 in order(g) = g.

    F_w <= 0: default request-level FIFO admission (everything admitted at arrival).
    F_w  > 0: FGD (Eq. 5-6): only requests of frontier groups are in flight.
    Returns (request_done [R, K], group_done [R], frontier_trace) where frontier_trace is the list of
    (time, frontier as a list of group orders) after every change of F.
    """
    work = np.asarray(work, dtype=np.float64)
    R, K = work.shape
    remaining = work.copy()
    done_t = np.full((R, K), np.nan)
    group_done = np.full(R, np.nan)
    finished_req = np.zeros((R, K), dtype=bool)
    finished_grp = np.zeros(R, dtype=bool)
    t = 0.0
    trace = []

    def current_frontier():
        unfinished = [g for g in range(R) if not finished_grp[g]]
        return unfinished if F_w <= 0 else fgd_frontier(unfinished, F_w)

    F = current_frontier()
    trace.append((t, list(F)))
    # zero-work requests finish at once
    while True:
        inflight = [(g, i) for g in F for i in range(K) if not finished_req[g, i]]
        if not inflight:
            if finished_grp.all():
                break
            F = current_frontier()          # RP2: refill immediately
            trace.append((t, list(F)))
            continue
        n = len(inflight)
        rate = capacity / n
        if max_rate > 0.0:
            rate = min(rate, max_rate)
        # next completion among in-flight requests
        rem = np.array([remaining[g, i] for g, i in inflight])
        dt = float(rem.min() / rate)
        t = t + dt
        dec = rate * dt
        changed = False
        for (g, i), r in zip(inflight, rem):
            left = r - dec
            if left <= 1e-12 * max(work[g, i], 1.0) or r == rem.min():
                remaining[g, i] = 0.0
                finished_req[g, i] = True
                done_t[g, i] = t
            else:
                remaining[g, i] = left
        for g in list(F):
            if not finished_grp[g] and finished_req[g].all():
                finished_grp[g] = True       # "When g completes K requests it leaves F"
                group_done[g] = t
                changed = True
        if changed:
            F = current_frontier()
            trace.append((t, list(F)))
    return done_t, group_done, trace


# ------------------------------------------------------------------------------- control + training node
@dataclass
class Timeline:
    fifo_order: List[int]                 # groups in ActorGroup-FIFO order (RP4)
    trainable: np.ndarray                 # [R] time each group became trainable
    ready: List[float]                    # per logical update: time its U groups are all in the FIFO / handed over
    start: List[float]
    end: List[float]
    update_groups: List[List[int]]
    t_first_U: float
    t_complete: float
    dt_cgp: float                         # Eq. 3
    t_start: float                        # Eq. 2 (for the mode simulated)
    t_train_end: float
    compute: float                        # total active trainer time
    wait: float                           # trainer idle time between rollout start and train end
    w_train_eq4: float                    # Eq. 4
    w_train_alt: float                    # wait / (wait + compute)


def cgp_timeline(trainable: Sequence[float], train_s: Sequence[float], U: int, mode: int) -> Timeline:
    """CGP_Handoff + Train of Alg. 1 for given trainable times (rollout start = 0, RP6)."""
    trainable = np.asarray(trainable, dtype=np.float64)
    train_s = np.asarray(train_s, dtype=np.float64)
    R = trainable.size
    order = sorted(range(R), key=lambda g: (trainable[g], g))         # RP4
    t_complete = float(trainable.max()) if R else 0.0
    n_full = R // U
    updates = [order[j * U:(j + 1) * U] for j in range(n_full)]
    if R % U:
        updates.append(order[n_full * U:])                            # RP5
    t_first_U = float(trainable[order[min(U, R) - 1]]) if R else 0.0  # Eq. 2: the first U groups materialised
    ready, start, end = [], [], []
    prev_end = 0.0
    for j, grp in enumerate(updates):
        if mode == MODE_SLIME:
            r = t_complete                                            # handed over when the rollout completes
        else:
            r = float(max(trainable[g] for g in grp))                 # FIFO holds these U groups
            if len(grp) < U:
                r = t_complete                                        # RP5: flush at the end of the round
        s = max(r, prev_end)
        e = s + float(sum(train_s[g] for g in grp))
        ready.append(r); start.append(s); end.append(e)
        prev_end = e
    compute = float(train_s.sum())
    t_start = start[0] if start else 0.0
    t_end = end[-1] if end else 0.0
    wait = t_end - compute
    return Timeline(order, trainable, ready, start, end, updates, t_first_U, t_complete, t_complete - t_first_U,
                    t_start, t_end, compute, wait,
                    (t_start - 0.0) / (t_end - 0.0) if t_end > 0 else 0.0,
                    wait / (wait + compute) if (wait + compute) > 0 else 0.0)


def simulate(work, capacity, max_rate, F_w, U, mode, materialize_s, train_s) -> Timeline:
    """RolloutPipe (Alg. 1 l.1-7) for one rollout round: FGD_Admit/Rollout_Worker, then CGP_Handoff/Train."""
    fw = F_w if mode == MODE_CGP_FGD else 0
    _, group_done, _ = rollout(work, capacity, max_rate, fw)
    trainable = group_done + np.asarray(materialize_s, dtype=np.float64)   # RP3
    return cgp_timeline(trainable, train_s, U, mode)
