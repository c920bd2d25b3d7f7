"""NEXT-1: pins of the RolloutPipe scheduling oracle (oracle/rollout_pipe_oracle.py) against
the paper's worked examples, Eq. 2-4 and textbook closed forms; then parity of the C++ implementation behind
the C ABI (include/rollout_pipe.h) with the oracle on seeded synthetic rounds.  CPU only."""
import os

import numpy as np
import pytest

from oracle import rollout_pipe_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "rollout_pipe_examples.txt")


def _golden():
    out = {}
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        name, inp, exp, cite = [s.strip() for s in line.split("|")]
        kv = lambda s: dict(tok.split("=") for tok in s.split())
        out[name] = (kv(inp), kv(exp), cite)
    return out


# ------------------------------------------------------------------------------------------- paper examples
def test_paper_example_slime_barrier():
    """first group at 200 s, last at 400 s, R = 96: Slime dispatches everything at 400 s and the
    earliest group has waited 200 s."""
    inp, exp, _ = _golden()["slime_barrier"]
    R = int(inp["R"])
    trainable = np.linspace(float(inp["first"]), float(inp["last"]), R)
    tl = O.cgp_timeline(trainable, np.ones(R), U=2, mode=O.MODE_SLIME)
    assert all(r == float(exp["dispatch_all"]) for r in tl.ready)
    assert tl.t_start == float(exp["dispatch_all"])                      # Eq. 2, Slime
    assert tl.ready[0] - trainable.min() == float(exp["earliest_wait"])
    # the same round under CGP starts at t_first^(U) (Eq. 2) and recovers dt_CGP (Eq. 3)
    tc = O.cgp_timeline(trainable, np.ones(R), U=2, mode=O.MODE_CGP)
    assert tc.t_start == tc.t_first_U == trainable[1]
    assert tc.dt_cgp == pytest.approx(400.0 - trainable[1])


def test_paper_example_arrival_gap():
    """U = 2, group 0 at 210 s, group 1 at 250 s: the trainer waits 40 s to form a batch."""
    inp, exp, _ = _golden()["arrival_gap"]
    tl = O.cgp_timeline([float(inp["g0"]), float(inp["g1"])], [10.0, 10.0], U=int(inp["U"]), mode=O.MODE_CGP)
    assert tl.t_first_U == float(exp["t_first_U"])
    assert tl.start[0] - float(inp["g0"]) == float(exp["gap"])
    assert tl.update_groups == [[0, 1]]


def test_paper_example_frontier():
    """F_w = 2, groups 1-6: F = {1,2}; after group 1 completes, F = {2,3}; the trainer starts
    (|Q^(r)| >= U = 2) while groups 3-6 are still in rollout."""
    K = 4
    work = np.array([[10.0] * K, [20.0] * K, [20.0] * K, [20.0] * K, [20.0] * K, [20.0] * K])
    _, gdone, trace = O.rollout(work, capacity=8.0, F_w=2)
    names = lambda F: {g + 1 for g in F}                                  # the paper numbers groups from 1
    assert names(trace[0][1]) == {1, 2}
    assert names(trace[1][1]) == {2, 3}
    assert trace[1][0] == gdone[0]
    tl = O.cgp_timeline(gdone, np.ones(6), U=2, mode=O.MODE_CGP)
    assert tl.update_groups[0] == [0, 1]
    assert tl.start[0] < gdone[2:].min()                                  # groups 3-6 still in rollout
    assert O.fgd_frontier([5, 3, 1, 2, 4, 6], 2) == [1, 2]                # Eq. 5 directly


# ------------------------------------------------------------------------------------------- Eq. 2-4 by hand
def test_eq2_eq3_eq4_by_hand():
    # trainable times 10, 30, 20, 60 (FIFO order 0, 2, 1, 3); U = 2; 5 s of training per group
    tl = O.cgp_timeline([10.0, 30.0, 20.0, 60.0], [5.0] * 4, U=2, mode=O.MODE_CGP)
    assert tl.fifo_order == [0, 2, 1, 3]
    assert tl.t_first_U == 20.0 and tl.t_complete == 60.0 and tl.dt_cgp == 40.0
    assert tl.ready == [20.0, 60.0] and tl.start == [20.0, 60.0] and tl.end == [30.0, 70.0]
    assert tl.w_train_eq4 == pytest.approx(20.0 / 70.0)                  # Eq. 4
    assert tl.wait == pytest.approx(50.0) and tl.w_train_alt == pytest.approx(50.0 / 70.0)
    ts = O.cgp_timeline([10.0, 30.0, 20.0, 60.0], [5.0] * 4, U=2, mode=O.MODE_SLIME)
    assert ts.start == [60.0, 70.0] and ts.end == [70.0, 80.0]
    assert ts.w_train_eq4 == pytest.approx(60.0 / 80.0)
    assert ts.compute == tl.compute                                      # same work, moved earlier
    assert tl.t_train_end <= ts.t_train_end


def test_partial_last_update_is_flushed():
    tl = O.cgp_timeline([1.0, 2.0, 3.0], [1.0, 1.0, 1.0], U=2, mode=O.MODE_CGP)
    assert tl.update_groups == [[0, 1], [2]] and tl.ready == [2.0, 3.0]


# ------------------------------------------------------------------------------------------- processor sharing
def test_processor_sharing_closed_form():
    """Egalitarian processor sharing of capacity C among n jobs that all start at 0 (textbook): with sorted
    works w_(1) <= ... <= w_(n), t_(i) = t_(i-1) + (n - i + 1) (w_(i) - w_(i-1)) / C."""
    rng = np.random.default_rng(5)
    w = rng.integers(1, 4000, size=(6, 8)).astype(np.float64)
    C = 1234.0
    done, gdone, _ = O.rollout(w, capacity=C, F_w=0)
    flat = np.sort(w.reshape(-1))
    n = flat.size
    t, prev, expect = 0.0, 0.0, {}
    for i, wi in enumerate(flat):
        t += (n - i) * (wi - prev) / C
        prev = wi
        expect[wi] = t
    for g in range(6):
        for i in range(8):
            assert done[g, i] == pytest.approx(expect[w[g, i]], rel=1e-12)
    assert np.allclose(gdone, done.max(axis=1))
    assert done.max() == pytest.approx(w.sum() / C, rel=1e-12)          # work conservation


def test_rate_cap_makes_requests_independent():
    w = np.array([[100.0, 300.0], [50.0, 200.0]])
    done, _, _ = O.rollout(w, capacity=1e9, max_rate=10.0, F_w=0)
    assert np.allclose(done, w / 10.0)


def test_fgd_with_wide_frontier_is_default_admission():
    rng = np.random.default_rng(6)
    w = rng.integers(1, 500, size=(5, 4)).astype(np.float64)
    a = O.rollout(w, 100.0, 0.0, F_w=0)[1]
    b = O.rollout(w, 100.0, 0.0, F_w=5)[1]
    c = O.rollout(w, 100.0, 0.0, F_w=99)[1]
    assert np.array_equal(a, b) and np.array_equal(a, c)


def test_fgd_serves_groups_in_submission_order_and_conserves_work():
    rng = np.random.default_rng(7)
    w = rng.integers(1, 500, size=(8, 4)).astype(np.float64)
    done, gdone, trace = O.rollout(w, 64.0, 0.0, F_w=1)
    # F_w = 1: groups are served one at a time, each finishing after its own total work / capacity
    assert np.allclose(gdone, np.cumsum(w.sum(axis=1)) / 64.0)
    assert all(len(F) <= 1 for _, F in trace)
    done2, gdone2, trace2 = O.rollout(w, 64.0, 0.0, F_w=3)
    assert all(len(F) <= 3 for _, F in trace2)                            # |F| <= F_w
    assert gdone2.max() == pytest.approx(w.sum() / 64.0)                  # no cap: capacity never idles
    assert gdone2[0] <= O.rollout(w, 64.0, 0.0, F_w=0)[1][0]              # the earliest group finishes no later


def test_modes_do_the_same_training_work_and_cgp_is_never_later():
    rng = np.random.default_rng(8)
    R, K, U = 12, 4, 2
    w = rng.geometric(1 / 300.0, size=(R, K)).astype(np.float64)
    mat = rng.uniform(0.5, 2.0, size=R)
    tr = w.sum(axis=1) / 500.0
    res = [O.simulate(w, 800.0, 0.0, 2, U, m, mat, tr) for m in (O.MODE_SLIME, O.MODE_CGP, O.MODE_CGP_FGD)]
    assert res[0].compute == res[1].compute == res[2].compute
    assert res[1].t_train_end <= res[0].t_train_end + 1e-9
    assert res[1].t_start <= res[0].t_start
    assert res[2].t_first_U <= res[1].t_first_U + 1e-9                    # FGD lowers t_first^(U)
    for r in res:
        assert sorted(g for u in r.update_groups for g in u) == list(range(R))
        assert all(s >= rd for s, rd in zip(r.start, r.ready))
        assert all(r.start[j + 1] >= r.end[j] for j in range(len(r.start) - 1))
