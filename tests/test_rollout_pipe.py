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


# ------------------------------------------------------------------------------------------- C ABI vs oracle
@pytest.fixture(scope="module")
def rp():
    from paper_2606_26997_b200.build import build
    build()
    from paper_2606_26997_b200 import rollout_pipe
    return rollout_pipe


def test_abi_exports_every_declared_symbol(rp):
    import re
    root = os.path.dirname(os.path.dirname(__file__))
    header = open(os.path.join(root, "include", "rollout_pipe.h")).read()
    declared = set(re.findall(r"^int32_t\s+(rp_\w+)\s*\(", header, flags=re.M))
    assert declared == set(rp.RP_EXPORTS)
    from paper_2606_26997_b200.binding import load_library
    lib = load_library()
    for name in declared:
        getattr(lib, name)


def test_abi_paper_examples(rp):
    assert rp.rp_fgd_frontier([5, 3, 1, 2, 4, 6], 2) == [1, 2]                       # Eq. 5
    K = 4
    work = np.array([[10.0] * K] + [[20.0] * K] * 5)
    _, gdone, trace = rp.rp_rollout(work, 8.0, 0.0, F_w=2, trace_cap=16)
    assert trace[0][1] == [0, 1] and trace[1][1] == [1, 2]
    tl = rp.rp_cgp_timeline([210.0, 250.0], [10.0, 10.0], 2, rp.MODE_CGP)
    assert tl["t_first_U"] == 250.0 and tl["start"][0] - 210.0 == 40.0
    ts = rp.rp_cgp_timeline(np.linspace(200.0, 400.0, 96), np.ones(96), 2, rp.MODE_SLIME)
    assert ts["t_start"] == 400.0 and all(r == 400.0 for r in ts["ready"])


def _round(seed, R, K):
    """Seeded synthetic round with the paper's shape parameters (K = 8, U = 2, F_w = 2, responses of a few
    thousand tokens); stands in for its workloads."""
    rng = np.random.default_rng(seed)
    work = np.minimum(rng.geometric(1.0 / 2000.0, size=(R, K)), 8192).astype(np.float64)
    mat = rng.uniform(0.2, 3.0, size=R)
    train = work.sum(axis=1) / 4500.0          # ~4.5k response tokens/s whole-trainer rate
    return work, mat, train


@pytest.mark.parametrize("seed,R,K,U,F_w,cap", [(0, 32, 8, 2, 2, 0.0), (1, 96, 8, 2, 2, 0.0), (2, 17, 5, 3, 4, 40.0),
                                                (3, 64, 8, 2, 1, 0.0), (4, 6, 2, 4, 9, 25.0), (5, 1, 8, 2, 2, 0.0)])
def test_abi_matches_oracle(rp, seed, R, K, U, F_w, cap):
    work, mat, train = _round(seed, R, K)
    C_tok = 6000.0
    for fw in (0, F_w):
        rd_o, gd_o, tr_o = O.rollout(work, C_tok, cap, fw)
        rd, gd, tr = rp.rp_rollout(work, C_tok, cap, fw, trace_cap=4 * R)
        np.testing.assert_allclose(rd, rd_o, rtol=1e-10, atol=1e-9)
        np.testing.assert_allclose(gd, gd_o, rtol=1e-10, atol=1e-9)
        if fw > 0:                     # distinct geometric lengths: no simultaneous group completions
            assert [F for _, F in tr] == [F for _, F in tr_o]
            np.testing.assert_allclose([t for t, _ in tr], [t for t, _ in tr_o], rtol=1e-10, atol=1e-9)
    for mode in (O.MODE_SLIME, O.MODE_CGP, O.MODE_CGP_FGD):
        o = O.simulate(work, C_tok, cap, F_w, U, mode, mat, train)
        c = rp.rp_simulate(work, C_tok, cap, F_w, U, mode, mat, train)
        assert c["fifo_order"] == o.fifo_order
        for k in ("t_first_U", "t_complete", "dt_cgp", "t_start", "t_train_end", "compute", "wait", "w_train_eq4",
                  "w_train_alt"):
            assert c[k] == pytest.approx(getattr(o, k), rel=1e-10, abs=1e-9), k
        np.testing.assert_allclose(c["ready"], o.ready, rtol=1e-10, atol=1e-9)
        np.testing.assert_allclose(c["start"], o.start, rtol=1e-10, atol=1e-9)
        np.testing.assert_allclose(c["end"], o.end, rtol=1e-10, atol=1e-9)
        assert c["n_updates"] == len(o.update_groups)


def test_abi_edge_cases(rp):
    tl = rp.rp_cgp_timeline([], [], 2, rp.MODE_CGP)                                   # empty round
    assert tl["n_updates"] == 0 and tl["t_train_end"] == 0.0
    rd, gd, _ = rp.rp_rollout(np.zeros((3, 2)), 10.0)                                 # zero-length responses
    assert np.all(rd == 0.0) and np.all(gd == 0.0)
    with pytest.raises(ValueError):
        rp.rp_rollout(np.ones((2, 2)), 0.0)                                           # capacity must be > 0
    with pytest.raises(ValueError):
        rp.rp_cgp_timeline([1.0], [1.0], 0, rp.MODE_CGP)                              # U >= 1


def test_paper_trend_cgp_gain_grows_with_R(rp):
    """Qualitative claim of section 5.2: the reduction of rollout-to-train-end time over Slime
    grows with R; CGP+FGD starts the trainer earlier than Slime at every R.  Model-level check only."""
    gains = []
    for R in (32, 64, 96):
        work, mat, train = _round(100 + R, R, 8)
        cap_tok = work.sum() / (train.sum())          # rollout and training take about equally long
        s = rp.rp_simulate(work, cap_tok, 0.0, 2, 2, rp.MODE_SLIME, mat, train)
        f = rp.rp_simulate(work, cap_tok, 0.0, 2, 2, rp.MODE_CGP_FGD, mat, train)
        assert f["t_start"] < s["t_start"] and f["compute"] == pytest.approx(s["compute"])
        gains.append(1.0 - f["t_train_end"] / s["t_train_end"])
    assert gains[0] < gains[1] < gains[2]
    assert 0.2 < gains[2] < 0.5


def test_abi_matches_oracle_on_random_small_rounds(rp):
    """Property test: random small rounds (ties between completion times included: integer works, zero-length
    responses, equal materialization latencies) — every output of the C++ model equals the oracle's."""
    from hypothesis import given, settings, strategies as st

    @settings(max_examples=150, deadline=None)
    @given(st.integers(1, 9), st.integers(1, 4), st.integers(1, 4), st.integers(0, 5), st.sampled_from([0.0, 3.0]),
           st.integers(0, 2 ** 31 - 1))
    def check(R, K, U, F_w, cap, seed):
        rng = np.random.default_rng(seed)
        work = rng.integers(0, 6, size=(R, K)).astype(np.float64)
        mat = rng.integers(0, 3, size=R).astype(np.float64)
        train = rng.integers(1, 4, size=R).astype(np.float64)
        rd_o, gd_o, _ = O.rollout(work, 7.0, cap, F_w)
        rd, gd, _ = rp.rp_rollout(work, 7.0, cap, F_w)
        np.testing.assert_allclose(rd, rd_o, rtol=1e-10, atol=1e-9)
        np.testing.assert_allclose(gd, gd_o, rtol=1e-10, atol=1e-9)
        for mode in (O.MODE_SLIME, O.MODE_CGP, O.MODE_CGP_FGD):
            # feed both timelines the oracle's trainable times so that ties are broken on identical inputs
            trainable = (O.rollout(work, 7.0, cap, F_w if mode == O.MODE_CGP_FGD else 0)[1] + mat)
            o = O.cgp_timeline(trainable, train, U, mode)
            c = rp.rp_cgp_timeline(trainable, train, U, mode)
            assert c["fifo_order"] == o.fifo_order
            np.testing.assert_allclose(c["start"], o.start, rtol=1e-12, atol=1e-12)
            np.testing.assert_allclose(c["end"], o.end, rtol=1e-12, atol=1e-12)
            for k in ("t_first_U", "t_complete", "dt_cgp", "t_start", "t_train_end", "compute", "wait"):
                assert c[k] == pytest.approx(getattr(o, k), rel=1e-12, abs=1e-12), k
            assert o.t_train_end >= o.t_complete - 1e-12 or R == 0          # training cannot end before the rollout

    check()
