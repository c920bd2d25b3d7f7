"""GPU tests of the CGP boundary: complete groups enqueued one at a time in
FIFO order, dispatched in logical updates of U groups, cut into launches by
the feasible-prefix rule, gradients and loss only ever accumulated.

BASELINE.json configs[4] ("Streaming CGP arrival"): per-group launches vs 4-group batched launches on
separate CUDA streams vs a single full-batch step must agree to fp32 summation-order noise, and every one of
them must match the float64 oracle of the full batch."""
import numpy as np
import pytest
import torch

from tests.parity_util import TOL_GRAD_REL, TOL_LOGP_ABS, TOL_LOSS_REL, make_ctx, rel_l2, run_cuda, run_oracle, to64
from workloads.synth import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2606_26997_b200.build import build
    build()


@pytest.fixture(scope="module")
def batch():
    # configs[4] shape recipe (32 groups x G=8, geometric lengths, arrival order seeded), shrunk: 8 groups,
    # d=128, V=3000, lengths / 25 (T ~ 5k): several 128x256 tiles, ragged tails, multiple backward chunks
    b = make_config(5, device="cuda", d=128, V=3000, n_groups=8, len_div=25.0, w_std=0.08, old_sigma=0.3,
                    kl_beta=0.002)
    ref = run_oracle(b, loss_denom=float(b.T))
    return b, ref


def _group_descs(ctx, b, order, want_dh=True, want_logp=True):
    """One descriptor per group in arrival `order`, plus the per-group output tensors."""
    descs, outs = [], {}
    for g in order:
        t0, t1 = b.group_token_range(int(g))
        dh = torch.zeros(t1 - t0, b.d, dtype=torch.bfloat16, device="cuda") if want_dh else None
        lp = torch.zeros(t1 - t0, dtype=torch.float32, device="cuda") if want_logp else None
        outs[int(g)] = (dh, lp)
        descs.append(ctx.make_group_desc(
            int(g), b.seqlens[g * b.G:(g + 1) * b.G], b.hidden[t0:t1], b.targets[t0:t1], b.old_logp[t0:t1],
            b.rewards[g * b.G:(g + 1) * b.G].contiguous(), None if b.ref_logp is None else b.ref_logp[t0:t1],
            None if b.mask is None else b.mask[t0:t1], dh, lp))
    return descs, outs


def _gather(b, outs):
    dH = torch.empty(b.T, b.d, dtype=torch.bfloat16, device="cuda")
    lp = torch.empty(b.T, dtype=torch.float32, device="cuda")
    for g, (dh, l) in outs.items():
        t0, t1 = b.group_token_range(g)
        dH[t0:t1] = dh
        lp[t0:t1] = l
    return dH, lp


def _stream_run(b, U, n_streams, token_budget=0, loss_denom=None, per_call=1, order=None, drain=False):
    """Enqueue groups `per_call` at a time in arrival order; returns accumulated outputs + bookkeeping.
    drain: a call runs at most ONE logical update, so with several groups per call keep calling with n = 0 while
    a whole update is pending, and flush until the FIFO is empty."""
    order = list(b.arrival_order if order is None else order)
    ctx = make_ctx(b, groups_per_update=U, token_budget=token_budget, groups_per_round=len(order),
                   max_tokens=b.T, n_slots=n_streams, bwd_chunk_tokens=1024)
    streams = [torch.cuda.Stream() for _ in range(n_streams)]
    dW = torch.zeros(b.V, b.d, dtype=torch.float32, device="cuda")
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")
    metrics = torch.zeros(4, dtype=torch.float32, device="cuda")
    descs, outs = _group_descs(ctx, b, order)
    torch.cuda.synchronize()
    denom = float(b.T) if loss_denom is None else loss_denom
    log = []
    for i in range(0, len(descs), per_call):
        consumed, boundary = ctx.grpo_enqueue_groups(descs[i:i + per_call], b.W, dW, loss, metrics, loss_denom=denom,
                                                     streams=streams)
        log.append((consumed, boundary))
        while drain and ctx.grpo_queue_state()["pending_groups"] >= U:
            log.append(ctx.grpo_enqueue_groups([], b.W, dW, loss, metrics, loss_denom=denom, streams=streams))
    while ctx.grpo_queue_state()["pending_groups"]:
        consumed, boundary = ctx.grpo_flush(b.W, dW, loss, metrics, loss_denom=denom, streams=streams)
        log.append((consumed, boundary))
        if not drain:
            break
    torch.cuda.synchronize()
    assert ctx.grpo_check_errors_sync() == 0
    state = ctx.grpo_queue_state()
    launches = ctx.grpo_kernel_launches()
    ctx.close()
    dH, lp = _gather(b, outs)
    return dict(dW=dW, loss=loss, metrics=metrics, dH=dH, logp=lp, log=log, state=state, launches=launches)


def _assert_oracle(b, out, ref):
    assert np.abs(to64(out["logp"]) - ref["logp"]).max() <= TOL_LOGP_ABS
    assert abs(out["loss"].item() - ref["loss"]) <= TOL_LOSS_REL * max(abs(ref["loss"]), ref["abs_loss"])
    assert rel_l2(to64(out["dH"]), ref["dH"]) <= TOL_GRAD_REL
    assert rel_l2(to64(out["dW"]), ref["dW"]) <= TOL_GRAD_REL
    np.testing.assert_allclose(to64(out["metrics"]), ref["metrics"], rtol=1e-4, atol=1e-3)


def test_per_group_vs_batched_vs_full_batch(batch):
    b, ref = batch
    per_group = _stream_run(b, U=1, n_streams=1)                       # (i) one launch per complete group
    batched = _stream_run(b, U=4, n_streams=2)                         # (ii) 4-group launches on 2 streams
    ctx = make_ctx(b, bwd_chunk_tokens=1024)
    full = run_cuda(ctx, b, loss_denom=float(b.T))                     # (iii) a single full-batch step
    ctx.close()
    for out in (per_group, batched, full):
        _assert_oracle(b, out, ref)
    for out in (per_group, batched):
        # Batch invariance (CGP changes "only group dispatch timing and order - not samples,
        # advantages, or gradient computation"): the vocab split of A2 and the K split of A5 depend on V alone, so
        # a token's log-prob and dHidden row have the same BITS whatever launch it was part of; dW and the loss are
        # sums over tokens accumulated with fp32 atomics, equal up to summation order (1e-5).
        assert torch.equal(out["logp"], full["logp"])
        assert torch.equal(out["dH"], full["dH"])
        assert rel_l2(to64(out["dW"]), to64(full["dW"])) <= 1e-5
        np.testing.assert_allclose(out["loss"].item(), full["loss"].item(), rtol=1e-5)
    # bookkeeping: U=1 -> a boundary after every group; U=4 -> after the 4th and 8th group
    assert [l[1] for l in per_group["log"]] == [True] * 8
    assert [l[0] for l in per_group["log"]] == list(range(1, 9))
    assert [l[1] for l in batched["log"]] == [False, False, False, True, False, False, False, True]
    assert batched["state"]["round_complete"] and batched["state"]["consumed_groups"] == 8
    assert per_group["launches"]["gemm_lse"] == 8 and batched["launches"]["gemm_lse"] == 2


def test_token_budget_cuts_update_into_whole_group_launches(batch):
    b, ref = batch
    toks = [int(b.seqlens[g * b.G:(g + 1) * b.G].sum()) for g in b.arrival_order]
    budget = max(toks) + min(toks)                                      # some pairs fit, not all 8 groups
    from paper_2606_26997_b200 import grpo_cgp_plan
    plan = grpo_cgp_plan(toks, U=8, token_budget=budget)
    assert sum(plan) == 8 and len(plan) > 1
    out = _stream_run(b, U=8, n_streams=3, token_budget=budget)
    _assert_oracle(b, out, ref)
    assert out["launches"]["gemm_lse"] == len(plan)
    assert [l[1] for l in out["log"]] == [False] * 7 + [True]


def test_implicit_denominator_is_the_whole_update(batch):
    """loss_denom <= 0: the library counts the loss-bearing tokens of ALL groups of the update before the
    first launch (R10), so a split update still equals the full-batch token mean."""
    b, ref = batch
    toks = [int(b.seqlens[g * b.G:(g + 1) * b.G].sum()) for g in b.arrival_order]
    out = _stream_run(b, U=8, n_streams=2, token_budget=max(toks), loss_denom=0.0, per_call=8)
    _assert_oracle(b, out, ref)
    assert out["launches"]["gemm_lse"] > 1


def test_flush_runs_a_short_final_update(batch):
    b, ref = batch
    out = _stream_run(b, U=3, n_streams=1)                             # 8 = 3 + 3 + 2 (flushed)
    assert [l[1] for l in out["log"]] == [False, False, True, False, False, True, False, False, True]
    assert out["log"][-1][0] == 8
    _assert_oracle(b, out, ref)


def test_fifo_is_by_arrival_not_by_group_order(batch):
    """groups are consumed in the order they are appended; group_order is informational."""
    b, ref = batch
    order = list(reversed(range(b.n_groups)))
    out = _stream_run(b, U=2, n_streams=2, order=order)
    _assert_oracle(b, out, ref)


def test_incomplete_groups_are_rejected_and_nothing_is_appended(batch):
    from paper_2606_26997_b200.binding import GrpoError
    b, _ = batch
    ctx = make_ctx(b, groups_per_update=2, max_tokens=b.T, max_pending_groups=3)
    dW = torch.zeros(b.V, b.d, dtype=torch.float32, device="cuda")
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")
    descs, _ = _group_descs(ctx, b, [0, 1, 2, 3, 4])
    bad = ctx.make_group_desc(9, b.seqlens[:b.G - 1], b.hidden, b.targets, b.old_logp, b.rewards)   # G-1 responses
    with pytest.raises(GrpoError) as e:
        ctx.grpo_enqueue_groups([descs[0], bad], b.W, dW, loss)
    assert e.value.status == 6 and ctx.grpo_queue_state()["pending_groups"] == 0
    t0, t1 = b.group_token_range(0)
    no_rewards = ctx.make_group_desc(0, b.seqlens[:b.G], b.hidden[t0:t1], b.targets[t0:t1], b.old_logp[t0:t1], None)
    with pytest.raises(GrpoError) as e:
        ctx.grpo_enqueue_groups([no_rewards], b.W, dW, loss)
    assert e.value.status == 6
    # capacity: 3 pending at most; one group waits (U = 2), a 4-group append would overflow
    assert ctx.grpo_enqueue_groups(descs[:1], b.W, dW, loss) == (0, False)
    with pytest.raises(GrpoError) as e:
        ctx.grpo_enqueue_groups(descs[1:5], b.W, dW, loss)
    assert e.value.status == 7 and ctx.grpo_queue_state()["pending_groups"] == 1
    assert ctx.grpo_enqueue_groups(descs[1:2], b.W, dW, loss) == (2, True)
    torch.cuda.synchronize()
    ctx.grpo_reset_round()
    assert ctx.grpo_queue_state() == dict(pending_groups=0, pending_tokens=0, consumed_groups=0, round_complete=False)
    ctx.close()


def test_per_sequence_mean_under_a_budget_cut_equals_the_full_update(batch):
    """loss_agg = 1 (per-sequence mean, then mean over sequences): when the token budget cuts one logical update
    of U groups into several launches, every launch still divides by the sequence count of the WHOLE update
    (R10), so the result is the oracle's full-update step."""
    b0, _ = batch
    b = make_config(5, device="cuda", d=128, V=3000, n_groups=8, len_div=25.0, w_std=0.08, old_sigma=0.3,
                    kl_beta=0.002, loss_agg=1)
    ref = run_oracle(b)
    toks = [int(b.seqlens[g * b.G:(g + 1) * b.G].sum()) for g in b.arrival_order]
    out = _stream_run(b, U=8, n_streams=2, token_budget=max(toks) + min(toks), loss_denom=0.0, per_call=8)
    assert out["launches"]["gemm_lse"] > 1
    _assert_oracle(b, out, ref)
    out = _stream_run(b, U=4, n_streams=1, token_budget=max(toks), loss_denom=0.0)
    # two updates of 4 groups, each averaged over its own 4 x G sequences: the sum is 2 x the full 8-group mean
    assert abs(out["loss"].item() / 2 - ref["loss"]) <= TOL_LOSS_REL * max(abs(ref["loss"]), ref["abs_loss"])
    assert rel_l2(to64(out["dW"]) / 2, ref["dW"]) <= TOL_GRAD_REL


def test_direct_forward_in_micro_batches_with_seq_denom(batch):
    """grpo_set_seq_denom: a caller that cuts one loss_agg = 1 update into several direct forward calls."""
    b = make_config(5, device="cuda", d=128, V=3000, n_groups=4, len_div=25.0, w_std=0.08, old_sigma=0.3,
                    kl_beta=0.002, loss_agg=1)
    ref = run_oracle(b)
    ctx = make_ctx(b, max_tokens=b.T)
    ctx.grpo_set_seq_denom(b.S)
    adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")
    dW = torch.zeros(b.V, b.d, dtype=torch.float32, device="cuda")
    for g in range(b.n_groups):
        t0, t1 = b.group_token_range(g)
        cu = (b.cu_seqlens[g * b.G:(g + 1) * b.G + 1] - t0).contiguous()
        f = ctx.grpo_fused_logprob_loss_fwd(b.hidden[t0:t1], b.W, b.targets[t0:t1], cu, adv[g * b.G:(g + 1) * b.G].contiguous(),
                                            b.old_logp[t0:t1], b.ref_logp[t0:t1], loss_accum=loss)
        ctx.grpo_fused_logprob_loss_bwd(b.hidden[t0:t1], b.W, b.targets[t0:t1], f["lse"], f["coeff"], dW_accum=dW,
                                        want_dhidden=False)
    torch.cuda.synchronize()
    ctx.close()
    assert abs(loss.item() - ref["loss"]) <= TOL_LOSS_REL * max(abs(ref["loss"]), ref["abs_loss"])
    assert rel_l2(to64(dW), ref["dW"]) <= TOL_GRAD_REL


def test_an_update_that_cannot_run_is_rejected_before_anything_is_accumulated(batch):
    """An update whose SECOND launch does not fit the workspace: every launch is validated before the first kernel
    is enqueued, so the accumulators stay untouched, the FIFO keeps both groups and nothing is counted as
    consumed; after the workspace is enlarged the same update runs once and matches the oracle."""
    from paper_2606_26997_b200.binding import GrpoError
    b, _ = batch
    toks = [int(b.seqlens[g * b.G:(g + 1) * b.G].sum()) for g in range(b.n_groups)]
    small, big = int(np.argmin(toks)), int(np.argmax(toks))
    assert toks[small] < toks[big]
    ctx = make_ctx(b, groups_per_update=2, token_budget=toks[small], max_tokens=toks[small], bwd_chunk_tokens=1024)
    dW = torch.zeros(b.V, b.d, dtype=torch.float32, device="cuda")
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")
    descs, outs = _group_descs(ctx, b, [small, big])
    denom = float(toks[small] + toks[big])
    with pytest.raises(GrpoError) as e:
        ctx.grpo_enqueue_groups(descs, b.W, dW, loss, loss_denom=denom)     # launch 2 (the big group) cannot run
    assert e.value.status == 3                                              # GRPO_ERR_WORKSPACE
    torch.cuda.synchronize()
    st = ctx.grpo_queue_state()
    assert st["pending_groups"] == 2 and st["consumed_groups"] == 0
    assert loss.item() == 0.0 and not dW.any() and ctx.grpo_kernel_launches()["gemm_lse"] == 0
    ctx.ensure_workspace(toks[big])
    consumed, boundary = ctx.grpo_enqueue_groups([], b.W, dW, loss, loss_denom=denom)   # n = 0: retry the update
    torch.cuda.synchronize()
    assert (consumed, boundary) == (2, True) and ctx.grpo_kernel_launches()["gemm_lse"] == 2
    ctx.close()
    from workloads.synth import slice_groups
    sub = slice_groups(b, [small, big])
    ref = run_oracle(sub)
    assert abs(loss.item() - ref["loss"]) <= TOL_LOSS_REL * max(abs(ref["loss"]), ref["abs_loss"])
    assert rel_l2(to64(dW), ref["dW"]) <= TOL_GRAD_REL


def test_binding_drops_group_tensors_once_their_launches_have_run(batch):
    """The ctypes binding keeps a group's tensors alive while the library may still read them and not longer:
    queued descriptors wait in FIFO order, consumed ones behind an event on the launch streams."""
    b, _ = batch
    order = list(b.arrival_order)
    ctx = make_ctx(b, groups_per_update=2, max_tokens=b.T, bwd_chunk_tokens=1024)
    dW = torch.zeros(b.V, b.d, dtype=torch.float32, device="cuda")
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")
    descs, _ = _group_descs(ctx, b, order)
    ctx.grpo_enqueue_groups(descs[:1], b.W, dW, loss, loss_denom=float(b.T))
    assert len(ctx._keep) == 1 and not ctx._inflight            # U = 2: queued, nothing launched
    ctx.grpo_enqueue_groups(descs[1:2], b.W, dW, loss, loss_denom=float(b.T))
    assert len(ctx._keep) == 0 and sum(len(d) for _, d in ctx._inflight) in (0, 2)   # 0: already finished
    torch.cuda.synchronize()
    ctx.grpo_enqueue_groups(descs[2:3], b.W, dW, loss, loss_denom=float(b.T))
    assert len(ctx._keep) == 1 and not ctx._inflight            # the first update has run: dropped
    bad = ctx.make_group_desc(99, [0] * b.G, b.hidden, b.targets, b.old_logp, b.rewards[:b.G].contiguous())
    with pytest.raises(Exception):
        ctx.grpo_enqueue_groups([bad], b.W, dW, loss, loss_denom=float(b.T))
    assert len(ctx._keep) == 1                                  # a rejected group is not kept
    ctx.grpo_flush(b.W, dW, loss, loss_denom=float(b.T))
    torch.cuda.synchronize()
    ctx.grpo_flush(b.W, dW, loss, loss_denom=float(b.T))        # nothing pending; retires what has finished
    assert not ctx._keep and not ctx._inflight
    assert ctx.grpo_queue_state()["consumed_groups"] == 3
    ctx.close()


@pytest.mark.parametrize("case", range(12))
def test_random_dispatch_schedules_do_not_change_the_results(case):
    """Seeded random CGP schedules (groups per update, token budget, number of streams, groups per call, arrival
    order, both aggregations): whatever the schedule, every token's log-prob and dHidden row have the bits of the
    single full-batch step, dW and the loss agree to summation order, the launches are the planner's, and the
    result matches the oracle of the full batch."""
    from paper_2606_26997_b200 import grpo_cgp_plan
    rng = np.random.default_rng(9100 + case)
    n_groups = int(rng.integers(3, 9))
    loss_agg = int(rng.integers(0, 2))
    b = make_config(5, device="cuda", seed=case, d=int(rng.choice([64, 128, 200])), V=int(rng.integers(300, 3000)),
                    n_groups=n_groups, G=int(rng.integers(2, 5)), len_div=float(rng.choice([25.0, 60.0])), w_std=0.08,
                    old_sigma=0.3, kl_beta=float(rng.choice([0.0, 0.002])), mask_frac=float(rng.choice([0.0, 0.2])),
                    loss_agg=loss_agg)
    order = list(rng.permutation(n_groups))
    toks = [int(b.seqlens[g * b.G:(g + 1) * b.G].sum()) for g in order]
    U = int(rng.integers(1, n_groups + 1))
    budget = int(rng.choice([0, max(toks), max(toks) + min(toks), sum(toks) // 2 + 1]))
    n_streams = int(rng.integers(1, 4))
    ref = run_oracle(b, loss_denom=float(b.T))
    out = _stream_run(b, U=U, n_streams=n_streams, token_budget=budget, per_call=int(rng.integers(1, 4)), order=order,
                      drain=True)
    ctx = make_ctx(b, bwd_chunk_tokens=1024)
    full = run_cuda(ctx, b, loss_denom=float(b.T))
    ctx.close()
    if loss_agg == 0 or U >= n_groups:
        # (per-sequence mean: the logical update is the unit the mean is taken over, so only a schedule with ONE
        # update equals the full-batch step; the token mean has its denominator passed in)
        _assert_oracle(b, out, ref)
        assert torch.equal(out["logp"], full["logp"]) and torch.equal(out["dH"], full["dH"])
        assert rel_l2(to64(out["dW"]), to64(full["dW"])) <= 1e-5
    else:
        assert torch.equal(out["logp"], full["logp"])
    # the launches are the planner's: whole-group prefixes per update of U groups, the last update flushed short
    expect, pos = 0, 0
    while pos < n_groups:
        plan = grpo_cgp_plan(toks[pos:], U=U, token_budget=budget, flush=True)
        expect += len(plan)
        pos += sum(plan)
    assert out["launches"]["gemm_lse"] == expect and out["state"]["consumed_groups"] == n_groups
