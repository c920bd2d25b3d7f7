"""GPU parity of the NEXT-2 rows: k1 / k2 KL estimators, dual clip, and zero-coefficient
tile skipping in the backward, through the C ABI against the float64 oracle (same gates as test_parity_gpu)."""
import numpy as np
import pytest
import torch

from tests.parity_util import assert_gates, gates, make_ctx, rel_l2, run_cuda, run_oracle, to64
from workloads.synth import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2606_26997_b200.build import build
    build()


@pytest.mark.parametrize("kl_type,dual", [(1, 0.0), (2, 0.0), (0, 1.6), (2, 1.6), (1, 1.5)])
def test_kl_estimators_and_dual_clip(kl_type, dual):
    b = make_config(1, device="cuda", seed=11, variant="1b", old_sigma=0.6, kl_beta=0.05)
    ctx = make_ctx(b, kl_type=kl_type, dual_clip=dual, dhidden_fp32=1)
    try:
        out = run_cuda(ctx, b)
    finally:
        ctx.close()
    ref = run_oracle(b, kl_type=kl_type, dual_clip=dual)
    e = gates(b, out, ref)
    assert_gates(e)
    assert to64(out["metrics"])[3] == ref["metrics"][3]                  # the same tokens lose their gradient
    if dual:
        base = run_oracle(b, kl_type=kl_type)
        assert ref["metrics"][3] > base["metrics"][3]                    # the dual clip is active in this case


def test_bad_variant_arguments_are_rejected():
    from paper_2606_26997_b200 import GrpoContext, GrpoError
    with pytest.raises(GrpoError):
        GrpoContext(64, 1000, kl_type=3)
    with pytest.raises(GrpoError):
        GrpoContext(64, 1000, dual_clip=0.5)


def _skippable_batch(beta=0.0):
    # 6 groups x 4 responses of ~190 tokens (T ~ 4.5k: ~18 pair tiles of 256 rows); groups 1, 3, 4 are
    # zero-variance, so at beta = 0 every token of theirs has coefficient exactly 0; plus a masked span
    b = make_config(3, device="cuda", seed=2, d=64, V=1000, n_groups=6, G=4, len_div=8.0, kl_beta=beta)
    r = b.rewards.clone().reshape(6, 4)
    r[0] = torch.tensor([1.0, 0.0, 0.0, 1.0]); r[2] = torch.tensor([0.0, 1.0, 1.0, 1.0]); r[5] = torch.tensor([1.0, 0.0, 0.0, 0.0])
    r[1] = 1.0; r[3] = 0.0; r[4] = 1.0
    b.rewards = r.reshape(-1).contiguous()
    m = torch.ones(b.T, dtype=torch.uint8, device="cuda")
    lo, hi = b.group_token_range(0)
    m[lo:lo + 300] = 0
    b.mask = m
    return b


@pytest.mark.parametrize("cg", [2, 1])
def test_zero_coefficient_rows_are_skipped_and_results_match_the_oracle(cg):
    b = _skippable_batch()
    ctx = make_ctx(b, gemm_cta_group=cg, bwd_chunk_tokens=2048, dhidden_fp32=1)
    try:
        ctx.ensure_workspace(b.T)
        ctx.grpo_bwd_row_stats_sync()
        out = run_cuda(ctx, b)
        active, total = ctx.grpo_bwd_row_stats_sync()
    finally:
        ctx.close()
    ref = run_oracle(b)
    assert_gates(gates(b, out, ref))
    assert total == b.T and active == int((ref["coeff"] != 0.0).sum()) and active <= 0.75 * total, (active, total)
    # rows of zero-coefficient tokens are exact zeros, as in the dense computation
    zero_rows = ref["coeff"] == 0.0
    assert zero_rows.sum() > 1000
    assert torch.all(out["dH"][torch.from_numpy(zero_rows).cuda()] == 0)


def test_skipping_on_and_off_agree():
    b = _skippable_batch()
    outs = []
    for skip in (0, -1):
        ctx = make_ctx(b, bwd_skip_zero_tiles=skip, bwd_chunk_tokens=2048)
        try:
            ctx.ensure_workspace(b.T)
            ctx.grpo_bwd_row_stats_sync()
            outs.append(run_cuda(ctx, b))
            st = ctx.grpo_bwd_row_stats_sync()
            assert (st[1] > 0) == (skip == 0)
        finally:
            ctx.close()
    assert torch.equal(outs[0]["dH"], outs[1]["dH"])                     # every active row is computed identically
    assert rel_l2(to64(outs[0]["dW"]), to64(outs[1]["dW"])) < 1e-5       # other rows share a k block: summation order only


def test_nothing_is_skipped_when_the_kl_term_gives_every_token_a_gradient():
    b = _skippable_batch(beta=0.01)
    b.mask = None
    ctx = make_ctx(b, bwd_chunk_tokens=2048)
    try:
        ctx.ensure_workspace(b.T)
        ctx.grpo_bwd_row_stats_sync()
        out = run_cuda(ctx, b)
        active, total = ctx.grpo_bwd_row_stats_sync()
    finally:
        ctx.close()
    assert active == total > 0
    assert_gates(gates(b, out, run_oracle(b)))


def test_all_tiles_zero_gives_zero_gradients():
    b = make_config(1, device="cuda", seed=8, kl_beta=0.0)
    b.rewards = torch.ones_like(b.rewards)                               # every group zero-variance
    ctx = make_ctx(b)
    try:
        out = run_cuda(ctx, b)
    finally:
        ctx.close()
    assert torch.all(out["dH"] == 0) and torch.all(out["dW"] == 0)


# ------------------------------------------------------------------ per-token entropy output (R28)
@pytest.mark.parametrize("fused", [False, True])
@pytest.mark.parametrize("w_std,scale", [(0.02, 1.0), (1.0, 0.8), (3.0, 1.3)])
def test_entropy_output(fused, w_std, scale):
    """V = 1000 leaves 24 padding columns in the last 32-column chunk and T ~ 320 splits the vocab over many
    CTA pairs (partial sums combined in A3); w_std spans near-uniform to sharply peaked policies."""
    from oracle.grpo_oracle import token_entropy
    b = make_config(1, device="cuda", seed=13, variant="1b", w_std=w_std, bad_target_frac=0.1)
    ctx = make_ctx(b, logit_scale=scale, bwd_chunk_tokens=128)
    try:
        ent = torch.full((b.T,), float("nan"), dtype=torch.float32, device="cuda")
        ctx.grpo_set_entropy_out(ent)
        out = run_cuda(ctx, b, fused=fused)
        ctx.grpo_set_entropy_out(None)
        ent2 = ent.clone()
        run_cuda(ctx, b, fused=fused)                                      # off again: the buffer is not touched
        assert torch.equal(ent, ent2)
    finally:
        ctx.close()
    x = b.numpy_f64()
    ref = token_entropy(x["H"], x["W"], logit_scale=scale)
    assert np.abs(to64(ent) - ref).max() <= 2e-3, np.abs(to64(ent) - ref).max()
    assert_gates(gates(b, out, run_oracle(b, logit_scale=scale), logit_scale=scale))   # the rest is unchanged


def test_entropy_output_full_vocab_sampled_rows():
    from oracle.grpo_oracle import token_entropy
    b = make_config(2, device="cuda", seed=1, len_div=16.0)               # d = 2048, V = 151936, T ~ 1.2k
    ctx = make_ctx(b)
    try:
        ent = torch.zeros(b.T, dtype=torch.float32, device="cuda")
        ctx.grpo_set_entropy_out(ent)
        run_cuda(ctx, b, want_dw=False, want_dh=False)
    finally:
        ctx.close()
    rows = np.unique(np.concatenate([[0, 127, 128, b.T - 1], np.random.default_rng(0).choice(b.T, 24, replace=False)]))
    x = b.numpy_f64()
    ref = token_entropy(x["H"][rows], x["W"])
    assert np.abs(to64(ent)[rows] - ref).max() <= 2e-3
    assert 11.0 < ref.min() and ref.max() < np.log(151936.0)              # near-uniform synthetic softmax
