"""GPU parity of the 3-contraction variant:
grpo_fused_logprob_loss_fwd_bwd stashes each chunk's logits (fp16) in the forward and converts them to dZ in
place instead of recomputing them.  Same oracle, same gates as the north_star path (tests/test_parity_gpu.py)."""
import numpy as np
import pytest
import torch

from tests.parity_util import (TOL_GRAD_REL, TOL_LOGP_ABS, assert_gates, gates, make_ctx, rel_l2, run_cuda,
                               run_oracle, to64)
from tests.test_fullsize_gpu import _check_sampled, _colsum_rel, _oracle_sampled, _sample_tokens
from tests.test_variants_gpu import _skippable_batch
from workloads.synth import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2606_26997_b200.build import build
    build()


def _check(b, ctx_kw=None, oracle_kw=None, loss_denom=0.0, grad_scale=1.0):
    ctx = make_ctx(b, **(ctx_kw or {}))
    try:
        out = run_cuda(ctx, b, loss_denom=loss_denom, grad_scale=grad_scale, fused=True)
        assert ctx.grpo_check_errors_sync() == 0
        n = ctx.grpo_kernel_launches()
        assert n["gemm_dz"] == 0 and n["stash_dz"] > 0 and n["gemm_lse"] == n["stash_dz"]    # nothing recomputed
    finally:
        ctx.close()
    okw = dict(oracle_kw or {})
    ref = run_oracle(b, loss_denom=loss_denom if loss_denom > 0 else None, **okw)
    if grad_scale != 1.0:
        ref["dH"] *= grad_scale
        ref["dW"] *= grad_scale
    e = gates(b, out, ref, logit_scale=okw.get("logit_scale", 1.0), grad_scale=grad_scale)
    assert_gates(e)
    return out, ref, e


@pytest.mark.parametrize("cg", [2, 1])
def test_config1_and_clip_variant(cg):
    out, ref, e = _check(make_config(1, device="cuda"), ctx_kw=dict(gemm_cta_group=cg))
    np.testing.assert_allclose(to64(out["metrics"]), ref["metrics"], rtol=1e-4, atol=1e-4)
    out, ref, _ = _check(make_config(1, device="cuda", variant="1b"), ctx_kw=dict(gemm_cta_group=cg, dhidden_fp32=1))
    assert to64(out["metrics"])[3] == ref["metrics"][3]


@pytest.mark.parametrize("kw", [
    dict(mask_frac=0.25), dict(loss_agg=1, mask_frac=0.3), dict(bad_target_frac=0.15), dict(kl_beta=0.05),
    dict(w_std=1.5), dict(kl_beta=0.0),
])
def test_config1_variants_in_several_chunks(kw):
    # bwd_chunk_tokens = 128 -> 3 chunks of <= 128 rows at T ~ 320: the per-chunk forward must use the
    # whole call's denominators and sequence lookup
    b = make_config(1, device="cuda", seed=3, variant="1b", **kw)
    _check(b, ctx_kw=dict(dhidden_fp32=1, bwd_chunk_tokens=128))


def test_temperature_sample_std_explicit_denominator_and_grad_scale():
    b = make_config(1, device="cuda", seed=4, variant="1b", w_std=0.3)
    _check(b, ctx_kw=dict(std_ddof=1, logit_scale=0.7, bwd_chunk_tokens=256), oracle_kw=dict(std_ddof=1, logit_scale=0.7))
    _check(b, ctx_kw=dict(logit_scale=1.9, dhidden_fp32=1), oracle_kw=dict(logit_scale=1.9), grad_scale=0.25,
           loss_denom=float(b.T) / 3.0)


def test_large_logits_keep_their_precision():
    """|z| up to ~100 (w_std = 3, d = 64, temperature 1/1.3): what is stashed is the exponential relative to the
    row's running max, not the logit, so the relative error of every probability stays at fp16's 2^-11."""
    b = make_config(1, device="cuda", seed=13, variant="1b", w_std=3.0)
    _check(b, ctx_kw=dict(logit_scale=1.3, bwd_chunk_tokens=128, dhidden_fp32=1), oracle_kw=dict(logit_scale=1.3))


def test_agrees_with_the_recompute_path():
    b = make_config(3, device="cuda", seed=5, d=128, V=3000, n_groups=3, G=4, len_div=8.0)
    outs = []
    for fused in (False, True):
        ctx = make_ctx(b, dhidden_fp32=1, bwd_chunk_tokens=1024)
        try:
            outs.append(run_cuda(ctx, b, fused=fused))
        finally:
            ctx.close()
    a, f = outs
    assert np.abs(to64(a["logp"]) - to64(f["logp"])).max() < 1e-5
    assert abs(a["loss"].item() - f["loss"].item()) < 1e-6 * max(1.0, abs(a["loss"].item()))
    assert rel_l2(to64(f["dH"]), to64(a["dH"])) < 5e-3               # fp16 rounding of the stashed logit only
    assert rel_l2(to64(f["dW"]), to64(a["dW"])) < 5e-3


def test_zero_coefficient_rows_are_compacted_in_the_stash_path_too():
    b = _skippable_batch()
    ctx = make_ctx(b, bwd_chunk_tokens=2048, dhidden_fp32=1)
    try:
        ctx.ensure_workspace(b.T)
        ctx.grpo_bwd_row_stats_sync()
        out = run_cuda(ctx, b, fused=True)
        active, total = ctx.grpo_bwd_row_stats_sync()
    finally:
        ctx.close()
    ref = run_oracle(b)
    assert_gates(gates(b, out, ref))
    assert total == b.T and active == int((ref["coeff"] != 0.0).sum()) < total
    assert torch.all(out["dH"][torch.from_numpy(ref["coeff"] == 0.0).cuda()] == 0)


def test_scattered_zeros_and_the_dense_stash_backward_agree():
    """config-1b recipe with beta = 0 and a mask: 20-40 % of the rows, scattered, have a zero coefficient; the
    compacted 3-contraction backward equals the dense one (dHidden rows bit for bit) and the oracle."""
    b = make_config(1, device="cuda", seed=7, variant="1b", n_groups=6, G=8, d=128, V=3000, len_div=0.1, w_std=0.1,
                    kl_beta=0.0, mask_frac=0.15)
    outs = []
    for skip in (0, -1):
        ctx = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=1024, bwd_skip_zero_tiles=skip, dhidden_fp32=1)
        outs.append(run_cuda(ctx, b, fused=True))
        ctx.close()
    assert torch.equal(outs[0]["dH"], outs[1]["dH"])
    assert rel_l2(to64(outs[0]["dW"]), to64(outs[1]["dW"])) < 1e-5
    ref = run_oracle(b)
    assert_gates(gates(b, outs[0], ref))
    assert 0.15 * b.T < (ref["coeff"] == 0).sum() < 0.85 * b.T


def test_step_host_with_stash_logits():
    b = make_config(1, device="cuda", seed=7, variant="1b", kl_beta=0.0)
    ctx = make_ctx(b, stash_logits=1, max_tokens=b.T)
    try:
        dW = torch.zeros(b.V, b.d, dtype=torch.float32, device="cuda")
        pin = lambda t: t.cpu().pin_memory()
        h_logp = torch.empty(b.T, dtype=torch.float32).pin_memory()
        h_dh = torch.empty(b.T, b.d, dtype=torch.bfloat16).pin_memory()
        h_loss = torch.zeros(1, dtype=torch.float32).pin_memory()
        ctx.grpo_step_host(pin(b.hidden), pin(b.targets), pin(b.cu_seqlens), pin(b.rewards), pin(b.old_logp),
                           b.n_groups, b.G, b.W, dW, loss_h=h_loss, logp_h=h_logp, dhidden_h=h_dh)
        n = ctx.grpo_kernel_launches()
        assert n["gemm_dz"] == 0 and n["stash_dz"] > 0
    finally:
        ctx.close()
    ref = run_oracle(b)
    assert np.abs(h_logp.double().numpy() - ref["logp"]).max() <= TOL_LOGP_ABS
    assert rel_l2(h_dh.double().numpy(), ref["dH"]) <= TOL_GRAD_REL
    assert rel_l2(to64(dW), ref["dW"]) <= TOL_GRAD_REL


def test_config3_full_size_sampled_stash():
    """Full size (d = 2048, V = 151936, ~70k tokens, KL, zero-variance groups) in several 9472-token chunks."""
    b = make_config(3, seed=0, device="cuda")
    ctx = make_ctx(b, max_tokens=b.T)
    out = run_cuda(ctx, b, fused=True)
    assert ctx.grpo_check_errors_sync() == 0
    ctx.close()
    rows = _sample_tokens(b, 40, seed=3)
    _check_sampled(b, out, rows, _oracle_sampled(b, rows, float(b.T)))
    assert _colsum_rel(out["dW"]) <= 2e-3
    assert to64(out["metrics"])[0] == b.T
