"""Batch invariance and token-granular compaction of the CUDA path (DESIGN.md sections 5 and 10).

* Batch invariance: CGP changes "only group dispatch timing and order - not samples, advantages, or gradient
  computation".  The vocab split of A2 and the K split of A5 are functions of V alone, so the bits
  of a token's lse / logp / coeff / dHidden row do not depend on which other tokens share its launch, on its
  position in the launch, on the backward chunk length or on the zero-coefficient compaction.
* Compaction: tokens whose coefficient is exactly zero (masked, ignored, clipped at beta = 0 - PAPER.md:38, 40 -
  and zero-variance groups at beta = 0) are removed from the backward at row granularity; the results are those of
  the dense computation and of the float64 oracle, with exact zeros in the skipped dHidden rows."""
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


def _fwd_bwd(ctx, b, rows, denom, adv_tok_seq):
    """Direct forward + backward over the packed rows `rows` (a LongTensor) treated as ONE sequence per token run:
    returns logp, lse, coeff, dH of those rows.  adv_tok_seq: (adv per sequence, cu_seqlens) of the sub-stream."""
    adv, cu = adv_tok_seq
    H = b.hidden[rows].contiguous()
    y = b.targets[rows].contiguous()
    old = b.old_logp[rows].contiguous()
    ref = None if b.ref_logp is None else b.ref_logp[rows].contiguous()
    mask = None if b.mask is None else b.mask[rows].contiguous()
    f = ctx.grpo_fused_logprob_loss_fwd(H, b.W, y, cu, adv, old, ref, mask, loss_denom=denom)
    dH = ctx.grpo_fused_logprob_loss_bwd(H, b.W, y, f["lse"], f["coeff"], dW_accum=None)
    torch.cuda.synchronize()
    return f["logp"], f["lse"], f["coeff"], dH


@pytest.mark.parametrize("V,d", [(6000, 128), (1000, 64), (20000, 256)])
def test_token_results_do_not_depend_on_the_launch_they_are_part_of(V, d):
    b = make_config(5, device="cuda", d=d, V=V, n_groups=6, len_div=20.0, w_std=0.1, old_sigma=0.3, kl_beta=0.002,
                    mask_frac=0.1)
    ctx = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=1024)
    adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
    denom = float(b.T)
    all_rows = torch.arange(b.T, device="cuda")
    full = _fwd_bwd(ctx, b, all_rows, denom, (adv, b.cu_seqlens))
    # (a) every group on its own, (b) the groups in reverse order as one launch, (c) another chunk length
    for g in range(b.n_groups):
        t0, t1 = b.group_token_range(g)
        cu = (b.cu_seqlens[g * b.G:(g + 1) * b.G + 1] - t0).contiguous()
        part = _fwd_bwd(ctx, b, all_rows[t0:t1], denom, (adv[g * b.G:(g + 1) * b.G].contiguous(), cu))
        for a, f in zip(part, full):
            assert torch.equal(a, f[t0:t1])
    order = list(reversed(range(b.n_groups)))
    rows = torch.cat([all_rows[slice(*b.group_token_range(g))] for g in order])
    lens = np.concatenate([b.seqlens[g * b.G:(g + 1) * b.G] for g in order])
    cu = torch.from_numpy(np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)).cuda()
    adv_r = torch.cat([adv[g * b.G:(g + 1) * b.G] for g in order]).contiguous()
    rev = _fwd_bwd(ctx, b, rows, denom, (adv_r, cu))
    for a, f in zip(rev, full):
        assert torch.equal(a, f[rows])
    ctx.close()
    ctx2 = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=512, bwd_skip_zero_tiles=-1)    # other chunks, dense backward
    other = _fwd_bwd(ctx2, b, all_rows, denom, (adv, b.cu_seqlens))
    ctx2.close()
    for a, f in zip(other, full):
        assert torch.equal(a, f)
    # (d) fewer CTAs (SMs left to a concurrent kernel, grpo_config.gemm_max_ctas): another unit-to-CTA deal, same bits
    ctx3 = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=1024, gemm_max_ctas=36)
    fewer = _fwd_bwd(ctx3, b, all_rows, denom, (adv, b.cu_seqlens))
    ctx3.close()
    for a, f in zip(fewer, full):
        assert torch.equal(a, f)


def _offpolicy_batch(beta=0.0, **kw):
    # config-1b recipe at a size spanning several tiles and chunks: old-log-prob noise sigma 0.3 puts 20-40 % of the
    # tokens into the clip regions; beta = 0 makes their coefficient exactly zero
    return make_config(1, device="cuda", seed=7, variant="1b", n_groups=6, G=8, d=128, V=3000, len_div=0.1,
                       w_std=0.1, kl_beta=beta, **kw)


@pytest.mark.parametrize("cg", [2, 1])
def test_clipped_and_masked_tokens_are_compacted_out_of_the_backward(cg):
    b = _offpolicy_batch(mask_frac=0.15, bad_target_frac=0.05)
    assert b.T > 5000
    ctx = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=1024, gemm_cta_group=cg, dhidden_fp32=1)
    ctx.grpo_bwd_row_stats_sync()
    out = run_cuda(ctx, b)
    active, total = ctx.grpo_bwd_row_stats_sync()
    n = ctx.grpo_kernel_launches()
    ctx.close()
    ref = run_oracle(b)
    assert_gates(gates(b, out, ref))
    zero = ref["coeff"] == 0.0
    assert total == b.T and active == int((~zero).sum())
    assert 0.15 * b.T < zero.sum() < 0.85 * b.T                           # scattered zeros, not whole tiles
    assert torch.all(out["dH"][torch.from_numpy(zero).cuda()] == 0)       # exact zeros, as the oracle gives
    assert to64(out["metrics"])[3] == ref["metrics"][3]
    assert n["compact"] > 0 and n["dh_reduce"] == n["gemm_dh"]


def test_compacted_backward_equals_the_dense_backward():
    b = _offpolicy_batch(mask_frac=0.15)
    outs = []
    for skip in (0, -1):
        ctx = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=1024, bwd_skip_zero_tiles=skip)
        outs.append(run_cuda(ctx, b))
        ctx.close()
    assert torch.equal(outs[0]["dH"], outs[1]["dH"])                       # rows are independent: same bits
    assert rel_l2(to64(outs[0]["dW"]), to64(outs[1]["dW"])) < 1e-5        # other rows share a k block: order only


def test_everything_zero_and_nothing_zero():
    # all tokens masked: no backward work at all, gradients exactly zero (R14)
    b = _offpolicy_batch()
    b.mask = torch.zeros(b.T, dtype=torch.uint8, device="cuda")
    ctx = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=1024)
    out = run_cuda(ctx, b)
    assert ctx.grpo_bwd_row_stats_sync() == (0, b.T)
    ctx.close()
    assert not out["dH"].any() and not out["dW"].any() and out["loss"].item() == 0.0
    # KL on: every loss-bearing token has a gradient, nothing is compacted away
    b = _offpolicy_batch(beta=0.01)
    ctx = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=1024)
    out = run_cuda(ctx, b)
    assert ctx.grpo_bwd_row_stats_sync() == (b.T, b.T)
    ctx.close()
    assert_gates(gates(b, out, run_oracle(b)))
