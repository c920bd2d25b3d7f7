"""grpo_loss_from_partials_static: the A3 loss launch for callers that cannot allocate GPU memory.

Who that is: a trainer whose framework already owns all of HBM through its caching allocator, a step that must not
stall the streams next to it with cudaMalloc's device-wide synchronisation (the rollout / training overlap of
PAPER.md:92-111), a loss-only rank of a vocab-parallel job that holds no vocab shard.  The entry point takes no
context and no workspace; its scratch (block sums, arrival counter, token counts) is an array built into
libgrpo_b200.so, one per GPU, shared by every call and keeping the last call's contents.

What is checked: on two calls in a row with different shapes and switches (the second smaller than the first, so the
array still holds the first call's block sums and counts), every output equals what the existing workspace path
(GrpoContext.grpo_loss_from_partials) gives on the same gathered partials, within the tolerances the vocab-parallel
tests use for two CUDA runs of the same arithmetic; a third call repeats the first and must reproduce it bit for bit.
Sizes beyond the stated maximum are refused before anything is launched.

This file is named to be collected last: `pytest -x` stops at the first failure and a failure here must not hide the
other tests.  It needs nothing from them and passes alone in a fresh process (the first call does the per-device
set-up itself).
"""
import pytest
import torch

from tests.parity_util import rel_l2, to64
from workloads.synth import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2606_26997_b200.build import build
    build()


def _gathered_partials(b, bounds):
    """The existing path up to the exchange: one context per vocab shard, stacked [n_shards, T] partials."""
    from paper_2606_26997_b200 import GrpoContext
    parts = []
    for r in range(len(bounds) - 1):
        ctx = GrpoContext(b.d, bounds[r + 1] - bounds[r], max_tokens=b.T, group_size=b.G)
        y_loc = torch.where(b.targets < 0, torch.full_like(b.targets, -1), b.targets - bounds[r]).contiguous()
        parts.append(ctx.grpo_vocab_shard_partials(b.hidden, b.W[bounds[r]:bounds[r + 1]].contiguous(), y_loc))
        torch.cuda.synchronize()
        ctx.close()
    return tuple(torch.stack([p[i] for p in parts]).contiguous() for i in range(3))


def _existing(b, parts, **switches):
    from paper_2606_26997_b200 import GrpoContext
    ctx = GrpoContext(b.d, b.V, max_tokens=b.T, group_size=b.G, eps_std=b.eps_std, **switches)
    adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
    metrics = torch.zeros(4, dtype=torch.float32, device="cuda")
    f = ctx.grpo_loss_from_partials(*parts, b.targets, b.V, b.cu_seqlens, adv, b.old_logp, b.ref_logp, b.mask,
                                    metrics_accum=metrics)
    torch.cuda.synchronize()
    ctx.close()
    return dict(adv=adv, metrics=metrics, **f)


def _static(b, parts, adv, **switches):
    from paper_2606_26997_b200 import grpo_loss_from_partials_static
    out = dict(logp=torch.full((b.T,), 7.0, device="cuda"), lse=torch.full((b.T,), 7.0, device="cuda"),
               coeff=torch.full((b.T,), 7.0, device="cuda"), loss=torch.zeros(1, device="cuda"),
               metrics=torch.zeros(4, device="cuda"))
    err = torch.zeros(1, dtype=torch.int32, device="cuda")
    grpo_loss_from_partials_static(*parts, b.targets, b.V, b.cu_seqlens, adv, b.old_logp, out, ref_logp=b.ref_logp,
                                   mask=b.mask, err_flags=err, **switches)
    torch.cuda.synchronize()
    assert err.item() == 0
    return out


def _same(new, old):
    assert (new["logp"] - old["logp"]).abs().max().item() <= 2e-5
    assert (new["lse"] - old["lse"]).abs().max().item() <= 2e-5
    assert rel_l2(to64(new["coeff"]), to64(old["coeff"])) <= 1e-6
    assert abs(new["loss"].item() - old["loss"].item()) <= 1e-6 * max(abs(old["loss"].item()), 1e-6)
    m_new, m_old = to64(new["metrics"]), to64(old["metrics"])
    assert m_new[0] == m_old[0] and m_new[3] == m_old[3]            # token and clip counts are integers
    assert abs(m_new[1] - m_old[1]) <= 1e-5 * abs(m_old[1]) and abs(m_new[2] - m_old[2]) <= 1e-5 * abs(m_old[2]) + 1e-7


def test_static_scratch_loss_equals_the_workspace_path_on_consecutive_calls():
    # call 1: token mean with the denominator counted on the device, clip populated, KL off
    big = make_config(1, device="cuda", seed=20, variant="1b", n_groups=6, G=4, d=128, V=3000, len_div=0.25, w_std=0.1,
                      mask_frac=0.2, bad_target_frac=0.1)
    sw_big = dict(clip_lo=big.clip_lo, clip_hi=big.clip_hi, kl_beta=big.kl_beta, loss_agg=0)
    parts_big = _gathered_partials(big, [0, 1024, 2048, 3000])
    # call 2: fewer tokens and sequences, per-sequence mean, k3 KL: the array still holds call 1's sums and counts
    small = make_config(1, device="cuda", seed=23, variant="1b", n_groups=3, G=4, d=128, V=3000, len_div=0.5, w_std=0.1,
                        loss_agg=1, kl_beta=0.05)
    sw_small = dict(clip_lo=small.clip_lo, clip_hi=small.clip_hi, kl_beta=small.kl_beta, loss_agg=1)
    parts_small = _gathered_partials(small, [0, 1504, 3000])
    assert small.T < big.T and small.cu_seqlens.numel() < big.cu_seqlens.numel()

    ref_big, ref_small = _existing(big, parts_big, **sw_big), _existing(small, parts_small, **sw_small)
    got_big = _static(big, parts_big, ref_big["adv"], **sw_big)
    got_small = _static(small, parts_small, ref_small["adv"], **sw_small)
    _same(got_big, ref_big)
    _same(got_small, ref_small)
    assert ref_big["metrics"][3].item() > 0 and ref_small["metrics"][2].item() > 0      # clip and KL legs are live
    again = _static(big, parts_big, ref_big["adv"], **sw_big)
    for k in ("logp", "lse", "coeff", "loss", "metrics"):
        assert torch.equal(again[k], got_big[k]), k


def test_static_scratch_rejects_sizes_beyond_its_array():
    from paper_2606_26997_b200 import GrpoError
    from paper_2606_26997_b200.binding import STATIC_MAX_SEQUENCES, STATIC_MAX_TOKENS, grpo_loss_from_partials_static

    def call(T, S):
        f = lambda n, v=0.0, dt=torch.float32: torch.full((n,), v, dtype=dt, device="cuda")
        out = dict(logp=f(T, 7.0), lse=f(T, 7.0), coeff=f(T, 7.0), loss=f(1))
        cu = torch.linspace(0, T, S + 1, device="cuda").to(torch.int32)
        # one shard with max 0 and sum 1: lse = 0, logp = 0, rho = 1; zero advantages: loss = 0, coeff = 0
        grpo_loss_from_partials_static(f(T).view(1, T), f(T, 1.0).view(1, T), f(T).view(1, T), f(T, 0, torch.int32), 100,
                                       cu, f(S), f(T), out, loss_denom=float(T))
        return out

    for T, S, word in ((STATIC_MAX_TOKENS + 1, 4, "GRPO_STATIC_MAX_TOKENS"),
                       (1024, STATIC_MAX_SEQUENCES + 1, "GRPO_STATIC_MAX_SEQUENCES")):
        with pytest.raises(GrpoError) as e:
            call(T, S)
        assert e.value.status == 3 and word in str(e.value)                 # GRPO_ERR_WORKSPACE, nothing launched
    # exactly at the token limit the call is accepted and the launch covers every row up to T - 1
    out = call(STATIC_MAX_TOKENS, 4)
    torch.cuda.synchronize()
    assert out["loss"].item() == 0.0
    for k in ("logp", "lse", "coeff"):
        assert torch.count_nonzero(out[k]).item() == 0, k
