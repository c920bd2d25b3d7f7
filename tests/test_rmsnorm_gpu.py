"""GPU parity of NEXT-4: the final RMSNorm in front of the path and its backward fused behind A5,
against the float64 oracle (oracle.grpo_step_from_prenorm) on the same seeded pre-norm activations.

Tolerances are north_star's (log-prob 2e-3 abs, loss 1e-3 rel, gradients 1e-2 rel-L2), applied to dx and dgamma as
they are to dHidden and dW.  H itself is compared bit for bit: the oracle rounds gamma * x * rstd to bf16 from
float64, the kernel from fp32, so a value within an fp32 rounding error of a bf16 rounding boundary may land on
the other side (R29): at most one bf16 ulp, on a vanishing fraction of the elements."""
import numpy as np
import pytest
import torch

from oracle.grpo_oracle import (OracleConfig, dH_rows, group_advantage, grpo_step_from_prenorm, loss_terms, rmsnorm_bwd,
                                rmsnorm_fwd, token_advantage, token_rows)
from tests.parity_util import TOL_GRAD_REL, TOL_LOGP_ABS, TOL_LOSS_REL, make_ctx, rel_l2, to64
from workloads.synth import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2606_26997_b200.build import build
    build()


def _bf16_ulps_apart(a, b):
    """|a - b| in units of bf16 ulps of b, for tensors on the bf16 grid."""
    ia = a.view(torch.int16).to(torch.int32)
    ib = b.view(torch.int16).to(torch.int32)
    return (ia - ib).abs()


def _run(b, ctx_kw=None, grad_scale=1.0):
    ctx = make_ctx(b, max_tokens=b.T, **(ctx_kw or {}))
    H, rstd = ctx.grpo_rmsnorm_fwd(b.x_prenorm, b.gamma, b.eps_rms)
    adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
    f = ctx.grpo_fused_logprob_loss_fwd(H, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp, b.mask)
    dW = torch.zeros(b.V, b.d, dtype=torch.float32, device="cuda")
    dgamma = torch.zeros(b.d, dtype=torch.float32, device="cuda")
    dx = ctx.grpo_fused_logprob_loss_bwd_prenorm(b.x_prenorm, b.gamma, rstd, H, b.W, b.targets, f["lse"], f["coeff"],
                                                 dgamma, dW_accum=dW, grad_scale=grad_scale)
    torch.cuda.synchronize()
    assert ctx.grpo_check_errors_sync() == 0
    n = ctx.grpo_kernel_launches()
    ctx.close()
    return dict(H=H, rstd=rstd, dx=dx, dgamma=dgamma, dW=dW, launches=n, **f)


def _oracle(b, grad_scale=1.0, **kw):
    x = b.numpy_f64()
    cfg = OracleConfig(eps_std=b.eps_std, clip_lo=b.clip_lo, clip_hi=b.clip_hi, kl_beta=b.kl_beta, loss_agg=b.loss_agg, **kw)
    return grpo_step_from_prenorm(x["x"], x["gamma"], x["W"], x["y"], x["cu_seqlens"], x["rewards"], x["old_logp"],
                                  x["ref_logp"], mask=x["mask"], cfg=cfg, G=b.G, eps_rms=b.eps_rms, grad_scale=grad_scale)


def _assert_parity(b, out, ref):
    ulps = _bf16_ulps_apart(out["H"], torch.tensor(ref["H"], dtype=torch.float32).to(torch.bfloat16).cuda())
    assert ulps.max().item() <= 1 and (ulps != 0).float().mean().item() < 2e-3
    np.testing.assert_allclose(to64(out["rstd"]), ref["rstd"], rtol=2e-6)
    assert np.abs(to64(out["logp"]) - ref["logp"]).max() <= TOL_LOGP_ABS
    assert abs(out["loss"].item() - ref["loss"]) <= TOL_LOSS_REL * max(abs(ref["loss"]), ref["abs_loss"])
    assert rel_l2(to64(out["dx"]), ref["dx"]) <= TOL_GRAD_REL
    assert rel_l2(to64(out["dgamma"]), ref["dgamma"]) <= TOL_GRAD_REL
    assert rel_l2(to64(out["dW"]), ref["dW"]) <= TOL_GRAD_REL
    zero = ref["coeff"] == 0.0
    if zero.any():
        assert torch.all(out["dx"][torch.from_numpy(zero).cuda()] == 0)


@pytest.mark.parametrize("kw", [dict(), dict(variant="1b"), dict(variant="1b", mask_frac=0.2, bad_target_frac=0.1),
                                dict(variant="1b", loss_agg=1, kl_beta=0.0), dict(w_std=0.5)])
def test_config1_from_prenorm_activations(kw):
    b = make_config(1, device="cuda", seed=2, prenorm=True, **kw)
    out = _run(b)
    _assert_parity(b, out, _oracle(b))
    assert out["launches"]["rmsnorm"] == 1 and out["launches"]["dh_reduce"] == out["launches"]["gemm_dh"]


@pytest.mark.parametrize("fp32", [0, 1])
def test_several_tiles_chunks_and_compaction(fp32):
    # clip regions populated, masks: ~half of the rows are compacted away; d = 256 (J = 1), several chunks
    b = make_config(1, device="cuda", seed=4, variant="1b", n_groups=6, G=8, d=256, V=5000, len_div=0.15, w_std=0.1,
                    kl_beta=0.0, mask_frac=0.15, prenorm=True)
    out = _run(b, ctx_kw=dict(bwd_chunk_tokens=1024, dhidden_fp32=fp32), grad_scale=0.5)
    assert out["dx"].dtype == (torch.float32 if fp32 else torch.bfloat16)
    _assert_parity(b, out, _oracle(b, grad_scale=0.5))


def test_wide_hidden_state_and_temperature():
    # d = 2304: J = 3 -> the 4-vector instantiation with a ragged last vector; logit_scale != 1
    b = make_config(1, device="cuda", seed=5, variant="1b", n_groups=2, G=4, d=2304, V=1200, len_div=0.5, prenorm=True)
    ctx_kw = dict(logit_scale=0.8, dhidden_fp32=1)
    out = _run(b, ctx_kw=ctx_kw)
    _assert_parity(b, out, _oracle(b, logit_scale=0.8))


@pytest.mark.parametrize("dh_dtype", [torch.float32, torch.bfloat16])
def test_standalone_backward(dh_dtype):
    b = make_config(1, device="cuda", seed=6, n_groups=3, G=4, d=512, V=1000, len_div=0.3, prenorm=True)
    x = b.numpy_f64()
    g = torch.Generator(device="cuda")
    g.manual_seed(1)
    dH = torch.randn(b.T, b.d, generator=g, device="cuda").to(dh_dtype)
    _, rstd_ref = rmsnorm_fwd(x["x"], x["gamma"], b.eps_rms)
    dx_ref, dg_ref = rmsnorm_bwd(x["x"], x["gamma"], rstd_ref, to64(dH))
    ctx = make_ctx(b, max_tokens=b.T, dhidden_fp32=1)
    H, rstd = ctx.grpo_rmsnorm_fwd(b.x_prenorm, b.gamma, b.eps_rms)
    dgamma = torch.zeros(b.d, dtype=torch.float32, device="cuda")
    dx = ctx.grpo_rmsnorm_bwd(b.x_prenorm, b.gamma, rstd, dH, dgamma)
    dx2 = ctx.grpo_rmsnorm_bwd(b.x_prenorm, b.gamma, rstd, dH, dgamma)      # dgamma accumulates, dx is overwritten
    torch.cuda.synchronize()
    ctx.close()
    assert rel_l2(to64(dx), dx_ref) <= 2e-6 and torch.equal(dx, dx2)
    assert rel_l2(to64(dgamma), 2 * dg_ref) <= 2e-6


def test_full_size_sampled_rows():
    """configs[1] shape (d = 2048, V = 151936, T ~ 18.7k) from pre-norm activations, in the launch configuration
    bench.py --prenorm times: sampled tokens against the oracle (H row, rstd, logp, dx row)."""
    b = make_config(2, seed=0, device="cuda", prenorm=True)
    assert (b.d, b.V) == (2048, 151936)
    out = _run(b)
    rng = np.random.default_rng(7)
    rows = np.unique(np.concatenate([rng.choice(b.T, 32, replace=False), [0, 255, 256, b.T - 1]]))
    r = torch.from_numpy(rows).cuda()
    xs = b.x_prenorm[r].double().cpu().numpy()
    gm = b.gamma.double().cpu().numpy()
    W64 = b.W.double().cpu().numpy()
    y = b.targets.cpu().numpy().astype(np.int64)[rows]
    H_ref, rstd_ref = rmsnorm_fwd(xs, gm, b.eps_rms)
    ulps = _bf16_ulps_apart(out["H"][r], torch.tensor(H_ref, dtype=torch.float32).to(torch.bfloat16).cuda())
    assert ulps.max().item() <= 1 and (ulps != 0).float().mean().item() < 2e-3
    np.testing.assert_allclose(to64(out["rstd"][r]), rstd_ref, rtol=2e-6)
    idx = np.arange(len(rows))
    lse, logp = token_rows(H_ref, W64, y, idx)
    assert np.abs(to64(out["logp"][r]) - logp).max() <= TOL_LOGP_ABS
    adv, _ = group_advantage(b.rewards.double().cpu().numpy(), G=b.G, eps_std=b.eps_std)
    A_tok = token_advantage(adv, b.cu_seqlens.cpu().numpy())[rows]
    lt = loss_terms(logp, b.old_logp.double().cpu().numpy()[rows], None, None, A_tok, np.array([0, len(rows)]),
                    OracleConfig(eps_std=b.eps_std, clip_lo=b.clip_lo, clip_hi=b.clip_hi), loss_denom=float(b.T))
    dH = dH_rows(H_ref, W64, y, lse, lt["coeff"], idx)
    dx_ref, _ = rmsnorm_bwd(xs, gm, rstd_ref, dH)
    dx = to64(out["dx"][r])
    assert rel_l2(dx, dx_ref) <= TOL_GRAD_REL
    assert max(rel_l2(dx[i], dx_ref[i]) for i in range(len(rows))) <= 2 * TOL_GRAD_REL
    assert torch.isfinite(out["dgamma"]).all() and out["dgamma"].abs().max() > 0
