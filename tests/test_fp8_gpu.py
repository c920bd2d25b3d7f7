"""FP8 precision study (R32): grpo_config.fp8_logits = 1 runs the two
logit contractions (A2, A4 recompute) on e4m3 operands (tcgen05 kind::f8f6f4).

Two comparisons, both against the float64 oracle:
  (a) CORRECTNESS of the FP8 path: against the oracle evaluated on the SAME quantised operands
      (oracle.fp8_dequantized_operands: per-row scale amax/448 for H, one scale for W, E4M3 round-to-nearest-even) the
      usual north_star tolerances must hold - products of e4m3 values are exact in the fp32 accumulator.
  (b) the STUDY: against the oracle on the original bf16 operands the log-prob error is the e4m3 rounding of the
      operands; it is reported and bracketed (well above north_star's 2e-3, which is why this is a study and not the
      path), and so is the gradient error it causes through rho and the clip decisions."""
import numpy as np
import pytest
import torch

from oracle.grpo_oracle import OracleConfig, fp8_dequantized_operands, grpo_step
from tests.parity_util import TOL_GRAD_REL, TOL_LOGP_ABS, TOL_LOSS_REL, make_ctx, rel_l2, run_cuda, run_oracle, to64
from workloads.synth import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2606_26997_b200.build import build
    build()


def _oracle_fp8(b, **kw):
    x = b.numpy_f64()
    Hq, Wq = fp8_dequantized_operands(x["H"], x["W"])
    cfg = OracleConfig(eps_std=b.eps_std, clip_lo=b.clip_lo, clip_hi=b.clip_hi, kl_beta=b.kl_beta, loss_agg=b.loss_agg, **kw)
    out = grpo_step(Hq, Wq, x["y"], x["cu_seqlens"], x["rewards"], x["old_logp"], x["ref_logp"], mask=x["mask"], cfg=cfg, G=b.G)
    # the backward contractions A5 / A6 use the ORIGINAL bf16 W and H (only the logits are FP8): dH = dz W, dW = dz^T H
    dH = np.zeros_like(x["H"])
    dW = np.zeros_like(x["W"])
    T = x["H"].shape[0]
    for t0 in range(0, T, 512):
        t1 = min(T, t0 + 512)
        z = cfg.logit_scale * (Hq[t0:t1] @ Wq.T)
        dz = -np.exp(z - out["lse"][t0:t1, None])
        ok = (x["y"][t0:t1] >= 0) & (x["y"][t0:t1] < b.V)
        dz[np.arange(t1 - t0)[ok], x["y"][t0:t1][ok]] += 1.0
        dz *= out["coeff"][t0:t1, None] * cfg.logit_scale
        dH[t0:t1] = dz @ x["W"]
        dW += dz.T @ x["H"][t0:t1]
    out["dH"], out["dW"] = dH, dW
    return out


@pytest.mark.parametrize("kw", [dict(d=64), dict(d=128, V=3000, n_groups=6, G=8, len_div=0.2, mask_frac=0.1),
                                dict(d=256, V=2000, n_groups=3, G=4, len_div=0.3, w_std=0.3)])
def test_fp8_path_matches_the_oracle_on_the_same_quantised_operands(kw):
    b = make_config(1, device="cuda", seed=9, variant="1b", **kw)
    ctx = make_ctx(b, max_tokens=b.T, fp8_logits=1, bwd_chunk_tokens=1024, dhidden_fp32=1)
    out = run_cuda(ctx, b)
    n = ctx.grpo_kernel_launches()
    assert ctx.grpo_check_errors_sync() == 0
    ctx.close()
    assert n["quantize"] > 0
    ref = _oracle_fp8(b)
    assert np.abs(to64(out["logp"]) - ref["logp"]).max() <= TOL_LOGP_ABS
    assert np.abs(to64(out["lse"]) - ref["lse"]).max() <= TOL_LOGP_ABS
    assert abs(out["loss"].item() - ref["loss"]) <= TOL_LOSS_REL * max(abs(ref["loss"]), ref["abs_loss"])
    assert rel_l2(to64(out["coeff"]), ref["coeff"]) <= 1e-3
    assert rel_l2(to64(out["dH"]), ref["dH"]) <= TOL_GRAD_REL
    assert rel_l2(to64(out["dW"]), ref["dW"]) <= TOL_GRAD_REL
    y = b.targets.cpu().numpy()
    non_target = np.ones(b.V, dtype=bool)
    non_target[y[(y >= 0) & (y < b.V)]] = False
    assert rel_l2(to64(out["dW"])[non_target], ref["dW"][non_target]) <= TOL_GRAD_REL      # the dense softmax term alone


def test_precision_study_against_the_bf16_definition():
    b = make_config(1, device="cuda", seed=9, variant="1b", d=256, V=5000, n_groups=6, G=8, len_div=0.2)
    ref = run_oracle(b)
    errs = {}
    for name, flag in (("bf16", 0), ("fp8", 1)):
        ctx = make_ctx(b, max_tokens=b.T, fp8_logits=flag, bwd_chunk_tokens=1024)
        out = run_cuda(ctx, b)
        ctx.close()
        errs[name] = dict(logp=float(np.abs(to64(out["logp"]) - ref["logp"]).max()),
                          dH=rel_l2(to64(out["dH"]), ref["dH"]), dW=rel_l2(to64(out["dW"]), ref["dW"]))
    print("precision study (max |logp err|, dH rel-L2, dW rel-L2):", errs)
    assert errs["bf16"]["logp"] <= 1e-4
    # e4m3 operands carry 2^-4 relative rounding per element: the logits move by ~4e-2, far above north_star's 2e-3;
    # in this off-policy (config-1b) regime that moves rho by ~4 % and flips clip decisions, so the gradients move
    # by ~10 % (measured 0.135): the reason FP8 logits are a study, not the path
    assert 2e-3 < errs["fp8"]["logp"] < 0.5, errs
    assert errs["bf16"]["dH"] <= TOL_GRAD_REL and errs["bf16"]["dW"] <= TOL_GRAD_REL
    assert 1e-2 < errs["fp8"]["dW"] < 0.5 and errs["fp8"]["dH"] < 0.5, errs
