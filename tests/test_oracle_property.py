"""Property pin of the float64 oracle (CPU only): on RANDOM small problems and RANDOM settings of every switch the
oracle's loss and gradients equal float64 torch autograd of the objective written out below from SURVEY.md §8(c)
steps 1-9 / DESIGN.md R1-R28 with stock torch ops (log_softmax, clamp, minimum, maximum) — an independent second
derivation: the oracle codes the backward by hand (`c_t`, `dz = c_t (1[v=y] - p)`), autograd differentiates the
forward.  Complements P14 (one fixed configuration) by sweeping shapes, masks, invalid targets, zero-variance
groups, both aggregations, the three KL estimators, dual clip, temperature, explicit denominators and grad_scale.
"""
import numpy as np
import torch
from hypothesis import given, settings, strategies as st

from oracle.grpo_oracle import OracleConfig, grpo_step


@st.composite
def problems(draw):
    seed = draw(st.integers(0, 2**31 - 1))
    n_groups = draw(st.integers(1, 3))
    G = draw(st.integers(2, 4))
    d = draw(st.integers(1, 6))
    V = draw(st.integers(2, 9))
    cfg = dict(std_ddof=draw(st.sampled_from([0, 1])), clip_lo=draw(st.sampled_from([0.1, 0.2, 0.35])),
               clip_hi=draw(st.sampled_from([0.1, 0.28, 0.5])), kl_beta=draw(st.sampled_from([0.0, 0.01, 0.3])),
               loss_agg=draw(st.sampled_from([0, 1])), logit_scale=draw(st.sampled_from([1.0, 0.6, 1.7])),
               kl_type=draw(st.sampled_from([0, 1, 2])), dual_clip=draw(st.sampled_from([0.0, 1.5, 3.0])))
    extra = dict(mask_p=draw(st.sampled_from([0.0, 0.3])), bad_p=draw(st.sampled_from([0.0, 0.2])),
                 explicit_denom=draw(st.booleans()), grad_scale=draw(st.sampled_from([1.0, 0.25])),
                 flat_group=draw(st.booleans()), spread=draw(st.sampled_from([0.05, 0.4, 1.2])))
    return seed, n_groups, G, d, V, cfg, extra


@settings(max_examples=120, deadline=None)
@given(problems())
def test_P15_oracle_equals_autograd_on_random_problems(p):
    seed, n_groups, G, d, V, ckw, ex = p
    rng = np.random.default_rng(seed)
    S = n_groups * G
    lens = rng.integers(1, 6, size=S)
    cu = np.concatenate([[0], np.cumsum(lens)])
    T = int(cu[-1])
    H = rng.normal(size=(T, d))
    W = rng.normal(size=(V, d))
    y = rng.integers(0, V, size=T)
    bad = rng.random(T) < ex["bad_p"]
    y_in = np.where(bad, np.where(rng.random(T) < 0.5, -1 - rng.integers(0, 3, size=T), V + rng.integers(0, 3, size=T)), y)
    rewards = rng.integers(0, 2, size=S).astype(np.float64)
    if ex["flat_group"]:
        rewards[:G] = 1.0                                             # a zero-variance group (R4)
    mask = (rng.random(T) >= ex["mask_p"]).astype(np.uint8)
    s_ = ckw["logit_scale"]
    base = torch.log_softmax(torch.tensor(H @ W.T * s_), dim=-1).numpy()[np.arange(T), y]
    old = base + rng.normal(size=T) * ex["spread"]
    ref = base + rng.normal(size=T) * 0.3
    denom = float(T) * 1.5 if ex["explicit_denom"] and ckw["loss_agg"] == 0 else None
    cfg = OracleConfig(**ckw)
    out = grpo_step(H, W, y_in, cu, rewards, old, ref, mask=mask, cfg=cfg, G=G, loss_denom=denom,
                    grad_scale=ex["grad_scale"])

    # ---- the objective, written out with stock torch ops
    Ht = torch.tensor(H, requires_grad=True)
    Wt = torch.tensor(W, requires_grad=True)
    r = torch.tensor(rewards).reshape(n_groups, G)
    sig = r.std(1, unbiased=bool(ckw["std_ddof"]), keepdim=True)
    adv = torch.where(sig > 0, (r - r.mean(1, keepdim=True)) / (sig + cfg.eps_std), torch.zeros_like(r)).reshape(-1)
    A = torch.repeat_interleave(adv, torch.tensor(lens))
    valid = (y_in >= 0) & (y_in < V)
    m = torch.tensor((valid & (mask != 0)).astype(np.float64))
    lp = torch.log_softmax(s_ * (Ht @ Wt.T), dim=-1).gather(1, torch.tensor(np.where(valid, y_in, 0))[:, None])[:, 0]
    rho = torch.exp(lp - torch.tensor(old))
    surr = torch.minimum(rho * A, torch.clamp(rho, 1 - cfg.clip_lo, 1 + cfg.clip_hi) * A)
    if cfg.dual_clip > 0:
        surr = torch.where(A < 0, torch.maximum(surr, cfg.dual_clip * A), surr)
    dl = torch.tensor(ref) - lp
    kl = [torch.exp(dl) - dl - 1, -dl, 0.5 * dl * dl][cfg.kl_type]
    ell = -surr + cfg.kl_beta * kl
    if cfg.loss_agg == 0:
        loss = (ell * m).sum() / (denom if denom else max(float(m.sum()), 1.0))
    else:
        seq = torch.repeat_interleave(torch.arange(S), torch.tensor(lens))
        num = torch.zeros(S, dtype=torch.float64).index_add(0, seq, ell * m)
        den = torch.zeros(S, dtype=torch.float64).index_add(0, seq, m).clamp(min=1)
        loss = (num / den).sum() / S
    (loss * ex["grad_scale"]).backward()
    scale = max(abs(loss.item()), 1e-30)
    assert abs(out["loss"] - loss.item()) <= 1e-11 * max(scale, float(out["abs_loss"]))
    np.testing.assert_allclose(out["logp"][valid], lp.detach().numpy()[valid], rtol=0, atol=1e-11)
    g = max(float(Ht.grad.abs().max()), float(Wt.grad.abs().max()), 1e-30)
    np.testing.assert_allclose(out["dH"], Ht.grad.numpy(), rtol=1e-9, atol=1e-11 * g)
    np.testing.assert_allclose(out["dW"], Wt.grad.numpy(), rtol=1e-9, atol=1e-11 * g)
