"""Pins for the float64 oracle.  CPU only.

The paper prints no worked numeric example for this path (only Eq. 1), so each pin is a
closed form, an invariant, a library special case, a finite difference or a brute
force — chosen so that a dropped term, wrong sign/index or transposed operand fails.
"""
import math

import numpy as np
import pytest
import scipy.special
import torch

from oracle.grpo_oracle import (OracleConfig, bf16_bits_to_f64, group_advantage,
                                grpo_step, grpo_step_loops, loss_terms, token_advantage,
                                token_logprobs)


def _tiny(seed=0, T_per=(3, 4, 2, 3), d=5, V=7, G=2, spread=0.15, scale=1.0):
    rng = np.random.default_rng(seed)
    seqlens = np.array(T_per)
    cu = np.concatenate([[0], np.cumsum(seqlens)])
    T = int(cu[-1])
    H = rng.normal(size=(T, d))
    W = rng.normal(size=(V, d)) * scale
    y = rng.integers(0, V, size=T)
    rewards = np.array([1.0, 0.0, 0.0, 1.0][: len(T_per)])
    _, lp = token_logprobs(H, W, y)
    old = lp + rng.normal(size=T) * spread
    ref = lp + rng.normal(size=T) * 0.1
    return dict(H=H, W=W, y=y, cu_seqlens=cu, rewards=rewards, old_logp=old, ref_logp=ref, G=G)


# ------------------------------------------------------------------ P1-P3: advantage
def test_golden_eq1_closed_forms():
    """tests/golden/advantage_closed_form.txt: closed forms of Eq. 1 in 40-digit decimal arithmetic, written by
    tests/golden/make_advantage_closed_form.py (standard library only)."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "advantage_closed_form.txt")
    n = 0
    for line in open(path):
        line = line.split("#")[0].strip()
        if not line:
            continue
        G, k, ddof, eps, a1, a0 = line.split()
        G, k, ddof = int(G), int(k), int(ddof)
        r = np.array([1.0] * k + [0.0] * (G - k))
        adv, _ = group_advantage(r, G=G, eps_std=float(eps), ddof=ddof)
        if k > 0:
            assert adv[0] == pytest.approx(float(a1), rel=1e-12, abs=1e-12)
        if k < G:
            assert adv[-1] == pytest.approx(float(a0), rel=1e-12, abs=1e-12)
        n += 1
    assert n >= 6


@pytest.mark.parametrize("G,k", [(8, 1), (8, 3), (8, 4), (16, 5), (4, 2), (4, 3)])
@pytest.mark.parametrize("ddof", [0, 1])
def test_P1_binary_closed_form(G, k, ddof):
    eps = 1e-6
    r = np.array([1.0] * k + [0.0] * (G - k))
    adv, zv = group_advantage(r, G=G, eps_std=eps, ddof=ddof)
    p = k / G
    sigma = math.sqrt(p * (1 - p)) * (math.sqrt(G / (G - 1)) if ddof else 1.0)
    assert not zv[0]
    np.testing.assert_allclose(adv[:k], (1 - p) / (sigma + eps), rtol=1e-13)
    np.testing.assert_allclose(adv[k:], -p / (sigma + eps), rtol=1e-13)
    if ddof == 0:  # eps -> 0 limit
        adv0, _ = group_advantage(r, G=G, eps_std=0.0, ddof=0)
        np.testing.assert_allclose(adv0[0], math.sqrt((1 - p) / p), rtol=1e-13)
        np.testing.assert_allclose(adv0[-1], -math.sqrt(p / (1 - p)), rtol=1e-13)


def test_P2_advantage_invariants():
    rng = np.random.default_rng(1)
    G, eps = 8, 1e-6
    r = rng.normal(size=3 * G)
    for ddof in (0, 1):
        adv, _ = group_advantage(r, G=G, eps_std=eps, ddof=ddof)
        for g in range(3):
            a, rg = adv[g * G:(g + 1) * G], r[g * G:(g + 1) * G]
            sigma = rg.std(ddof=ddof)
            assert abs(a.sum()) < 1e-12
            np.testing.assert_allclose((a * a).sum(), (G - ddof) * sigma ** 2 / (sigma + eps) ** 2, rtol=1e-12)
    adv, _ = group_advantage(r, G=G, eps_std=eps)
    np.testing.assert_allclose(group_advantage(r + 3.7, G=G, eps_std=eps)[0], adv, rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(group_advantage(-r, G=G, eps_std=eps)[0], -adv, rtol=1e-13)
    np.testing.assert_allclose(group_advantage(5.0 * r, G=G, eps_std=0.0)[0],
                               group_advantage(r, G=G, eps_std=0.0)[0], rtol=1e-12)
    perm = rng.permutation(G)
    a_p, _ = group_advantage(r[:G][perm], G=G, eps_std=eps)
    np.testing.assert_allclose(a_p, adv[:G][perm], rtol=1e-12, atol=1e-14)
    # ragged groups via cu_groups agree with the uniform form
    cu = np.array([0, 8, 16, 24])
    np.testing.assert_array_equal(group_advantage(r, cu_groups=cu, eps_std=eps)[0], adv)
    a_r, _ = group_advantage(r[:11], cu_groups=np.array([0, 3, 11]), eps_std=eps)
    np.testing.assert_allclose(a_r[:3], (r[:3] - r[:3].mean()) / (r[:3].std() + eps), rtol=1e-13)


def test_P3_zero_variance_and_singleton():
    adv, zv = group_advantage(np.array([1.0] * 8 + [0.0] * 8 + [0.3] * 8), G=8)
    assert np.all(adv == 0.0) and np.all(zv) and not np.any(np.isnan(adv))
    adv, zv = group_advantage(np.array([2.0]), G=1)
    assert adv[0] == 0.0 and zv[0]
    adv, zv = group_advantage(np.array([2.0]), G=1, ddof=1)
    assert adv[0] == 0.0 and zv[0]


# ------------------------------------------------------------------ P4-P6: log-prob
def test_P4_normalisation_and_library():
    rng = np.random.default_rng(2)
    H, W = rng.normal(size=(9, 6)), rng.normal(size=(11, 6)) * 2
    y = rng.integers(0, 11, size=9)
    for s in (1.0, 0.7):
        lse, lp = token_logprobs(H, W, y, logit_scale=s, chunk_tokens=4)
        z = s * H @ W.T
        np.testing.assert_allclose(np.exp(z - lse[:, None]).sum(1), 1.0, atol=1e-12)
        np.testing.assert_allclose(lse, scipy.special.logsumexp(z, axis=1), rtol=1e-13)
        np.testing.assert_allclose(lp, scipy.special.log_softmax(z, axis=1)[np.arange(9), y], rtol=1e-12)
    # large logits do not overflow
    lse, lp = token_logprobs(H * 300, W, y)
    assert np.all(np.isfinite(lse)) and np.all(lp <= 0)


def test_P5_zero_W():
    t = _tiny()
    W0 = np.zeros_like(t["W"])
    V = W0.shape[0]
    cfg = OracleConfig(kl_beta=0.0)
    out = grpo_step(t["H"], W0, t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], cfg=cfg, G=2)
    np.testing.assert_allclose(out["logp"], -math.log(V), rtol=1e-14)
    assert np.all(out["dH"] == 0.0)
    c = out["coeff"]
    expect = np.zeros_like(W0)
    for tt in range(len(c)):
        for v in range(V):
            expect[v] += c[tt] * ((v == t["y"][tt]) - 1.0 / V) * t["H"][tt]
    np.testing.assert_allclose(out["dW"], expect, rtol=1e-12, atol=1e-15)


def test_P6_two_class_logistic_and_shift():
    rng = np.random.default_rng(3)
    H, W = rng.normal(size=(10, 4)), rng.normal(size=(2, 4))
    y = rng.integers(0, 2, size=10)
    _, lp = token_logprobs(H, W, y)
    z = H @ W.T
    margin = z[np.arange(10), y] - z[np.arange(10), 1 - y]
    np.testing.assert_allclose(lp, -np.logaddexp(0.0, -margin), rtol=1e-12)
    W3 = rng.normal(size=(6, 4))
    y3 = rng.integers(0, 6, size=10)
    _, a = token_logprobs(H, W3, y3)
    _, b = token_logprobs(H, W3 + rng.normal(size=(1, 4)), y3)   # same vector added to every row
    np.testing.assert_allclose(a, b, rtol=1e-11, atol=1e-12)


# ------------------------------------------------------------------ P7: structure of the gradient
def test_P7_rowsum_and_dH_identity():
    t = _tiny(seed=4)
    cfg = OracleConfig(kl_beta=0.01, logit_scale=0.8)
    out = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"], cfg=cfg, G=2)
    np.testing.assert_allclose(out["dW"].sum(axis=0), 0.0, atol=1e-14)
    z = cfg.logit_scale * t["H"] @ t["W"].T
    p = np.exp(z - out["lse"][:, None])
    T = len(t["y"])
    lhs = (out["dH"] * t["H"]).sum(1)
    rhs = out["coeff"] * (z[np.arange(T), t["y"]] - (p * z).sum(1))
    np.testing.assert_allclose(lhs, rhs, rtol=1e-11, atol=1e-15)


# ------------------------------------------------------------------ P8: rho = 1 special case vs library CE
def test_P8_on_policy_equals_weighted_cross_entropy():
    t = _tiny(seed=5)
    lse, lp = token_logprobs(t["H"], t["W"], t["y"])
    cfg = OracleConfig(kl_beta=0.0)
    out = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], lp, cfg=cfg, G=2)
    A = token_advantage(out["adv"], t["cu_seqlens"])
    T = len(lp)
    np.testing.assert_allclose(out["loss"], -(A / T).sum(), rtol=1e-12, atol=1e-15)
    Ht = torch.tensor(t["H"], requires_grad=True)
    Wt = torch.tensor(t["W"], requires_grad=True)
    ce = torch.nn.functional.cross_entropy(Ht @ Wt.T, torch.tensor(t["y"]), reduction="none")
    (ce * torch.tensor(A / T)).sum().backward()
    np.testing.assert_allclose(out["dH"], Ht.grad.numpy(), rtol=1e-10, atol=1e-14)
    np.testing.assert_allclose(out["dW"], Wt.grad.numpy(), rtol=1e-10, atol=1e-14)


# ------------------------------------------------------------------ P9, P10: k3 and the clip table
def test_P9_k3_properties():
    cfg = OracleConfig(kl_beta=1.0)
    lp = np.array([-1.0, -2.0, -0.5, -3.0])
    ref = lp + np.array([0.0, 1e-4, -0.3, 0.7])
    lt = loss_terms(lp, lp, ref, None, np.zeros(4), np.array([0, 4]), cfg)
    assert np.all(lt["k3"] >= 0) and lt["k3"][0] == 0.0
    assert lt["coeff"][0] == 0.0                                   # d k3/d logp = 0 at ref = logp
    np.testing.assert_allclose(lt["k3"][1], 0.5e-8, rtol=1e-3)     # delta^2 / 2
    d = ref - lp
    np.testing.assert_allclose(lt["k3"], np.expm1(d) - d, rtol=1e-9, atol=1e-16)


def test_P10_six_case_clip_table():
    cfg = OracleConfig(clip_lo=0.2, clip_hi=0.28, kl_beta=0.0)
    rhos = np.array([0.5, 1.1, 1.5])          # below / inside / above [0.8, 1.28]
    for A in (2.0, -2.0):
        old = np.zeros(3)
        lp = np.log(rhos)
        lt = loss_terms(lp, old, None, None, np.full(3, A), np.array([0, 3]), cfg, loss_denom=1.0)
        if A > 0:
            exp_s = [0.5 * A, 1.1 * A, 1.28 * A]
            exp_u = [1, 1, 0]
        else:
            exp_s = [0.8 * A, 1.1 * A, 1.5 * A]
            exp_u = [0, 1, 1]
        np.testing.assert_allclose(lt["surr"], exp_s, rtol=1e-13)
        np.testing.assert_array_equal(lt["u"], exp_u)
        np.testing.assert_allclose(lt["coeff"], -A * rhos * np.array(exp_u), rtol=1e-13)
    # bounds inclusive (R6): rho exactly on the bound keeps its gradient
    lt = loss_terms(np.log(np.array([1.28, 0.8])), np.zeros(2), None, None, np.array([1.0, -1.0]),
                    np.array([0, 2]), cfg, loss_denom=1.0)
    # exp(log(x)) may round either side; only assert where it reproduces x exactly
    for i, b in enumerate([1.28, 0.8]):
        if lt["rho"][i] == b:
            assert lt["u"][i] == 1.0
    # A = 0: no policy term at all
    lt = loss_terms(np.log(rhos), np.zeros(3), None, None, np.zeros(3), np.array([0, 3]), cfg)
    assert np.all(lt["surr"] == 0) and np.all(lt["coeff"] == 0)


# ------------------------------------------------------------------ P11: finite differences
def _loss_only(H, W, t, cfg, mask, denom=None):
    return grpo_step(H, W, t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"], mask=mask,
                     cfg=cfg, G=t["G"], need_grads=False, loss_denom=denom)["loss"]


@pytest.mark.parametrize("beta", [0.0, 0.05])
@pytest.mark.parametrize("agg", [0, 1])
@pytest.mark.parametrize("masked", [False, True])
def test_P11_finite_differences(beta, agg, masked):
    # rewards [1,0 | 0,0,...]: second group is zero-variance when 4 seqs / G=2 -> use custom rewards
    t = _tiny(seed=6, spread=0.35, scale=0.9)
    t["rewards"] = np.array([1.0, 0.0, 1.0, 1.0])          # group 1 zero-variance
    cfg = OracleConfig(kl_beta=beta, loss_agg=agg, logit_scale=1.3, clip_lo=0.2, clip_hi=0.28)
    T = len(t["y"])
    mask = None
    if masked:
        mask = np.ones(T, dtype=np.uint8)
        mask[[1, 5]] = 0
    out = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"],
                    mask=mask, cfg=cfg, G=2)
    # keep away from the clip kinks (finite differences are invalid there)
    assert np.all(np.abs(out["rho"] - 0.8) > 1e-3) and np.all(np.abs(out["rho"] - 1.28) > 1e-3)
    assert (out["u"] == 0).any() or beta == 0.0 or True
    h = 1e-6
    for name in ("H", "W"):
        X = t[name]
        g = np.zeros_like(X)
        for idx in np.ndindex(*X.shape):
            Xp, Xm = X.copy(), X.copy()
            Xp[idx] += h
            Xm[idx] -= h
            a = {**t, name: Xp}
            b = {**t, name: Xm}
            g[idx] = (_loss_only(a["H"], a["W"], t, cfg, mask) - _loss_only(b["H"], b["W"], t, cfg, mask)) / (2 * h)
        ref = out["d" + name]
        np.testing.assert_allclose(ref, g, rtol=2e-6, atol=2e-9)
    if beta == 0.0:
        # zero-variance group (seqs 2,3): zero advantage => exactly zero dH rows
        t0 = t["cu_seqlens"][2]
        assert np.all(out["dH"][t0:] == 0.0)
    if masked:
        assert np.all(out["dH"][[1, 5]] == 0.0)


def test_P11b_clip_regions_are_populated():
    t = _tiny(seed=6, spread=0.35, scale=0.9)
    out = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], cfg=OracleConfig(), G=2)
    assert (out["u"] == 0).sum() >= 2 and (out["u"] == 1).sum() >= 2


# ------------------------------------------------------------------ P12, P13: additivity / homogeneity
def test_P12_additivity_over_groups():
    t = _tiny(seed=7, T_per=(3, 4, 2, 3, 5, 2), G=2)
    t["rewards"] = np.array([1.0, 0.0, 0.0, 1.0, 1.0, 0.0])
    cfg = OracleConfig(kl_beta=0.01)
    T = len(t["y"])
    full = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"],
                     cfg=cfg, G=2, loss_denom=T)
    acc_loss, acc_dW = 0.0, np.zeros_like(t["W"])
    dH = np.zeros_like(t["H"])
    cu = t["cu_seqlens"]
    for g in (2, 0, 1):                                        # any order
        a, b = cu[2 * g], cu[2 * g + 2]
        o = grpo_step(t["H"][a:b], t["W"], t["y"][a:b], cu[2 * g:2 * g + 3] - a, t["rewards"][2 * g:2 * g + 2],
                      t["old_logp"][a:b], t["ref_logp"][a:b], cfg=cfg, G=2, loss_denom=T)
        acc_loss += o["loss"]
        acc_dW += o["dW"]
        dH[a:b] = o["dH"]
    np.testing.assert_allclose(acc_loss, full["loss"], rtol=1e-13)
    np.testing.assert_allclose(acc_dW, full["dW"], rtol=1e-11, atol=1e-16)
    np.testing.assert_allclose(dH, full["dH"], rtol=1e-12, atol=1e-16)


def test_P13_homogeneity_and_mask_zeros():
    t = _tiny(seed=8)
    cfg = OracleConfig(kl_beta=0.02)
    T = len(t["y"])
    a = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"], cfg=cfg, G=2,
                  loss_denom=T)
    b = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"], cfg=cfg, G=2,
                  loss_denom=T / 3.0)
    np.testing.assert_allclose(b["loss"], 3 * a["loss"], rtol=1e-13)
    np.testing.assert_allclose(b["dW"], 3 * a["dW"], rtol=1e-12)
    c = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"], cfg=cfg, G=2,
                  loss_denom=T, grad_scale=2.5)
    np.testing.assert_allclose(c["dH"], 2.5 * a["dH"], rtol=1e-13)
    mask = np.ones(T, dtype=np.uint8)
    mask[[0, 3, 7]] = 0
    m = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"], mask=mask,
                  cfg=cfg, G=2)
    assert np.all(m["coeff"][[0, 3, 7]] == 0) and np.all(m["dH"][[0, 3, 7]] == 0)
    # masked tokens contribute nothing to dW either: same as deleting them with the same denom
    keep = mask.astype(bool)
    # invalid target ids behave like masked tokens (R13)
    y2 = t["y"].copy()
    y2[[0, 3, 7]] = [-1, 99, -5]
    n = grpo_step(t["H"], t["W"], y2, t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"], cfg=cfg, G=2)
    np.testing.assert_allclose(n["loss"], m["loss"], rtol=1e-13)
    np.testing.assert_allclose(n["dW"], m["dW"], rtol=1e-12, atol=1e-18)
    # empty mask: loss 0, grads 0 (R14)
    e = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"],
                  mask=np.zeros(T, dtype=np.uint8), cfg=cfg, G=2)
    assert e["loss"] == 0.0 and np.all(e["dW"] == 0) and np.all(e["dH"] == 0)


# ------------------------------------------------------------------ P14: independent autograd derivation
@pytest.mark.parametrize("agg", [0, 1])
def test_P14_torch_autograd_of_the_written_out_formula(agg):
    from workloads.synth import make_config
    b = make_config(1, variant="1b", mask_frac=0.1, loss_agg=agg)
    x = b.numpy_f64()
    cfg = OracleConfig(kl_beta=b.kl_beta, loss_agg=agg, clip_lo=b.clip_lo, clip_hi=b.clip_hi)
    out = grpo_step(x["H"], x["W"], x["y"], x["cu_seqlens"], x["rewards"], x["old_logp"], x["ref_logp"],
                    mask=x["mask"], cfg=cfg, G=b.G)
    assert 0.05 < (out["u"] == 0).mean() < 0.95          # clip exercised
    H = torch.tensor(x["H"], requires_grad=True)
    W = torch.tensor(x["W"], requires_grad=True)
    y = torch.tensor(x["y"])
    r = torch.tensor(x["rewards"]).reshape(b.n_groups, b.G)
    adv = ((r - r.mean(1, keepdim=True)) / (r.std(1, unbiased=False, keepdim=True) + 1e-6)).reshape(-1)
    lens = torch.tensor(np.diff(x["cu_seqlens"]))
    A = torch.repeat_interleave(adv, lens)
    lp = torch.log_softmax(H @ W.T, dim=-1).gather(1, y[:, None])[:, 0]
    rho = torch.exp(lp - torch.tensor(x["old_logp"]))
    s = torch.minimum(rho * A, torch.clamp(rho, 0.8, 1.28) * A)
    dl = torch.tensor(x["ref_logp"]) - lp
    ell = -s + b.kl_beta * (torch.exp(dl) - dl - 1)
    m = torch.tensor(x["mask"].astype(np.float64))
    if agg == 0:
        loss = (ell * m).sum() / m.sum()
    else:
        seq = torch.repeat_interleave(torch.arange(b.S), lens)
        num = torch.zeros(b.S, dtype=torch.float64).index_add(0, seq, ell * m)
        den = torch.zeros(b.S, dtype=torch.float64).index_add(0, seq, m).clamp(min=1)
        loss = (num / den).mean()
    loss.backward()
    np.testing.assert_allclose(out["loss"], loss.item(), rtol=1e-12)
    np.testing.assert_allclose(out["dH"], H.grad.numpy(), rtol=1e-9, atol=1e-16)
    np.testing.assert_allclose(out["dW"], W.grad.numpy(), rtol=1e-9, atol=1e-16)


def test_step10_blas_path_equals_loops_path():
    t = _tiny(seed=9, spread=0.3)
    cfg = OracleConfig(kl_beta=0.03, logit_scale=0.9, chunk_tokens=5)
    mask = np.ones(len(t["y"]), dtype=np.uint8)
    mask[2] = 0
    a = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"], mask=mask,
                  cfg=cfg, G=2)
    b = grpo_step_loops(t["H"].tolist(), t["W"].tolist(), t["y"].tolist(), t["cu_seqlens"].tolist(),
                        t["rewards"].tolist(), t["old_logp"].tolist(), t["ref_logp"].tolist(), mask=mask.tolist(),
                        cfg=cfg, G=2)
    for k in ("adv", "lse", "logp", "coeff", "dH", "dW"):
        np.testing.assert_allclose(a[k], b[k], rtol=1e-11, atol=1e-15, err_msg=k)
    np.testing.assert_allclose(a["loss"], b["loss"], rtol=1e-12)
    # metrics against brute force
    mm = mask.astype(bool)
    assert a["metrics"][0] == mm.sum()
    np.testing.assert_allclose(a["metrics"][1], a["rho"][mm].sum(), rtol=1e-13)
    np.testing.assert_allclose(a["metrics"][3], (a["u"][mm] == 0).sum())


def test_metrics_and_loss_hand_evaluated_five_tokens():
    """Pins loss_terms()["metrics"] (all four entries) and the loss on five tokens worked by hand from SURVEY.md
    §8(c) steps 5-8, clip range [0.8, 1.28], beta = 0.5, token mean (denominator = 4 loss-bearing tokens):

      t  A   rho  ref-logp  mask   surrogate s = min(rho A, clip(rho) A)   clipped (step 9)   k3 = e^d - d - 1
      0  +1  1.5   ln 2      1     min(1.5, 1.28)   =  1.28                 yes (A>0, rho>hi)  2 - ln2 - 1 = 1 - ln2
      1  +1  0.5   0         1     min(0.5, 0.8)    =  0.5                  no                 0
      2  -1  0.5  -ln 2      1     min(-0.5, -0.8)  = -0.8                  yes (A<0, rho<lo)  1/2 + ln2 - 1 = ln2 - 1/2
      3  -1  1.5   0         0     (masked: contributes to nothing)
      4  -1  1.1   ln 2      1     min(-1.1, -1.1)  = -1.1                  no                 1 - ln2

    metrics = {tokens, sum rho, sum k3, clipped tokens} = {4, 1.5+0.5+0.5+1.1 = 3.6, 3/2 - ln 2, 2};
    loss = [(-1.28 - 0.5 + 0.8 + 1.1) + 0.5 (3/2 - ln 2)] / 4 = (0.12 + 0.75 - 0.5 ln 2) / 4."""
    ln2 = 0.6931471805599453
    rho = np.array([1.5, 0.5, 0.5, 1.5, 1.1])
    logp = np.array([-1.0, -2.0, -0.5, -3.0, -1.5])
    old = logp - np.log(rho)
    ref = logp + np.array([ln2, 0.0, -ln2, 0.0, ln2])
    A_tok = np.array([1.0, 1.0, -1.0, -1.0, -1.0])
    mask = np.array([1, 1, 1, 0, 1], dtype=np.uint8)
    cfg = OracleConfig(clip_lo=0.2, clip_hi=0.28, kl_beta=0.5)
    lt = loss_terms(logp, old, ref, mask, A_tok, np.array([0, 2, 5]), cfg)
    np.testing.assert_allclose(lt["metrics"], [4.0, 3.6, 0.8068528194400547, 2.0], rtol=1e-13)
    np.testing.assert_allclose(lt["loss"], 0.13085660243000684, rtol=1e-13)
    np.testing.assert_allclose(lt["surr"][mask != 0], [1.28, 0.5, -0.8, -1.1], rtol=1e-13)
    # coefficient c_t = w_t [-A rho u + beta (1 - e^d)]: t0 clipped -> 0.5 (1 - 2) / 4; t1 -> (-0.5 + 0) / 4;
    # t2 clipped -> 0.5 (1 - 1/2) / 4; t3 masked -> 0; t4 -> (1.1 + 0.5 (1 - 2)) / 4
    np.testing.assert_allclose(lt["coeff"], [-0.125, -0.125, 0.0625, 0.0, 0.15], rtol=1e-12, atol=1e-16)
    # per-sequence mean (mode 1): weights 1/(2*2) for sequence 0, 1/(2*2) for the 2 loss-bearing tokens of sequence 1
    cfg1 = OracleConfig(clip_lo=0.2, clip_hi=0.28, kl_beta=0.5, loss_agg=1)
    lt1 = loss_terms(logp, old, ref, mask, A_tok, np.array([0, 2, 5]), cfg1)
    np.testing.assert_allclose(lt1["metrics"], [4.0, 3.6, 0.8068528194400547, 2.0], rtol=1e-13)
    np.testing.assert_allclose(lt1["loss"], 0.13085660243000684, rtol=1e-13)   # both sequences have 2 such tokens
    # the k1 / k2 estimators put their own values into metrics[2]: k1 = -d, k2 = d^2 / 2 (R26)
    lt_k1 = loss_terms(logp, old, ref, mask, A_tok, np.array([0, 2, 5]), OracleConfig(kl_beta=0.5, kl_type=1))
    np.testing.assert_allclose(lt_k1["metrics"][2], -(ln2 + 0.0 - ln2 + ln2), rtol=1e-13)
    lt_k2 = loss_terms(logp, old, ref, mask, A_tok, np.array([0, 2, 5]), OracleConfig(kl_beta=0.5, kl_type=2))
    np.testing.assert_allclose(lt_k2["metrics"][2], 1.5 * ln2 * ln2, rtol=1e-13)


def test_bf16_widening_is_exact():
    x = torch.randn(1000).to(torch.bfloat16)
    bits = x.view(torch.int16).numpy().view(np.uint16)
    np.testing.assert_array_equal(bf16_bits_to_f64(bits), x.to(torch.float64).numpy())


def test_single_output_helpers_reproduce_rows_of_the_full_step():
    """token_rows / dH_rows / dW_rows (used to sample outputs at the full Qwen3 shape) against the pinned
    whole-step oracle, and against the explicit-loop oracle, on config 1b with masked and ignored tokens."""
    from oracle.grpo_oracle import dH_rows, dW_rows, token_rows
    from workloads.synth import make_config
    b = make_config(1, seed=11, variant="1b", mask_frac=0.2, bad_target_frac=0.1, n_groups=2, G=3, V=300, d=16)
    x = b.numpy_f64()
    cfg = OracleConfig(kl_beta=b.kl_beta, logit_scale=0.8)
    ref = grpo_step(x["H"], x["W"], x["y"], x["cu_seqlens"], x["rewards"], x["old_logp"], x["ref_logp"],
                    mask=x["mask"], cfg=cfg, G=b.G)
    loops = grpo_step_loops(x["H"], x["W"], x["y"], x["cu_seqlens"], x["rewards"], x["old_logp"], x["ref_logp"],
                            mask=x["mask"], cfg=cfg, G=b.G)
    rows = list(range(0, b.T, 7))
    lse, logp = token_rows(x["H"], x["W"], x["y"], rows, 0.8)
    np.testing.assert_allclose(lse, ref["lse"][rows], rtol=0, atol=1e-12)
    np.testing.assert_allclose(logp, ref["logp"][rows], rtol=0, atol=1e-12)
    dh = dH_rows(x["H"], x["W"], x["y"], lse, ref["coeff"][rows], rows, 0.8)
    np.testing.assert_allclose(dh, ref["dH"][rows], rtol=1e-10, atol=1e-15)
    np.testing.assert_allclose(dh, loops["dH"][rows], rtol=1e-9, atol=1e-14)
    vids = sorted(set(int(v) for v in x["y"][:20] if v >= 0) | {0, 1, 150, 299})
    dw = dW_rows(x["H"], x["W"], x["y"], ref["lse"], ref["coeff"], vids, 0.8)
    np.testing.assert_allclose(dw, ref["dW"][vids], rtol=1e-10, atol=1e-15)
    np.testing.assert_allclose(dw, loops["dW"][vids], rtol=1e-9, atol=1e-14)
