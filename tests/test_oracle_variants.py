"""NEXT-2: pins of the loss variants added to the oracle — k1 / k2 KL estimators and the
dual clip (R26, R27).  The paper prints nothing about them (it names only the "clipped surrogate",
PAPER.md:38), so each pin is a mathematical property, a hand-evaluated table, a finite difference or an
independent torch-autograd derivation.  CPU only."""
import numpy as np
import pytest
import torch

from oracle.grpo_oracle import OracleConfig, grpo_step, grpo_step_loops, loss_terms
from tests.test_oracle_pins import _tiny, _loss_only


def _kl_terms(kl_type, logp, ref):
    cfg = OracleConfig(kl_beta=1.0, kl_type=kl_type)
    T = len(logp)
    lt = loss_terms(logp, logp.copy(), ref, None, np.zeros(T), np.array([0, T]), cfg, loss_denom=1.0)
    return lt["k3"], lt["coeff"]          # A = 0, rho = 1, w = 1: coeff = beta * d k / d logp


def test_k1_and_k3_are_unbiased_for_the_kl_divergence_and_k2_is_its_second_order_term():
    """With samples v ~ pi and r = pi_ref(v) / pi(v): E[k1] = E[k3] = KL(pi || pi_ref) exactly (E[r] = 1);
    k2 = (log r)^2 / 2 agrees with k3 to third order in log r."""
    rng = np.random.default_rng(0)
    V = 11
    p = rng.dirichlet(np.ones(V))
    q = rng.dirichlet(np.ones(V))
    kl = float(np.sum(p * (np.log(p) - np.log(q))))
    k1, _ = _kl_terms(1, np.log(p), np.log(q))
    k3, _ = _kl_terms(0, np.log(p), np.log(q))
    assert np.sum(p * k1) == pytest.approx(kl, rel=1e-12)
    assert np.sum(p * k3) == pytest.approx(kl, rel=1e-12)
    assert np.all(k3 >= 0)
    k2, _ = _kl_terms(2, np.log(p), np.log(q))
    assert np.all(k2 >= 0)
    # small perturbation: k2 - k3 = O(delta^3)
    lp = np.log(p)
    ref = lp + 1e-3 * rng.normal(size=V)
    k2s, _ = _kl_terms(2, lp, ref)
    k3s, _ = _kl_terms(0, lp, ref)
    assert np.max(np.abs(k2s - k3s)) < 1e-8 and np.max(k2s) > 1e-8


@pytest.mark.parametrize("kl_type", [0, 1, 2])
def test_kl_coefficient_is_the_derivative_of_the_kl_term(kl_type):
    rng = np.random.default_rng(1)
    lp = -rng.uniform(0.5, 4.0, size=9)
    ref = lp + rng.normal(size=9) * 0.3
    _, c = _kl_terms(kl_type, lp, ref)
    h = 1e-6
    kp, _ = _kl_terms(kl_type, lp + h, ref)
    km, _ = _kl_terms(kl_type, lp - h, ref)
    # old_logp moves with logp in _kl_terms (rho stays 1, A = 0), so only the KL term varies
    np.testing.assert_allclose(c, (kp - km) / (2 * h), rtol=1e-7, atol=1e-9)
    if kl_type == 1:
        assert np.all(c == 1.0)           # d(logp - ref)/d logp
    if kl_type == 2:
        np.testing.assert_allclose(c, lp - ref, rtol=1e-14)


def test_dual_clip_table_by_hand():
    """eps_lo = 0.2, eps_hi = 0.28, c = 3.  A < 0: s = max(min(rho A, clip(rho) A), c A).
    rho = 0.5 -> 0.8 A (lower clip, u = 0); 1.1 -> 1.1 A (u = 1); 2.0 -> 2 A (u = 1: min picks rho A);
    4.0 -> 3 A (dual clip, u = 0).  A > 0 is untouched by the dual clip."""
    cfg = OracleConfig(clip_lo=0.2, clip_hi=0.28, dual_clip=3.0)
    rhos = np.array([0.5, 1.1, 2.0, 4.0])
    A = -1.5
    lt = loss_terms(np.log(rhos), np.zeros(4), None, None, np.full(4, A), np.array([0, 4]), cfg, loss_denom=1.0)
    np.testing.assert_allclose(lt["surr"], [0.8 * A, 1.1 * A, 2.0 * A, 3.0 * A], rtol=1e-13)
    np.testing.assert_array_equal(lt["u"], [0, 1, 1, 0])
    np.testing.assert_allclose(lt["coeff"], -A * rhos * np.array([0, 1, 1, 0]), rtol=1e-13)
    A = 1.5
    base = loss_terms(np.log(rhos), np.zeros(4), None, None, np.full(4, A), np.array([0, 4]),
                      OracleConfig(clip_lo=0.2, clip_hi=0.28), loss_denom=1.0)
    lt = loss_terms(np.log(rhos), np.zeros(4), None, None, np.full(4, A), np.array([0, 4]), cfg, loss_denom=1.0)
    np.testing.assert_array_equal(lt["surr"], base["surr"])
    np.testing.assert_array_equal(lt["coeff"], base["coeff"])
    # dual clip off: rho = 4, A < 0 keeps its (large) gradient
    off = loss_terms(np.log(rhos), np.zeros(4), None, None, np.full(4, -1.5), np.array([0, 4]),
                     OracleConfig(clip_lo=0.2, clip_hi=0.28), loss_denom=1.0)
    assert off["u"][3] == 1.0 and off["surr"][3] == pytest.approx(-6.0)


@pytest.mark.parametrize("kl_type,dual", [(1, 0.0), (2, 0.0), (0, 1.6), (2, 1.6)])
def test_finite_differences_of_the_variants(kl_type, dual):
    t = _tiny(seed=6, spread=0.45, scale=0.9)
    t["rewards"] = np.array([1.0, 0.0, 0.0, 1.0])
    cfg = OracleConfig(kl_beta=0.07, kl_type=kl_type, dual_clip=dual, logit_scale=1.2)
    out = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"], cfg=cfg, G=2)
    for b in (0.8, 1.28) + ((dual,) if dual else ()):
        assert np.all(np.abs(out["rho"] - b) > 1e-3)
    if dual:
        A_tok = np.repeat(out["adv"], np.diff(t["cu_seqlens"]))
        assert ((A_tok < 0) & (out["rho"] > dual)).any()       # the dual clip is active somewhere
    h = 1e-6
    for name in ("H", "W"):
        X = t[name]
        g = np.zeros_like(X)
        for idx in np.ndindex(*X.shape):
            Xp, Xm = X.copy(), X.copy()
            Xp[idx] += h
            Xm[idx] -= h
            a, b = {**t, name: Xp}, {**t, name: Xm}
            g[idx] = (_loss_only(a["H"], a["W"], t, cfg, None) - _loss_only(b["H"], b["W"], t, cfg, None)) / (2 * h)
        np.testing.assert_allclose(out["d" + name], g, rtol=3e-6, atol=3e-9)


@pytest.mark.parametrize("kl_type,dual", [(1, 0.0), (2, 2.0), (0, 2.0)])
def test_torch_autograd_of_the_written_out_variants(kl_type, dual):
    from workloads.synth import make_config
    b = make_config(1, variant="1b", old_sigma=0.6)
    x = b.numpy_f64()
    cfg = OracleConfig(kl_beta=0.05, kl_type=kl_type, dual_clip=dual, clip_lo=b.clip_lo, clip_hi=b.clip_hi)
    out = grpo_step(x["H"], x["W"], x["y"], x["cu_seqlens"], x["rewards"], x["old_logp"], x["ref_logp"], cfg=cfg,
                    G=b.G)
    H = torch.tensor(x["H"], requires_grad=True)
    W = torch.tensor(x["W"], requires_grad=True)
    y = torch.tensor(x["y"])
    r = torch.tensor(x["rewards"]).reshape(b.n_groups, b.G)
    adv = ((r - r.mean(1, keepdim=True)) / (r.std(1, unbiased=False, keepdim=True) + 1e-6)).reshape(-1)
    A = torch.repeat_interleave(adv, torch.tensor(np.diff(x["cu_seqlens"])))
    lp = torch.log_softmax(H @ W.T, dim=-1).gather(1, y[:, None])[:, 0]
    rho = torch.exp(lp - torch.tensor(x["old_logp"]))
    s = torch.minimum(rho * A, torch.clamp(rho, 0.8, 1.28) * A)
    if dual:
        s = torch.where(A < 0, torch.maximum(s, dual * A), s)
    logr = torch.tensor(x["ref_logp"]) - lp
    k = {0: torch.exp(logr) - 1 - logr, 1: -logr, 2: 0.5 * logr ** 2}[kl_type]
    loss = (-s + 0.05 * k).mean()
    loss.backward()
    np.testing.assert_allclose(out["loss"], loss.item(), rtol=1e-12)
    np.testing.assert_allclose(out["dH"], H.grad.numpy(), rtol=1e-9, atol=1e-16)
    np.testing.assert_allclose(out["dW"], W.grad.numpy(), rtol=1e-9, atol=1e-16)


def test_variants_loops_oracle_agrees():
    t = _tiny(seed=9, spread=0.5)
    for kl_type, dual in [(1, 0.0), (2, 1.7), (0, 1.7)]:
        cfg = OracleConfig(kl_beta=0.03, kl_type=kl_type, dual_clip=dual)
        a = grpo_step(t["H"], t["W"], t["y"], t["cu_seqlens"], t["rewards"], t["old_logp"], t["ref_logp"], cfg=cfg, G=2)
        b = grpo_step_loops(t["H"].tolist(), t["W"].tolist(), t["y"].tolist(), t["cu_seqlens"].tolist(),
                            t["rewards"].tolist(), t["old_logp"].tolist(), t["ref_logp"].tolist(), cfg=cfg, G=2)
        for k in ("coeff", "dH", "dW"):
            np.testing.assert_allclose(a[k], b[k], rtol=1e-11, atol=1e-15, err_msg=k)
        np.testing.assert_allclose(a["loss"], b["loss"], rtol=1e-12)


# ------------------------------------------------------------------------------------------- entropy (R28)
def test_entropy_pins():
    """Uniform policy -> ln V; two classes -> binary entropy of the logistic; library routine; bounds; the
    identity entropy = lse - sum_v p_v z_v that the kernel's online form uses."""
    import scipy.stats
    from oracle.grpo_oracle import token_entropy, token_logprobs
    rng = np.random.default_rng(3)
    H = rng.normal(size=(6, 5))
    assert np.allclose(token_entropy(H, np.zeros((9, 5))), np.log(9.0), rtol=1e-14)
    W2 = rng.normal(size=(2, 5))
    q = 1.0 / (1.0 + np.exp(-(H @ (W2[0] - W2[1]))))
    np.testing.assert_allclose(token_entropy(H, W2), -(q * np.log(q) + (1 - q) * np.log(1 - q)), rtol=1e-10)
    W = rng.normal(size=(13, 5))
    ent = token_entropy(H, W, logit_scale=1.7)
    z = 1.7 * H @ W.T
    p = np.exp(z - z.max(1, keepdims=True)); p /= p.sum(1, keepdims=True)
    np.testing.assert_allclose(ent, scipy.stats.entropy(p, axis=1), rtol=1e-12)
    assert np.all(ent > 0) and np.all(ent < np.log(13.0))
    lse, _ = token_logprobs(H, W, np.zeros(6, dtype=np.int64), logit_scale=1.7)
    np.testing.assert_allclose(ent, lse - (p * z).sum(1), rtol=1e-12)
    # a sharply peaked policy has (almost) no entropy; chunking does not matter
    assert token_entropy(H, W, logit_scale=200.0).max() < 1e-3
    np.testing.assert_array_equal(token_entropy(H, W, chunk_tokens=2), token_entropy(H, W, chunk_tokens=100))
