"""Pins for the oracle's final-RMSNorm extension (R29-R31).  CPU only.

The paper never mentions the norm, so every pin is a hand-worked value, a library routine
(torch.nn.functional.rms_norm and its autograd), an identity or a finite difference."""
import math

import numpy as np
import pytest
import torch

from oracle.grpo_oracle import (OracleConfig, grpo_step, grpo_step_from_prenorm, rmsnorm_bwd, rmsnorm_fwd,
                                round_to_bf16)


def test_hand_worked_two_by_two():
    """x = [[3, 4], [0, -2]], gamma = [1, 2], eps = 0:  mean x^2 = 12.5 and 2;  rstd = 1/sqrt(12.5), 1/sqrt(2);
    H = [[3, 8] / sqrt(12.5), [0, -4] / sqrt(2)]."""
    H, rstd = rmsnorm_fwd(np.array([[3.0, 4.0], [0.0, -2.0]]), np.array([1.0, 2.0]), eps_rms=0.0, round_bf16=False)
    np.testing.assert_allclose(rstd, [0.282842712474619, 0.7071067811865476], rtol=1e-15)
    np.testing.assert_allclose(H, [[0.848528137423857, 2.262741699796952], [0.0, -2.8284271247461903]], rtol=1e-15)
    # backward by hand for row 0, dH = [1, 0]: g = gamma*dH = [1, 0]; xh = [3, 4]/sqrt(12.5);
    # mean(g xh) = 3 / (2 sqrt(12.5));  dx = rstd (g - xh mean) = [1 - 9/25, -12/25] / sqrt(12.5)
    dx, dg = rmsnorm_bwd(np.array([[3.0, 4.0]]), np.array([1.0, 2.0]), rstd[:1], np.array([[1.0, 0.0]]))
    np.testing.assert_allclose(dx, [[0.64 / math.sqrt(12.5), -0.48 / math.sqrt(12.5)]], rtol=1e-14)
    np.testing.assert_allclose(dg, [3.0 / math.sqrt(12.5), 0.0], rtol=1e-14, atol=1e-16)


def test_against_torch_rms_norm_and_its_autograd():
    rng = np.random.default_rng(0)
    T, d, eps = 7, 12, 1e-6
    x, gamma, dH = rng.normal(size=(T, d)) * 3, rng.normal(size=d) + 1.0, rng.normal(size=(T, d))
    H, rstd = rmsnorm_fwd(x, gamma, eps, round_bf16=False)
    xt = torch.tensor(x, requires_grad=True)
    gt = torch.tensor(gamma, requires_grad=True)
    Ht = torch.nn.functional.rms_norm(xt, (d,), gt, eps)
    np.testing.assert_allclose(H, Ht.detach().numpy(), rtol=1e-13)
    Ht.backward(torch.tensor(dH))
    dx, dgamma = rmsnorm_bwd(x, gamma, rstd, dH)
    np.testing.assert_allclose(dx, xt.grad.numpy(), rtol=1e-11, atol=1e-14)
    np.testing.assert_allclose(dgamma, gt.grad.numpy(), rtol=1e-12)


def test_identities():
    rng = np.random.default_rng(1)
    T, d = 5, 16
    x, gamma, dH = rng.normal(size=(T, d)), rng.normal(size=d), rng.normal(size=(T, d))
    H, rstd = rmsnorm_fwd(x, gamma, 0.0, round_bf16=False)
    np.testing.assert_allclose(((H / gamma) ** 2).mean(axis=1), 1.0, rtol=1e-13)         # unit RMS before the weight
    H2, _ = rmsnorm_fwd(7.5 * x, gamma, 0.0, round_bf16=False)
    np.testing.assert_allclose(H2, H, rtol=1e-13)                                         # scale invariance (eps = 0)
    dx, _ = rmsnorm_bwd(x, gamma, rstd, dH)
    np.testing.assert_allclose((dx * x).sum(axis=1), 0.0, atol=1e-13)                     # hence dx is orthogonal to x
    # with eps > 0 the radial component is rstd^3 eps (gamma dH . x) exactly
    eps = 0.37
    _, rstd_e = rmsnorm_fwd(x, gamma, eps, round_bf16=False)
    dx_e, _ = rmsnorm_bwd(x, gamma, rstd_e, dH)
    np.testing.assert_allclose((dx_e * x).sum(axis=1), rstd_e ** 3 * eps * ((gamma * dH) * x).sum(axis=1), rtol=1e-12)


def test_round_to_bf16_is_torch_bf16():
    x = np.concatenate([np.random.default_rng(2).normal(size=5000) * 3, [1.00390625, 1.01171875, 0.0, -0.0, 255.5]])
    want = torch.tensor(x, dtype=torch.float32).to(torch.bfloat16).double().numpy()
    np.testing.assert_array_equal(round_to_bf16(x), want)
    H, _ = rmsnorm_fwd(x[:5000].reshape(50, 100), np.ones(100))
    np.testing.assert_array_equal(H, round_to_bf16(H))                                    # H is on the bf16 grid (R29)


def _tiny(seed=3):
    rng = np.random.default_rng(seed)
    lens = np.array([3, 4, 2, 3])
    cu = np.concatenate([[0], np.cumsum(lens)])
    T, d, V = int(cu[-1]), 6, 7
    x = rng.normal(size=(T, d)) * 2.0
    gamma = 1.0 + 0.3 * rng.normal(size=d)
    W = rng.normal(size=(V, d)) * 0.7
    y = rng.integers(0, V, size=T)
    rewards = np.array([1.0, 0.0, 0.0, 1.0])
    H, _ = rmsnorm_fwd(x, gamma, 1e-6, round_bf16=False)
    z = H @ W.T
    lp = z[np.arange(T), y] - np.log(np.exp(z).sum(1))
    return dict(x=x, gamma=gamma, W=W, y=y, cu=cu, rewards=rewards, old=lp + 0.1 * rng.normal(size=T),
                ref=lp + 0.1 * rng.normal(size=T))


@pytest.mark.parametrize("loss_agg,beta", [(0, 0.0), (0, 0.05), (1, 0.05)])
def test_whole_step_finite_differences_wrt_prenorm_inputs(loss_agg, beta):
    """Central differences of the loss w.r.t. EVERY entry of x and gamma (rounding off: the rounded function is
    piecewise constant), through RMSNorm -> log-softmax -> clipped surrogate + k3 -> masked mean."""
    t = _tiny()
    cfg = OracleConfig(kl_beta=beta, loss_agg=loss_agg, logit_scale=0.9)
    mask = np.ones(len(t["y"]), dtype=np.uint8)
    mask[5] = 0

    def run(x, gamma, grads=False):
        o = grpo_step_from_prenorm(x, gamma, t["W"], t["y"], t["cu"], t["rewards"], t["old"], t["ref"], mask=mask,
                                   cfg=cfg, G=2, round_bf16=False)
        return o if grads else o["loss"]

    out = run(t["x"], t["gamma"], grads=True)
    rho = out["rho"]
    assert np.all(np.abs(rho - 0.8) > 1e-3) and np.all(np.abs(rho - 1.28) > 1e-3)         # away from the clip kinks
    h = 1e-6
    fd_x = np.zeros_like(t["x"])
    for i in range(t["x"].shape[0]):
        for k in range(t["x"].shape[1]):
            xp, xm = t["x"].copy(), t["x"].copy()
            xp[i, k] += h
            xm[i, k] -= h
            fd_x[i, k] = (run(xp, t["gamma"]) - run(xm, t["gamma"])) / (2 * h)
    np.testing.assert_allclose(out["dx"], fd_x, rtol=2e-6, atol=2e-9)
    fd_g = np.zeros_like(t["gamma"])
    for k in range(t["gamma"].size):
        gp, gm = t["gamma"].copy(), t["gamma"].copy()
        gp[k] += h
        gm[k] -= h
        fd_g[k] = (run(t["x"], gp) - run(t["x"], gm)) / (2 * h)
    np.testing.assert_allclose(out["dgamma"], fd_g, rtol=2e-6, atol=2e-9)
    assert np.all(out["dx"][5] == 0.0)                                                    # masked token: no gradient


def test_prenorm_step_is_the_plain_step_on_the_normalised_hidden_state():
    t = _tiny(seed=4)
    cfg = OracleConfig(kl_beta=0.01)
    a = grpo_step_from_prenorm(t["x"], t["gamma"], t["W"], t["y"], t["cu"], t["rewards"], t["old"], t["ref"], cfg=cfg, G=2)
    H, rstd = rmsnorm_fwd(t["x"], t["gamma"])
    b = grpo_step(H, t["W"], t["y"], t["cu"], t["rewards"], t["old"], t["ref"], cfg=cfg, G=2)
    for k in ("logp", "loss", "coeff", "dH", "dW"):
        np.testing.assert_array_equal(a[k], b[k])
    # and the float64 torch autograd of the written-out chain (straight-through rounding: use the unrounded chain)
    a = grpo_step_from_prenorm(t["x"], t["gamma"], t["W"], t["y"], t["cu"], t["rewards"], t["old"], None, cfg=OracleConfig(),
                               G=2, round_bf16=False)
    x = torch.tensor(t["x"], requires_grad=True)
    g = torch.tensor(t["gamma"], requires_grad=True)
    Ht = torch.nn.functional.rms_norm(x, (x.shape[1],), g, 1e-6)
    lp = torch.log_softmax(Ht @ torch.tensor(t["W"]).T, dim=-1)[torch.arange(len(t["y"])), torch.tensor(t["y"])]
    A = torch.tensor(np.repeat(a["adv"], np.diff(t["cu"])))
    rho = torch.exp(lp - torch.tensor(t["old"]))
    loss = -(torch.minimum(rho * A, rho.clamp(0.8, 1.28) * A)).mean()
    loss.backward()
    np.testing.assert_allclose(a["loss"], loss.item(), rtol=1e-12)
    np.testing.assert_allclose(a["dx"], x.grad.numpy(), rtol=1e-9, atol=1e-15)
    np.testing.assert_allclose(a["dgamma"], g.grad.numpy(), rtol=1e-9, atol=1e-15)


# ------------------------------------------------------------------ FP8 study: the E4M3 rounding of the oracle
def test_e4m3_round_is_torch_float8_e4m3fn():
    """Library routine: torch's float8_e4m3fn conversion (round to nearest even).  Every representable magnitude,
    every midpoint between neighbours (ties), random values over the whole range, and saturation at 448."""
    from oracle.grpo_oracle import e4m3_round, fp8_dequantized_operands
    grid = torch.arange(0, 256, dtype=torch.uint8).view(torch.float8_e4m3fn).float()
    grid = np.sort(np.unique(grid[torch.isfinite(grid)].double().numpy()))
    assert grid.max() == 448.0 and 2.0 ** -9 in grid and len(grid) == 253                  # 2 x 126 + zero
    mids = (grid[1:] + grid[:-1]) / 2
    rng = np.random.default_rng(0)
    rand = rng.normal(size=20000) * 10.0 ** rng.uniform(-4, 2.6, size=20000)
    x = np.concatenate([grid, mids, rand, [447.9, 448.0, 463.9, 1e-12, -1e-12, 0.0]])
    x = x[np.abs(x) <= 464.0]                  # beyond the last midpoint torch's e4m3fn gives NaN; the kernel saturates
    want = torch.tensor(x, dtype=torch.float32).to(torch.float8_e4m3fn).double().numpy()
    got = e4m3_round(np.float32(x))
    np.testing.assert_array_equal(got, want)
    np.testing.assert_array_equal(e4m3_round(np.array([500.0, -1e6, 449.0])), [448.0, -448.0, 448.0])   # satfinite
    # the recipe: per-row scale amax/448 for H, one scale for W; the row maximum itself is represented exactly
    H = rng.normal(size=(5, 16))
    H[3] = 0.0
    W = rng.normal(size=(7, 16)) * 0.02
    Hq, Wq = fp8_dequantized_operands(H, W)
    np.testing.assert_allclose(np.abs(Hq).max(axis=1), np.abs(np.float32(H)).max(axis=1), rtol=1e-6)
    assert np.all(Hq[3] == 0.0)
    np.testing.assert_allclose(np.abs(Wq).max(), np.abs(np.float32(W)).max(), rtol=1e-6)
    assert np.abs(Hq - H).max() <= np.abs(H).max() * 2.0 ** -4 and np.abs(Wq - W).max() <= np.abs(W).max() * 2.0 ** -4
