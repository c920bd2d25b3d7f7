"""CPU self-tests of the gates the GPU parity tests apply (tests/parity_util.py): each gate must accept a result
with the kernel's arithmetic (dZ rounded to bf16, fp32 accumulation) and must reject the mistake it exists to
catch.  The "kernel-like" result is built from the oracle's own float64 quantities plus bf16 rounding of dZ —
no CUDA code is involved."""
import numpy as np
import torch

from oracle.grpo_oracle import OracleConfig, grpo_step
from tests.parity_util import assert_gates, bf16_round, gates, worst_block_rel
from workloads.synth import make_config


def test_bf16_round_matches_torch():
    x = np.concatenate([np.random.default_rng(0).normal(size=4000) * 10.0 ** np.random.default_rng(1).integers(-8, 8, 4000),
                        [0.0, 1.0, -1.0, 1.00390625, 1.01171875, 3.0e38]])
    want = torch.tensor(x, dtype=torch.float32).to(torch.bfloat16).double().numpy()
    np.testing.assert_array_equal(bf16_round(x), want)


def _kernel_like(b, logit_scale=1.0, dense_gain=1.0, bad_block=None):
    """Oracle step on batch b, then dH / dW as the CUDA path forms them: dZ = bf16(c s (1[v=y] - p)), dH = dZ W,
    dW = dZ^T H.  dense_gain scales the v != y entries of dZ (a wrong softmax term)."""
    x = b.numpy_f64()
    cfg = OracleConfig(eps_std=b.eps_std, clip_lo=b.clip_lo, clip_hi=b.clip_hi, kl_beta=b.kl_beta, loss_agg=b.loss_agg,
                       logit_scale=logit_scale)
    ref = grpo_step(x["H"], x["W"], x["y"], x["cu_seqlens"], x["rewards"], x["old_logp"], x["ref_logp"], mask=x["mask"],
                    cfg=cfg, G=b.G)
    z = logit_scale * x["H"] @ x["W"].T
    dz = -np.exp(z - ref["lse"][:, None]) * dense_gain
    ok = (x["y"] >= 0) & (x["y"] < b.V)
    rows = np.arange(b.T)[ok]
    dz[rows, x["y"][ok]] = 1.0 - np.exp(ref["logp"][ok])
    dz = bf16_round(dz * (ref["coeff"] * logit_scale)[:, None])
    dH, dW = dz @ x["W"], dz.T @ x["H"]
    if bad_block is not None:
        r0, c0 = bad_block
        dW[r0:r0 + 32, c0:c0 + 32] *= 1.5
    out = dict(adv=torch.tensor(ref["adv"]), logp=torch.tensor(ref["logp"]), lse=torch.tensor(ref["lse"]),
               loss=torch.tensor(ref["loss"]), coeff=torch.tensor(ref["coeff"]),
               dH=torch.tensor(dH, dtype=torch.float32), dW=torch.tensor(dW, dtype=torch.float32))
    return out, ref


def test_gates_accept_bf16_dz_arithmetic():
    for kw in (dict(), dict(mask_frac=0.3, bad_target_frac=0.1), dict(w_std=1.5)):
        b = make_config(1, seed=5, variant="1b", **kw)
        out, ref = _kernel_like(b)
        e = gates(b, out, ref)
        assert_gates(e)
        assert e["dH_dense_rel"] < 5e-3 and e["dW_block_rel"] < 1e-2 and e["dH_row_rel"] < 5e-3, e


def test_dense_gate_rejects_a_wrong_softmax_term_the_global_norm_hides():
    """SURVEY.md §8(c) gate (ii): with the near-uniform synthetic softmax the dense part is ~2 % of ||dH||, so a
    dense term wrong by 5 % moves the whole-matrix rel-L2 by ~1e-3 (passes 1e-2) but must fail gate (ii)."""
    b = make_config(1, seed=5, variant="1b")
    out, ref = _kernel_like(b, dense_gain=1.05)
    e = gates(b, out, ref)
    assert e["dH_rel"] <= 1e-2                     # hidden in the Frobenius norm of the whole matrix
    assert e["dH_dense_rel"] > 3e-2                # caught by the dense-part gate
    try:
        assert_gates(e)
    except AssertionError:
        return
    raise AssertionError("a 5 % error of the dense softmax term passed the gates")


def test_block_gate_rejects_one_wrong_tile():
    b = make_config(1, seed=5, variant="1b")
    out, ref = _kernel_like(b, bad_block=(512, 32))
    e = gates(b, out, ref)
    assert e["dW_rel"] <= 1e-2 or True             # (reported) the global norm may or may not notice one tile
    assert e["dW_block_rel"] > 0.3
    try:
        assert_gates(e)
    except AssertionError:
        pass
    else:
        raise AssertionError("one wrong 32 x 32 block of dW passed the gates")
    # zero reference blocks must be exactly zero
    r = np.zeros((64, 64)); r[:32] = 1.0
    a = r.copy(); a[40, 3] = 1e-9
    assert worst_block_rel(a, r) == float("inf")
    assert worst_block_rel(r, r) == 0.0
