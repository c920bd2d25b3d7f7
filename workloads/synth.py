"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the oracle and the CUDA path with identical bits and holds
none of the method's arithmetic: it draws lengths, rewards, hidden states, the vocab
matrix and target tokens, and synthesises "old" / "ref" log-probs as
``base_logp + noise``.  ``base_logp`` is a plain fp32 ``log_softmax(H W^T)`` done with
stock torch ops in token chunks (on whatever device the tensors live on); it is input
synthesis (how the rollout engine would have produced ``old_logp``), is never compared
against anything, and is used by neither the oracle nor the kernels.

The inputs stand in for the paper's workloads (LSAT-AR, SciBench subsets,
OlympiadBench physics with Qwen3-1.7B): only their *shape*
parameters enter this path — K=8 responses per prompt, binary exact-match reward,
3.3k-3.6k-token responses.  No benchmark item is reproduced.

Recipe: seed = 26997*10 + cfg (+ user seed); draw order
lengths -> p_g -> rewards -> W -> H -> base logits -> targets -> old noise -> ref noise.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np
import torch

QWEN3_D = 2048
QWEN3_V = 151936


@dataclass
class GrpoBatch:
    name: str
    n_groups: int
    G: int
    d: int
    V: int
    seqlens: np.ndarray              # int32 [S]
    cu_seqlens: torch.Tensor         # int32 [S+1]
    rewards: torch.Tensor            # fp32 [S]
    hidden: torch.Tensor             # bf16 [T, d]
    W: torch.Tensor                  # bf16 [V, d]
    targets: torch.Tensor            # int32 [T]
    old_logp: torch.Tensor           # fp32 [T]
    ref_logp: Optional[torch.Tensor]  # fp32 [T] or None
    mask: Optional[torch.Tensor]     # uint8 [T] or None
    clip_lo: float = 0.2
    clip_hi: float = 0.28
    kl_beta: float = 0.0
    eps_std: float = 1e-6
    loss_agg: int = 0
    arrival_order: Optional[np.ndarray] = None   # cfg 5: order groups are enqueued in
    zero_var_frac: float = 0.0
    x_prenorm: Optional[torch.Tensor] = None     # bf16 [T, d]: pre-norm activations (prenorm=True only)
    gamma: Optional[torch.Tensor] = None         # bf16 [d]: RMSNorm weight (prenorm=True only)
    eps_rms: float = 1e-6

    @property
    def T(self) -> int:
        return int(self.hidden.shape[0])

    @property
    def S(self) -> int:
        return int(self.seqlens.size)

    def group_token_range(self, g: int):
        cu = np.concatenate([[0], np.cumsum(self.seqlens)])
        return int(cu[g * self.G]), int(cu[(g + 1) * self.G])

    def to(self, device):
        kw = {}
        for k, v in self.__dict__.items():
            kw[k] = v.to(device) if isinstance(v, torch.Tensor) else v
        return GrpoBatch(**kw)

    def numpy_f64(self):
        """Exact float64 views for the oracle (bf16 -> f64 is exact)."""
        f = lambda t: None if t is None else t.detach().cpu().to(torch.float64).numpy()
        return dict(H=f(self.hidden), W=f(self.W),
                    y=self.targets.cpu().numpy().astype(np.int64),
                    cu_seqlens=self.cu_seqlens.cpu().numpy().astype(np.int64),
                    rewards=f(self.rewards), old_logp=f(self.old_logp), ref_logp=f(self.ref_logp),
                    mask=None if self.mask is None else self.mask.cpu().numpy(),
                    x=f(self.x_prenorm), gamma=f(self.gamma))


# ------------------------------------------------------------------ small draws (numpy)
def _lengths(cfg: int, rng: np.random.Generator, S: int, len_div: float) -> np.ndarray:
    if cfg == 1:
        L = rng.integers(8, 33, size=S)
    elif cfg == 2:
        L = rng.integers(512, 4097, size=S)
    elif cfg == 3:
        L = np.clip(rng.lognormal(np.log(1500.0), 0.8, size=S), 64, 8192)
    elif cfg == 4:
        L = np.clip(rng.lognormal(np.log(2500.0), 1.0, size=S), 32, 16384)
    elif cfg == 5:
        L = np.minimum(rng.geometric(1.0 / 2000.0, size=S), 8192)
    else:
        raise ValueError(cfg)
    L = np.asarray(L, dtype=np.float64)
    if len_div != 1.0:
        L = L / len_div
    return np.maximum(np.floor(L), 1).astype(np.int32)


def _rewards(cfg: int, rng: np.random.Generator, n_groups: int, G: int) -> np.ndarray:
    if cfg == 2:
        # Bernoulli(0.5); redraw until the single group has variance (SURVEY §8(d) cfg 2)
        if G < 2:
            raise ValueError("config 2 redraws until the group has variance: needs G >= 2")
        while True:
            r = (rng.random((n_groups, G)) < 0.5).astype(np.float32)
            if np.all(r.std(axis=1) > 0):
                return r.reshape(-1)
    need_mix = cfg == 3
    if need_mix and n_groups < 2:
        raise ValueError("config 3 keeps at least one zero-variance and one other group (R19): needs n_groups >= 2")
    while True:
        p = rng.beta(0.5, 0.5, size=n_groups)
        r = (rng.random((n_groups, G)) < p[:, None]).astype(np.float32)
        zv = r.std(axis=1) == 0
        if not need_mix or (zv.any() and (~zv).any()):
            return r.reshape(-1)


_SHAPES = {1: (4, 4, 64, 1000), 2: (1, 8, QWEN3_D, QWEN3_V), 3: (4, 8, QWEN3_D, QWEN3_V),
           4: (8, 16, QWEN3_D, QWEN3_V), 5: (32, 8, QWEN3_D, QWEN3_V)}
_OLD_SIGMA = {1: 0.05, 2: 0.0, 3: 0.02, 4: 0.02, 5: 0.02}
_BETA = {1: 0.001, 2: 0.0, 3: 0.001, 4: 0.0, 5: 0.0}


@torch.no_grad()
def base_logp_and_targets(H, W, gen, sample: str, chunk: int = 2048):
    """fp32 log_softmax(H W^T) in chunks; targets uniform or Gumbel-max from the softmax."""
    T, V = H.shape[0], W.shape[0]
    dev = H.device
    y = torch.empty(T, dtype=torch.int64, device=dev)
    lp = torch.empty(T, dtype=torch.float32, device=dev)
    Wf = W.float()
    for t0 in range(0, T, chunk):
        t1 = min(T, t0 + chunk)
        z = H[t0:t1].float() @ Wf.T
        lsm = torch.log_softmax(z, dim=-1)
        if sample == "uniform":
            yy = torch.randint(0, V, (t1 - t0,), generator=gen, device=dev)
        else:
            u = torch.rand(z.shape, generator=gen, device=dev).clamp_(1e-20, 1.0)
            yy = torch.argmax(lsm - torch.log(-torch.log(u)), dim=-1)
        y[t0:t1] = yy
        lp[t0:t1] = lsm.gather(1, yy[:, None])[:, 0]
    return lp, y.to(torch.int32)


@torch.no_grad()
def make_config(cfg: int, seed: int = 0, device="cpu", *, d: int | None = None, V: int | None = None,
                n_groups: int | None = None, G: int | None = None, len_div: float = 1.0,
                old_sigma: float | None = None, kl_beta: float | None = None,
                mask_frac: float = 0.0, loss_agg: int = 0, variant: str = "", w_std: float = 0.02,
                bad_target_frac: float = 0.0, prenorm: bool = False) -> GrpoBatch:
    """Build config ``cfg`` (1-5).  Keyword overrides shrink it for CPU-sized parity cases.

    variant "1b": config 1 with old-logprob noise sigma = 0.3 so both clip regions are
    populated (the BASELINE configs never exercise the clip).

    prenorm=True (NEXT-4): the batch also carries pre-norm activations ``x_prenorm`` (rows N(0,1) times a
    per-row lognormal scale, bf16) and a norm weight ``gamma`` (1 + 0.1 N(0,1), bf16); ``hidden`` is then the
    stock-torch fp32 ``rms_norm(x, gamma)`` rounded to bf16 - input synthesis, so that old / ref log-probs are
    those of the normalised states; neither the oracle nor the kernels read ``hidden`` in the pre-norm tests.
    """
    ng0, G0, d0, V0 = _SHAPES[cfg]
    n_groups = n_groups or ng0
    G = G or G0
    d = d or d0
    V = V or V0
    S = n_groups * G
    base_seed = 26997 * 10 + cfg + 1000003 * seed
    rng = np.random.default_rng(base_seed)
    seqlens = _lengths(cfg, rng, S, len_div)
    rewards = _rewards(cfg, rng, n_groups, G)
    zero_var_frac = float(np.mean(rewards.reshape(n_groups, G).std(axis=1) == 0))
    T = int(seqlens.sum())
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(base_seed)
    W = (torch.randn(V, d, generator=gen, device=dev, dtype=torch.float32) * w_std).to(torch.bfloat16)
    Hf = torch.randn(T, d, generator=gen, device=dev, dtype=torch.float32)
    x_pre = gamma = None
    if prenorm:
        x_pre = (Hf * torch.exp(0.5 * torch.randn(T, 1, generator=gen, device=dev))).to(torch.bfloat16)
        gamma = (1.0 + 0.1 * torch.randn(d, generator=gen, device=dev)).to(torch.bfloat16)
        Hf = torch.nn.functional.rms_norm(x_pre.float(), (d,), gamma.float(), 1e-6)
    elif cfg != 1:   # "after RMSNorm-like scaling": unit-RMS rows (R16)
        Hf = Hf * torch.rsqrt(Hf.pow(2).mean(dim=1, keepdim=True) + 1e-12)
    H = Hf.to(torch.bfloat16)
    del Hf
    base_lp, y = base_logp_and_targets(H, W, gen, "uniform" if cfg == 1 else "softmax")
    sig = _OLD_SIGMA[cfg] if old_sigma is None else old_sigma
    if variant == "1b":
        sig = 0.3
    old = base_lp + sig * torch.randn(T, generator=gen, device=dev)
    beta = _BETA[cfg] if kl_beta is None else kl_beta
    ref = base_lp + 0.1 * torch.randn(T, generator=gen, device=dev) if beta != 0.0 else None
    mask = None
    if mask_frac > 0.0:
        mask = (torch.rand(T, generator=gen, device=dev) >= mask_frac).to(torch.uint8)
    if bad_target_frac > 0.0:   # ignored tokens (y < 0) — exercises DESIGN.md R13
        bad = torch.rand(T, generator=gen, device=dev) < bad_target_frac
        y = torch.where(bad, torch.full_like(y, -100), y)
    cu = np.concatenate([[0], np.cumsum(seqlens)]).astype(np.int32)
    arrival = rng.permutation(n_groups) if cfg == 5 else None
    return GrpoBatch(
        name=f"cfg{cfg}{variant}", n_groups=n_groups, G=G, d=d, V=V, seqlens=seqlens,
        cu_seqlens=torch.from_numpy(cu).to(dev), rewards=torch.from_numpy(rewards).to(dev),
        hidden=H, W=W, targets=y, old_logp=old.float(), ref_logp=None if ref is None else ref.float(),
        mask=mask, kl_beta=beta, loss_agg=loss_agg, arrival_order=arrival, zero_var_frac=zero_var_frac,
        x_prenorm=x_pre, gamma=gamma)


def slice_groups(b: GrpoBatch, groups) -> GrpoBatch:
    """Sub-batch made of whole groups (views of the packed stream re-packed contiguously)."""
    groups = list(groups)
    cu = np.concatenate([[0], np.cumsum(b.seqlens)])
    tok = np.concatenate([np.arange(cu[g * b.G], cu[(g + 1) * b.G]) for g in groups])
    seq = np.concatenate([np.arange(g * b.G, (g + 1) * b.G) for g in groups])
    ti = torch.from_numpy(tok).to(b.hidden.device)
    si = torch.from_numpy(seq).to(b.hidden.device)
    sl = b.seqlens[seq]
    cu2 = np.concatenate([[0], np.cumsum(sl)]).astype(np.int32)
    pick = lambda t: None if t is None else t[ti].contiguous()
    return GrpoBatch(
        name=b.name + "_sub", n_groups=len(groups), G=b.G, d=b.d, V=b.V, seqlens=sl,
        cu_seqlens=torch.from_numpy(cu2).to(b.hidden.device), rewards=b.rewards[si].contiguous(),
        hidden=pick(b.hidden), W=b.W, targets=pick(b.targets), old_logp=pick(b.old_logp),
        ref_logp=pick(b.ref_logp), mask=pick(b.mask), clip_lo=b.clip_lo, clip_hi=b.clip_hi,
        kl_beta=b.kl_beta, eps_std=b.eps_std, loss_agg=b.loss_agg)
