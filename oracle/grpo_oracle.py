"""Float64 CPU oracle for the fused GRPO policy-loss step.

TEST INFRASTRUCTURE ONLY.  Nothing in the product path (``paper_2606_26997_b200``)
imports this module; only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may call it.  It shares
no code, tables or helpers with the CUDA path.

What it computes is the *plain definition* of the step:
the method reaches an exactly defined result, so there is no tiling, no online
log-sum-exp and no fusion here.  Logits ARE materialised (in token chunks, only to
bound memory).  All arithmetic is float64; bf16 inputs are widened exactly.

Passages followed:
  * group advantage ............ Eq. 1, PAPER.md:86-90 (sigma reading: DESIGN.md R1-R4)
  * one advantage per response, broadcast over its tokens + loss mask ... PAPER.md:40
  * clipped surrogate with current/old ratios ...... PAPER.md:38 (form: north_star)
  * k3 KL, masked token mean, backward (softmax - onehot) * coeff ...... north_star
  * gradients only accumulated across groups of a logical update ..... PAPER.md:111

NEXT-2 switches (paper silent; R26-R28): k1 / k2 KL estimators, dual clip, per-token entropy —
pinned in tests/test_oracle_variants.py (E[k1] = E[k3] = KL, derivative checks, a hand-evaluated dual-clip
table, finite differences, torch autograd, closed-form / library entropies); "parity unpinned" by the paper.

NEXT-4 (R29-R31): the final RMSNorm in front of the path and its backward
(``rmsnorm_fwd`` / ``rmsnorm_bwd`` / ``grpo_step_from_prenorm``) — pinned in tests/test_oracle_rmsnorm.py by a
hand-worked example, ``torch.nn.functional.rms_norm`` and its autograd, scale invariance / orthogonality
identities and finite differences of the whole step w.r.t. the pre-norm activations and the norm weight;
"parity unpinned" by the paper (it never mentions the norm).  FP8 precision study (R32): ``e4m3_round`` is pinned
against torch's float8_e4m3fn conversion on every representable value, its midpoints and random inputs.

Pins (tests/test_oracle_pins.py): P1-P14 of SURVEY.md §8(c).  The paper prints no
worked number for the loss, so every pin is a closed form, invariant, library special
case, finite difference or brute force.  Unpinned by the paper: everything except
Eq. 1 — pinned here by P4-P14 only.  ``metrics`` (clip fraction etc.) are pinned by a five-token
case worked by hand (test_metrics_and_loss_hand_evaluated_five_tokens) and by brute-force loops.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

__all__ = [
    "OracleConfig", "bf16_bits_to_f64", "group_advantage", "token_advantage",
    "token_logprobs", "loss_terms", "backward", "grpo_step", "grpo_step_loops",
    "token_rows", "dH_rows", "dW_rows", "token_entropy",
    "round_to_bf16", "rmsnorm_fwd", "rmsnorm_bwd", "grpo_step_from_prenorm",
    "e4m3_round", "fp8_dequantized_operands",
]


@dataclass
class OracleConfig:
    eps_std: float = 1e-6        # Eq. 1 stabiliser ("a small stabilizer")
    std_ddof: int = 0            # 0 population std (default reading), 1 sample std
    clip_lo: float = 0.2
    clip_hi: float = 0.28
    kl_beta: float = 0.0         # 0 disables the k3 term
    loss_agg: int = 0            # 0 token mean over the logical update, 1 per-sequence mean
    logit_scale: float = 1.0     # 1 / temperature
    kl_type: int = 0             # NEXT-2: 0 = k3 (north_star), 1 = k1, 2 = k2 (R26)
    dual_clip: float = 0.0       # NEXT-2: 0 = off; c > 1: for A < 0 the surrogate is max(s, c A) (R27)
    chunk_tokens: int = 1024     # memory bound only; results do not depend on it


def bf16_bits_to_f64(bits: np.ndarray) -> np.ndarray:
    """uint16 bf16 bit patterns -> float64, exactly (bf16 is the top half of an fp32)."""
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


# --------------------------------------------------------------------------- step 1
def group_advantage(rewards, cu_groups=None, G=None, eps_std=1e-6, ddof=0):
    """Eq. 1:  A_i = (r_i - mu_group) / (sigma_group + eps_std).

    ``cu_groups`` [n_groups+1] gives ragged group boundaries; otherwise groups are
    uniform of size ``G``.  sigma uses divisor (G - ddof); if that is <= 0, sigma = 0.
    Returns (adv float64 [S], zero_var bool [n_groups]).
    """
    r = np.asarray(rewards, dtype=np.float64)
    if cu_groups is None:
        assert G is not None and r.size % G == 0
        cu = np.arange(0, r.size + 1, G, dtype=np.int64)
    else:
        cu = np.asarray(cu_groups, dtype=np.int64)
    adv = np.zeros_like(r)
    zero_var = np.zeros(cu.size - 1, dtype=bool)
    for g in range(cu.size - 1):
        rg = r[cu[g]:cu[g + 1]]
        n = rg.size
        if n == 0:
            zero_var[g] = True
            continue
        mu = rg.sum() / n
        dev = rg - mu
        div = n - ddof
        sigma = np.sqrt((dev * dev).sum() / div) if div > 0 else 0.0
        adv[cu[g]:cu[g + 1]] = dev / (sigma + eps_std)
        zero_var[g] = bool(sigma == 0.0)
    return adv, zero_var


# --------------------------------------------------------------------------- step 2
def token_advantage(adv, cu_seqlens):
    """A_t = A_seq(t): one advantage per response, broadcast to its tokens."""
    cu = np.asarray(cu_seqlens, dtype=np.int64)
    return np.repeat(np.asarray(adv, dtype=np.float64), np.diff(cu))


# ----------------------------------------------------------------------- steps 3, 4
def token_logprobs(H, W, y, logit_scale=1.0, chunk_tokens=1024):
    """z = s * H W^T ; lse_t = m + log sum_v exp(z_tv - m) ; logp_t = z_t[y_t] - lse_t.

    Tokens with y_t < 0 or y_t >= V are ignored (R13): logp = lse-only
    bookkeeping, ``zy`` taken as 0 and ``logp`` reported as 0.
    Returns (lse, logp) float64 [T].
    """
    H = np.asarray(H, dtype=np.float64)
    W = np.asarray(W, dtype=np.float64)
    y = np.asarray(y, dtype=np.int64)
    T, V = H.shape[0], W.shape[0]
    lse = np.zeros(T)
    logp = np.zeros(T)
    valid = (y >= 0) & (y < V)
    for t0 in range(0, T, chunk_tokens):
        t1 = min(T, t0 + chunk_tokens)
        z = logit_scale * (H[t0:t1] @ W.T)                       # [Tc, V] materialised
        m = z.max(axis=1)
        l = m + np.log(np.exp(z - m[:, None]).sum(axis=1))
        lse[t0:t1] = l
        yy = np.where(valid[t0:t1], y[t0:t1], 0)
        zy = z[np.arange(t1 - t0), yy]
        logp[t0:t1] = np.where(valid[t0:t1], zy - l, 0.0)
    return lse, logp


def token_entropy(H, W, logit_scale=1.0, chunk_tokens=1024):
    """NEXT-2 (R28): Shannon entropy of the policy at every packed row, in nats, by its definition
    on the materialised softmax:  p_tv = exp(z_tv - lse_t),  entropy_t = - sum_v p_tv log p_tv.
    A diagnostic output (no gradient flows through it).  Returns float64 [T]."""
    H = np.asarray(H, dtype=np.float64)
    W = np.asarray(W, dtype=np.float64)
    T = H.shape[0]
    ent = np.zeros(T)
    for t0 in range(0, T, chunk_tokens):
        t1 = min(T, t0 + chunk_tokens)
        z = logit_scale * (H[t0:t1] @ W.T)
        m = z.max(axis=1, keepdims=True)
        logp_all = z - (m + np.log(np.exp(z - m).sum(axis=1, keepdims=True)))
        p_all = np.exp(logp_all)
        ent[t0:t1] = -(p_all * logp_all).sum(axis=1)
    return ent


# ---------------------------------------------------------------------- steps 5 - 9a
def loss_terms(logp, old_logp, ref_logp, mask, adv_tok, cu_seqlens, cfg: OracleConfig,
               loss_denom=None, valid=None):
    """Per-token surrogate, k3, weights, loss, and c_t = d loss / d logp_t.

    rho = exp(logp - old);  s = min(rho A, clip(rho, 1-eps_lo, 1+eps_hi) A)
    delta = ref - logp;     k3 = exp(delta) - delta - 1
    l_t = -s_t + beta k3_t; loss = sum_t w_t l_t
    mode 0: w_t = m_t / denom, denom = max(sum m, 1) unless ``loss_denom`` given
    mode 1: w_t = m_t / (max(sum_{t' in seq(t)} m_t', 1) * S)
    u_t = 0 iff (A>0 and rho > 1+eps_hi) or (A<0 and rho < 1-eps_lo)   [bounds inclusive]
    c_t = w_t [ -A rho u + beta (1 - exp(ref - logp)) ]
    """
    logp = np.asarray(logp, dtype=np.float64)
    old = np.asarray(old_logp, dtype=np.float64)
    A = np.asarray(adv_tok, dtype=np.float64)
    T = logp.size
    cu = np.asarray(cu_seqlens, dtype=np.int64)
    S = cu.size - 1
    m = np.ones(T) if mask is None else (np.asarray(mask) != 0).astype(np.float64)
    if valid is not None:
        m = m * np.asarray(valid, dtype=np.float64)
    if cfg.loss_agg == 0:
        denom = max(m.sum(), 1.0) if (loss_denom is None or loss_denom <= 0) else float(loss_denom)
        w = m / denom
    else:
        w = np.zeros(T)
        for s in range(S):
            ms = m[cu[s]:cu[s + 1]]
            w[cu[s]:cu[s + 1]] = ms / (max(ms.sum(), 1.0) * S)
    rho = np.exp(logp - old)
    lo, hi = 1.0 - cfg.clip_lo, 1.0 + cfg.clip_hi
    surr = np.minimum(rho * A, np.clip(rho, lo, hi) * A)
    use_kl = cfg.kl_beta != 0.0 and ref_logp is not None
    if use_kl:
        # per-sample estimators of KL(pi || pi_ref) on samples from pi, with r = pi_ref / pi = exp(delta):
        #   k1 = -log r,   k2 = (log r)^2 / 2,   k3 = (r - 1) - log r      (R8, R26)
        delta = np.asarray(ref_logp, dtype=np.float64) - logp
        if cfg.kl_type == 1:
            k3 = -delta
            dk3 = np.ones(T)                           # d k1 / d logp
        elif cfg.kl_type == 2:
            k3 = 0.5 * delta * delta
            dk3 = -delta                               # d k2 / d logp
        else:
            k3 = np.exp(delta) - delta - 1.0
            dk3 = 1.0 - np.exp(delta)                  # d k3 / d logp
    else:
        k3 = np.zeros(T)
        dk3 = np.zeros(T)
    clipped = ((A > 0) & (rho > hi)) | ((A < 0) & (rho < lo))
    if cfg.dual_clip > 0.0:
        # dual clip (R27): a negative-advantage token whose ratio exceeds c contributes the
        # constant c A instead of rho A, so its policy gradient vanishes
        surr = np.where(A < 0, np.maximum(surr, cfg.dual_clip * A), surr)
        clipped = clipped | ((A < 0) & (rho > cfg.dual_clip))
    ell = -surr + cfg.kl_beta * k3
    u = np.where(clipped, 0.0, 1.0)
    coeff = w * (-A * rho * u + cfg.kl_beta * dk3)
    # w == 0 tokens (masked / invalid) contribute exact zeros even if ell is inf/nan-free
    ell_w = np.where(w != 0.0, w * ell, 0.0)
    coeff = np.where(w != 0.0, coeff, 0.0)
    loss = ell_w.sum()
    metrics = np.array([
        m.sum(),                                   # [0] loss-bearing tokens
        (m * rho).sum(),                           # [1] sum of rho over them
        (m * k3).sum(),                            # [2] sum of k3 over them
        (m * clipped).sum(),                       # [3] tokens whose policy gradient is clipped away
    ])
    return dict(rho=rho, surr=surr, k3=k3, ell=ell, w=w, coeff=coeff, loss=loss,
                abs_loss=np.abs(ell_w).sum(), metrics=metrics, u=u)


# --------------------------------------------------------------------------- step 9b
def backward(H, W, y, lse, coeff, logit_scale=1.0, chunk_tokens=1024, grad_scale=1.0):
    """p = exp(z - lse);  dz_tv = c_t (1[v = y_t] - p_tv);  dH = s dz W;  dW = s dz^T H.

    ("(softmax - onehot) * coeff" of north_star with coeff = -c_t.)
    """
    H = np.asarray(H, dtype=np.float64)
    W = np.asarray(W, dtype=np.float64)
    y = np.asarray(y, dtype=np.int64)
    c = np.asarray(coeff, dtype=np.float64) * grad_scale
    T, V = H.shape[0], W.shape[0]
    dH = np.zeros_like(H)
    dW = np.zeros_like(W)
    valid = (y >= 0) & (y < V)
    for t0 in range(0, T, chunk_tokens):
        t1 = min(T, t0 + chunk_tokens)
        z = logit_scale * (H[t0:t1] @ W.T)
        p = np.exp(z - np.asarray(lse, dtype=np.float64)[t0:t1, None])
        dz = -p
        rows = np.arange(t1 - t0)[valid[t0:t1]]
        dz[rows, y[t0:t1][valid[t0:t1]]] += 1.0
        dz *= c[t0:t1, None]
        dH[t0:t1] = logit_scale * (dz @ W)
        dW += logit_scale * (dz.T @ H[t0:t1])
    return dH, dW


# ------------------------------------------------------- single outputs, one by one
# For inputs too large to run the whole step in float64 (T x V x d at the Qwen3 shape), the same
# definitions evaluated for a SAMPLE of outputs: a token's (lse, logp), a row of dH, a row of dW.
# Each is the formula of steps 3, 4 and 9 written for one index; nothing is shared with `backward`
# beyond numpy (tests/test_oracle_pins.py checks they reproduce its rows).
def token_rows(H, W, y, rows, logit_scale=1.0):
    """(lse_t, logp_t) for t in ``rows``: the full logit row z_t = s W h_t is materialised."""
    H = np.asarray(H, dtype=np.float64)
    W = np.asarray(W, dtype=np.float64)
    V = W.shape[0]
    lse = np.zeros(len(rows))
    logp = np.zeros(len(rows))
    for i, t in enumerate(rows):
        z = logit_scale * (W @ H[t])
        m = z.max()
        lse[i] = m + np.log(np.exp(z - m).sum())
        yt = int(y[t])
        logp[i] = z[yt] - lse[i] if 0 <= yt < V else 0.0
    return lse, logp


def dH_rows(H, W, y, lse_rows, coeff_rows, rows, logit_scale=1.0):
    """dH[t,:] = s sum_v c_t (1[v = y_t] - p_tv) W[v,:] for t in ``rows`` (lse/coeff given for those t)."""
    H = np.asarray(H, dtype=np.float64)
    W = np.asarray(W, dtype=np.float64)
    V = W.shape[0]
    out = np.zeros((len(rows), H.shape[1]))
    for i, t in enumerate(rows):
        z = logit_scale * (W @ H[t])
        dz = -np.exp(z - lse_rows[i])
        yt = int(y[t])
        if 0 <= yt < V:
            dz[yt] += 1.0
        out[i] = logit_scale * coeff_rows[i] * (dz @ W)
    return out


def dW_rows(H, W, y, lse, coeff, vocab_ids, logit_scale=1.0):
    """dW[v,:] = s sum_t c_t (1[v = y_t] - p_tv) H[t,:] for v in ``vocab_ids`` (lse/coeff for ALL t)."""
    H = np.asarray(H, dtype=np.float64)
    W = np.asarray(W, dtype=np.float64)
    y = np.asarray(y, dtype=np.int64)
    lse = np.asarray(lse, dtype=np.float64)
    c = np.asarray(coeff, dtype=np.float64)
    out = np.zeros((len(vocab_ids), H.shape[1]))
    for i, v in enumerate(vocab_ids):
        z = logit_scale * (H @ W[v])                      # column v of the logits, all tokens
        dz = c * ((y == v).astype(np.float64) - np.exp(z - lse))
        out[i] = logit_scale * (dz @ H)
    return out


# ------------------------------------------------------------- NEXT-4: the final RMSNorm in front of the path
def round_to_bf16(a):
    """float64 -> nearest bfloat16 (round to nearest, ties to even), returned as float64.  bf16 is the top 16
    bits of an fp32; the value is first rounded to fp32 (every bf16 input of interest is far inside its range)."""
    u = np.asarray(a, dtype=np.float32).view(np.uint32).astype(np.uint64)
    u = ((u + 0x7FFF + ((u >> 16) & 1)) >> 16) << 16
    return u.astype(np.uint32).view(np.float32).astype(np.float64)


def rmsnorm_fwd(x, gamma, eps_rms=1e-6, round_bf16=True):
    """Final RMSNorm (the step before the path; BASELINE configs: "hidden ... after
    RMSNorm-like scaling"):  rstd_t = 1 / sqrt(mean_k x_tk^2 + eps_rms);  H_tk = gamma_k x_tk rstd_t.
    The path's contraction consumes H as bf16, so H is rounded to bf16 once (R29); round_bf16=False
    gives the unrounded function (used by the finite-difference pins).  Returns (H [T,d], rstd [T])."""
    x = np.asarray(x, dtype=np.float64)
    g = np.asarray(gamma, dtype=np.float64)
    rstd = 1.0 / np.sqrt((x * x).mean(axis=1) + eps_rms)
    H = g[None, :] * x * rstd[:, None]
    return (round_to_bf16(H) if round_bf16 else H), rstd


def rmsnorm_bwd(x, gamma, rstd, dH):
    """Backward of H = gamma * x * rstd (the bf16 rounding of H passes the gradient through unchanged, R30):
    with xh = x rstd and g = gamma * dH:   dx_t = rstd_t (g_t - xh_t mean_k(g_tk xh_tk));   dgamma = sum_t dH_t * xh_t.
    (mean_k x^2 + eps is differentiated exactly: d rstd / d x_k = - rstd^3 x_k / d.)"""
    x = np.asarray(x, dtype=np.float64)
    gm = np.asarray(gamma, dtype=np.float64)
    dH = np.asarray(dH, dtype=np.float64)
    xh = x * np.asarray(rstd, dtype=np.float64)[:, None]
    g = gm[None, :] * dH
    dx = np.asarray(rstd)[:, None] * (g - xh * (g * xh).mean(axis=1, keepdims=True))
    dgamma = (dH * xh).sum(axis=0)
    return dx, dgamma


def grpo_step_from_prenorm(x, gamma, W, y, cu_seqlens, rewards, old_logp, ref_logp=None, mask=None,
                           cfg: OracleConfig | None = None, G=None, loss_denom=None, eps_rms=1e-6,
                           round_bf16=True, grad_scale=1.0):
    """RMSNorm -> steps 1-9 -> RMSNorm backward: the whole step as a function of the pre-norm activations x and
    the norm weight gamma.  Adds H, rstd, dx, dgamma to grpo_step's outputs."""
    H, rstd = rmsnorm_fwd(x, gamma, eps_rms, round_bf16)
    out = grpo_step(H, W, y, cu_seqlens, rewards, old_logp, ref_logp, mask=mask, cfg=cfg, G=G,
                    loss_denom=loss_denom, grad_scale=grad_scale)
    out["H"], out["rstd"] = H, rstd
    out["dx"], out["dgamma"] = rmsnorm_bwd(x, gamma, rstd, out["dH"])
    return out


# ------------------------------------------------------ NEXT-4: FP8 precision study (R32)
def e4m3_round(y):
    """Nearest value of the 8-bit float format E4M3 (1 sign, 4 exponent bits with bias 7, 3 mantissa bits; no
    infinities; largest finite 448; smallest normal 2^-6; subnormals k 2^-9), round to nearest, ties to even,
    saturating at +-448.  Input: any float array; returns float64 values on the E4M3 grid."""
    y = np.asarray(y, dtype=np.float64)
    a = np.abs(y)
    e = np.floor(np.log2(np.maximum(a, 2.0 ** -6)))          # binade of |y| (>= the smallest normal's)
    step = 2.0 ** (e - 3)                                     # spacing inside that binade: 3 mantissa bits
    q = np.rint(a / step) * step                              # np.rint rounds halves to even
    q = np.minimum(q, 448.0)
    return np.sign(y) * q


def fp8_dequantized_operands(H, W):
    """The operands the FP8 study contracts (cfg.fp8_logits; R32), dequantised back to float64:
    every hidden row t is scaled by s_t = amax_t / 448 (1 for an all-zero row) and rounded to E4M3, the vocab matrix
    by ONE scale amax(W) / 448.  The rounding decision is taken in the kernel's precision (fp32:
    inv = 1 / s, y = x * inv - IEEE single operations, reproduced here with numpy float32), so both sides quantise
    to the same codes; everything after the decision is float64.  Returns (H~ = q s_t, W~ = q s_W)."""
    def quant(x, per_row):
        x32 = np.asarray(x, dtype=np.float32)
        amax = np.abs(x32).max(axis=1, keepdims=True) if per_row else np.abs(x32).max(keepdims=True).reshape(1, 1)
        s = np.where(amax > 0, amax * np.float32(1.0 / 448.0), np.float32(1.0)).astype(np.float32)
        inv = (np.float32(1.0) / s).astype(np.float32)
        q = e4m3_round((x32 * inv).astype(np.float32))
        return q * s.astype(np.float64)
    return quant(H, True), quant(W, False)


# ------------------------------------------------------------------------ whole step
def grpo_step(H, W, y, cu_seqlens, rewards, old_logp, ref_logp=None, mask=None,
              cfg: OracleConfig | None = None, G=None, cu_groups=None, loss_denom=None,
              adv=None, need_grads=True, grad_scale=1.0):
    """Steps 1-9 in order.  ``adv`` may be given directly (skips step 1)."""
    cfg = cfg or OracleConfig()
    H = np.asarray(H, dtype=np.float64)
    W = np.asarray(W, dtype=np.float64)
    y = np.asarray(y, dtype=np.int64)
    V = W.shape[0]
    zero_var = None
    if adv is None:
        adv, zero_var = group_advantage(rewards, cu_groups=cu_groups, G=G,
                                        eps_std=cfg.eps_std, ddof=cfg.std_ddof)
    A_tok = token_advantage(adv, cu_seqlens)
    lse, logp = token_logprobs(H, W, y, cfg.logit_scale, cfg.chunk_tokens)
    valid = (y >= 0) & (y < V)
    lt = loss_terms(logp, old_logp, ref_logp, mask, A_tok, cu_seqlens, cfg,
                    loss_denom=loss_denom, valid=valid)
    out = dict(adv=np.asarray(adv, dtype=np.float64), zero_var=zero_var, lse=lse, logp=logp, **lt)
    if need_grads:
        dH, dW = backward(H, W, y, lse, lt["coeff"], cfg.logit_scale, cfg.chunk_tokens, grad_scale)
        out["dH"], out["dW"] = dH, dW
    return out


def grpo_step_loops(H, W, y, cu_seqlens, rewards, old_logp, ref_logp=None, mask=None,
                    cfg: OracleConfig | None = None, G=None, loss_denom=None):
    """The same definition with explicit Python loops (tiny shapes only).

    Independent of the numpy-vectorised path above except for ``math``: used to check
    ``grpo_step`` against.
    """
    import math
    cfg = cfg or OracleConfig()
    T, d = len(H), len(H[0])
    V = len(W)
    S = len(cu_seqlens) - 1
    n_groups = S // G
    adv = [0.0] * S
    for g in range(n_groups):
        rs = [float(rewards[g * G + i]) for i in range(G)]
        mu = sum(rs) / G
        div = G - cfg.std_ddof
        sigma = math.sqrt(sum((r - mu) ** 2 for r in rs) / div) if div > 0 else 0.0
        for i in range(G):
            adv[g * G + i] = (rs[i] - mu) / (sigma + cfg.eps_std)
    seq_of = [0] * T
    for s in range(S):
        for t in range(cu_seqlens[s], cu_seqlens[s + 1]):
            seq_of[t] = s
    mk = [1.0 if (mask is None or mask[t]) else 0.0 for t in range(T)]
    for t in range(T):
        if y[t] < 0 or y[t] >= V:
            mk[t] = 0.0
    if cfg.loss_agg == 0:
        denom = max(sum(mk), 1.0) if (loss_denom is None or loss_denom <= 0) else float(loss_denom)
        w = [mk[t] / denom for t in range(T)]
    else:
        cnt = [max(sum(mk[cu_seqlens[s]:cu_seqlens[s + 1]]), 1.0) for s in range(S)]
        w = [mk[t] / (cnt[seq_of[t]] * S) for t in range(T)]
    logp = [0.0] * T
    lse = [0.0] * T
    z = [[cfg.logit_scale * sum(float(W[v][k]) * float(H[t][k]) for k in range(d))
          for v in range(V)] for t in range(T)]
    loss = 0.0
    coeff = [0.0] * T
    lo, hi = 1.0 - cfg.clip_lo, 1.0 + cfg.clip_hi
    for t in range(T):
        mx = max(z[t])
        lse[t] = mx + math.log(sum(math.exp(zv - mx) for zv in z[t]))
        if mk[t] == 0.0 and (y[t] < 0 or y[t] >= V):
            continue
        logp[t] = z[t][y[t]] - lse[t]
        A = adv[seq_of[t]]
        rho = math.exp(logp[t] - float(old_logp[t]))
        surr = min(rho * A, min(max(rho, lo), hi) * A)
        k3 = dk3 = 0.0
        if cfg.kl_beta != 0.0 and ref_logp is not None:
            delta = float(ref_logp[t]) - logp[t]
            if cfg.kl_type == 1:
                k3, dk3 = -delta, 1.0
            elif cfg.kl_type == 2:
                k3, dk3 = 0.5 * delta * delta, -delta
            else:
                k3 = math.exp(delta) - delta - 1.0
                dk3 = 1.0 - math.exp(delta)
        clipped = (A > 0 and rho > hi) or (A < 0 and rho < lo)
        if cfg.dual_clip > 0.0 and A < 0:
            surr = max(surr, cfg.dual_clip * A)
            clipped = clipped or rho > cfg.dual_clip
        if w[t] != 0.0:
            loss += w[t] * (-surr + cfg.kl_beta * k3)
            coeff[t] = w[t] * (-A * rho * (0.0 if clipped else 1.0) + cfg.kl_beta * dk3)
    dH = [[0.0] * d for _ in range(T)]
    dW = [[0.0] * d for _ in range(V)]
    for t in range(T):
        if coeff[t] == 0.0:
            continue
        for v in range(V):
            dz = coeff[t] * ((1.0 if v == y[t] else 0.0) - math.exp(z[t][v] - lse[t]))
            for k in range(d):
                dH[t][k] += cfg.logit_scale * dz * float(W[v][k])
                dW[v][k] += cfg.logit_scale * dz * float(H[t][k])
    return dict(adv=np.array(adv), lse=np.array(lse), logp=np.array(logp), loss=loss,
                coeff=np.array(coeff), dH=np.array(dH), dW=np.array(dW))
