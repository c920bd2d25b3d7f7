"""Helpers shared by the GPU parity tests: run the CUDA path through the C ABI, run the oracle on the
same bits, and compute the gates of BASELINE.json north_star plus the sub-block gates of SURVEY §8(c)."""
import numpy as np
import torch

from oracle.grpo_oracle import OracleConfig, grpo_step, round_to_bf16

TOL_LOGP_ABS = 2e-3      # per-token log-prob abs err (north_star)
TOL_LOSS_REL = 1e-3      # loss rel err, relative to max(|loss|, sum |w l|) (R21)
TOL_GRAD_REL = 1e-2      # dHidden / dW rel L2 (north_star)


def oracle_cfg(b, **kw):
    return OracleConfig(eps_std=b.eps_std, clip_lo=b.clip_lo, clip_hi=b.clip_hi, kl_beta=b.kl_beta,
                        loss_agg=b.loss_agg, **kw)


def run_oracle(b, loss_denom=None, std_ddof=0, logit_scale=1.0, need_grads=True, chunk=1024, kl_type=0,
               dual_clip=0.0):
    x = b.numpy_f64()
    cfg = oracle_cfg(b, std_ddof=std_ddof, logit_scale=logit_scale, chunk_tokens=chunk, kl_type=kl_type,
                     dual_clip=dual_clip)
    return grpo_step(x["H"], x["W"], x["y"], x["cu_seqlens"], x["rewards"], x["old_logp"], x["ref_logp"],
                     mask=x["mask"], cfg=cfg, G=b.G, loss_denom=loss_denom, need_grads=need_grads)


def make_ctx(b, **kw):
    from paper_2606_26997_b200 import GrpoContext
    args = dict(eps_std=b.eps_std, clip_lo=b.clip_lo, clip_hi=b.clip_hi, kl_beta=b.kl_beta, loss_agg=b.loss_agg,
                group_size=b.G)
    args.update(kw)
    return GrpoContext(b.d, b.V, **args)


def run_cuda(ctx, b, loss_denom=0.0, want_dw=True, want_dh=True, grad_scale=1.0, fused=False):
    """fused=False: grpo_fused_logprob_loss_fwd then _bwd (north_star: logits recomputed in the backward);
    fused=True: grpo_fused_logprob_loss_fwd_bwd (3-contraction variant, logits stashed per chunk)."""
    dev = b.hidden.device
    adv, zv = ctx.grpo_group_advantage(b.rewards, G=b.G, want_zero_var=True)
    metrics = torch.zeros(4, dtype=torch.float32, device=dev)
    dW = torch.zeros(b.V, b.d, dtype=torch.float32, device=dev) if want_dw else None
    if fused:
        f = ctx.grpo_fused_logprob_loss_fwd_bwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp,
                                                b.mask, loss_denom=loss_denom, grad_scale=grad_scale,
                                                metrics_accum=metrics, dW_accum=dW, want_dhidden=want_dh)
        dH = f.pop("dH")
    else:
        f = ctx.grpo_fused_logprob_loss_fwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp,
                                            b.mask, loss_denom=loss_denom, metrics_accum=metrics)
        dH = ctx.grpo_fused_logprob_loss_bwd(b.hidden, b.W, b.targets, f["lse"], f["coeff"], dW_accum=dW,
                                             grad_scale=grad_scale, want_dhidden=want_dh)
    torch.cuda.synchronize()
    return dict(adv=adv, zero_var=zv, metrics=metrics, dW=dW, dH=dH, **f)


def rel_l2(a, r):
    a = np.asarray(a, dtype=np.float64)
    r = np.asarray(r, dtype=np.float64)
    return float(np.linalg.norm(a - r) / max(np.linalg.norm(r), 1e-300))


def to64(t):
    return t.detach().double().cpu().numpy()


bf16_round = round_to_bf16      # float64 -> nearest bf16 (ties to even) as float64: the oracle's, pinned against torch


def _bf16_neighbours(x):
    """(nearest, next below, next above) bf16 values of x, as float64."""
    r = bf16_round(x)
    bits = r.astype(np.float32).view(np.uint32).astype(np.int64)
    mag = bits & 0x7FFFFFFF
    sign = bits & 0x80000000
    def mk(m):
        return (sign | np.clip(m, 0, 0x7F7F0000)).astype(np.uint32).view(np.float32).astype(np.float64)
    return r, mk(mag - 0x10000), mk(mag + 0x10000)


def _dense_part_rel(dH, dense_ref, entry, Wy):
    """rel-L2 of (dH - e W[y]) against dense_ref, with e per row the bf16 neighbour of `entry` that fits best."""
    best = None
    for cand in _bf16_neighbours(entry):
        r2 = (((dH - cand[:, None] * Wy) - dense_ref) ** 2).sum(1)
        best = r2 if best is None else np.minimum(best, r2)
    return float(np.sqrt(best.sum()) / np.linalg.norm(dense_ref))


def worst_block_rel(a, r, block=(32, 32)):
    """max over blocks of ||a - r||_F / max(||r||_F of the block, 1e-2 x the median block norm): a single wrong
    tile cannot hide in the Frobenius norm of the whole matrix.  Blocks where r is exactly zero must be exactly
    zero in a (returns inf otherwise)."""
    a = np.asarray(a, dtype=np.float64)
    r = np.asarray(r, dtype=np.float64)
    bm, bn = block
    M, N = r.shape
    pm, pn = (-M) % bm, (-N) % bn
    pad = lambda x: np.pad(x, ((0, pm), (0, pn)))
    blk = lambda x: np.sqrt((pad(x) ** 2).reshape((M + pm) // bm, bm, (N + pn) // bn, bn).sum(axis=(1, 3)))
    err, ref = blk(a - r), blk(r)
    nz = ref > 0
    if not nz.any():
        return float(err.max())
    if (err[~nz] != 0).any():
        return float("inf")
    floor = 1e-2 * np.median(ref[nz])
    return float((err[nz] / np.maximum(ref[nz], floor)).max())


def gates(b, out, ref, check_grads=True, logit_scale=1.0, grad_scale=1.0):
    """Return dict of errors; caller asserts against the TOL_* constants."""
    e = {}
    e["adv_abs"] = float(np.abs(to64(out["adv"]) - ref["adv"]).max())
    e["logp_abs"] = float(np.abs(to64(out["logp"]) - ref["logp"]).max())
    e["lse_abs"] = float(np.abs(to64(out["lse"]) - ref["lse"]).max())
    e["loss_rel"] = abs(out["loss"].item() - ref["loss"]) / max(abs(ref["loss"]), ref["abs_loss"], 1e-300)
    cn = np.linalg.norm(ref["coeff"])
    e["coeff_rel"] = rel_l2(to64(out["coeff"]), ref["coeff"]) if cn > 0 else float(np.abs(to64(out["coeff"])).max())
    if check_grads:
        dH, dW = to64(out["dH"]), to64(out["dW"])
        e["dH_rel"] = rel_l2(dH, ref["dH"]) if np.linalg.norm(ref["dH"]) > 0 else float(np.abs(dH).max())
        e["dW_rel"] = rel_l2(dW, ref["dW"]) if np.linalg.norm(ref["dW"]) > 0 else float(np.abs(dW).max())
        # worst 32 x 32 block of dW (one epilogue warp's TMA reduce box) and worst row of dH (one epilogue thread)
        e["dW_block_rel"] = worst_block_rel(dW, ref["dW"], (32, 32))
        e["dH_row_rel"] = worst_block_rel(dH, ref["dH"], (1, dH.shape[1]))
        # (i) rows of dW for vocab ids that never appear as a target: the dense softmax term alone
        y = b.targets.cpu().numpy()
        non_target = np.ones(b.V, dtype=bool)
        non_target[y[(y >= 0) & (y < b.V)]] = False
        if non_target.any() and np.linalg.norm(ref["dW"][non_target]) > 0:
            e["dW_nontarget_rel"] = rel_l2(dW[non_target], ref["dW"][non_target])
        # (ii) SURVEY.md §8(c): rel-L2 <= 1e-2 on the dense part of dH, sum_{v != y} (-c_t p_tv) s W[v,:], with the
        # target column's contribution removed.  The kernel rounds every dZ entry to bf16 before the dH
        # contraction, and the target entry c_t s (1 - p_ty) is ~50x larger than the rest of the row together, so
        # what is removed is that entry AS THE KERNEL HOLDS IT: bf16(c_t s g (1 - p_ty)) W[y_t].  Its fp32 value can
        # sit on a bf16 rounding boundary, so per row the candidate among {nearest, +-1 bf16 ulp} that leaves the
        # smallest residual is taken (one known entry, one ulp).  fp32 dH output only (a bf16 dH rounds the whole
        # row, one-hot part included, to 2^-9).
        if out["dH"].dtype == torch.float32:
            W64 = b.W.double().cpu().numpy()
            ok = (y >= 0) & (y < b.V)
            yy = np.clip(y, 0, b.V - 1)
            p_y = np.where(ok, np.exp(ref["logp"]), 0.0)
            # float64 value of the dZ target entry (R24: logit_scale and grad_scale are folded into dZ;
            # ref["dH"] is already multiplied by grad_scale by the caller)
            entry = ref["coeff"] * ok * logit_scale * grad_scale * (1.0 - p_y)
            dense_ref = ref["dH"] - entry[:, None] * W64[yy]                  # sum over v != y of dz_tv W[v,:]
            if np.linalg.norm(dense_ref) > 0:
                e["dH_dense_rel"] = _dense_part_rel(dH, dense_ref, entry, W64[yy])
        # (iii) rows of dZ sum to zero => sum_v dW[v,:] = 0 (P7); scale: bf16 rounding of dZ entries
        e["dW_colsum_rel"] = float(np.linalg.norm(dW.sum(0)) / max(np.linalg.norm(dW), 1e-300))
    return e


def assert_gates(e, check_grads=True):
    assert e["adv_abs"] <= 1e-5, e
    assert e["logp_abs"] <= TOL_LOGP_ABS, e
    assert e["loss_rel"] <= TOL_LOSS_REL, e
    assert e["coeff_rel"] <= 1e-3, e
    if check_grads:
        assert e["dH_rel"] <= TOL_GRAD_REL, e
        assert e["dW_rel"] <= TOL_GRAD_REL, e
        if "dW_nontarget_rel" in e:
            assert e["dW_nontarget_rel"] <= TOL_GRAD_REL, e
        if "dH_dense_rel" in e:
            assert e["dH_dense_rel"] <= TOL_GRAD_REL, e
        assert e["dW_block_rel"] <= 2 * TOL_GRAD_REL, e
        assert e["dH_row_rel"] <= 2 * TOL_GRAD_REL, e
