"""Vocab-parallel (tensor-parallel) forward / backward (the paper's trainer ran TP = 4,
PAPER.md:197), emulated on ONE GPU: the vocab matrix is cut into row shards, each "rank" (its own context, V = its
shard) produces per-token (max, sum-exp, target-logit) partials, the gathered partials go through
grpo_loss_from_partials, and every rank runs the backward on its shard with shard-local targets and the global
lse / coeff.  Concatenated dW shards and the SUM of the partial dHidden must match the float64 oracle of the
unsharded step within north_star's tolerances, and the unsharded CUDA path to fp32 noise.  The exchange itself (ONE
all-gather of [3, T] floats and ONE all-reduce of [T, d]) is `dp.py::GrpoVocabParallel`:
`test_two_tp_ranks_run_the_exchange` runs its `step` in two processes on cuda:0 (gloo, as NCCL refuses two ranks on
one device) against the oracle of the unsharded step; a one-rank NCCL group runs the NCCL calls
(tests/test_dp_gpu.py)."""
import os
import socket
import sys

import torch.distributed as dist
import torch.multiprocessing as mp
import numpy as np
import pytest
import torch

from tests.parity_util import (TOL_GRAD_REL, TOL_LOGP_ABS, TOL_LOSS_REL, make_ctx, rel_l2, run_cuda, run_oracle, to64)
from workloads.synth import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2606_26997_b200.build import build
    build()


def _tp_step(b, bounds, **ctx_kw):
    from paper_2606_26997_b200 import GrpoContext
    n = len(bounds) - 1
    kw = dict(eps_std=b.eps_std, clip_lo=b.clip_lo, clip_hi=b.clip_hi, kl_beta=b.kl_beta, loss_agg=b.loss_agg,
              group_size=b.G, dhidden_fp32=1, bwd_chunk_tokens=1024)
    kw.update(ctx_kw)
    ranks = [GrpoContext(b.d, bounds[r + 1] - bounds[r], max_tokens=b.T, **kw) for r in range(n)]
    shards = [b.W[bounds[r]:bounds[r + 1]].contiguous() for r in range(n)]
    y_loc = [(b.targets - bounds[r]).contiguous() for r in range(n)]
    for r in range(n):                                  # ignored tokens (y < 0) stay ignored in every shard
        y_loc[r] = torch.where(b.targets < 0, torch.full_like(b.targets, -1), y_loc[r])
    parts = [ranks[r].grpo_vocab_shard_partials(b.hidden, shards[r], y_loc[r]) for r in range(n)]
    m2, s2, zy = (torch.stack([p[i] for p in parts]).contiguous() for i in range(3))     # the "all-gather"
    adv = ranks[0].grpo_group_advantage(b.rewards, G=b.G)
    metrics = torch.zeros(4, dtype=torch.float32, device="cuda")
    f = ranks[0].grpo_loss_from_partials(m2, s2, zy, b.targets, b.V, b.cu_seqlens, adv, b.old_logp, b.ref_logp, b.mask,
                                         metrics_accum=metrics)
    dW = torch.zeros(b.V, b.d, dtype=torch.float32, device="cuda")
    dH = torch.zeros(b.T, b.d, dtype=torch.float32, device="cuda")
    for r in range(n):
        dW_r = torch.zeros(bounds[r + 1] - bounds[r], b.d, dtype=torch.float32, device="cuda")
        dH_r = ranks[r].grpo_fused_logprob_loss_bwd(b.hidden, shards[r], y_loc[r], f["lse"], f["coeff"], dW_accum=dW_r)
        dW[bounds[r]:bounds[r + 1]] = dW_r
        dH += dH_r                                                                        # the "all-reduce"
    torch.cuda.synchronize()
    for c in ranks:
        assert c.grpo_check_errors_sync() == 0
        c.close()
    return dict(dW=dW, dH=dH, metrics=metrics, **f)


@pytest.mark.parametrize("bounds,kw", [
    ([0, 1024, 2048, 3000], dict()),
    ([0, 1504, 3000], dict(mask_frac=0.2, bad_target_frac=0.1)),
    ([0, 256, 264, 2000, 3000], dict(loss_agg=1)),
])
def test_sharded_vocab_equals_the_unsharded_step(bounds, kw):
    b = make_config(1, device="cuda", seed=8, variant="1b", n_groups=4, G=4, d=128, V=3000, len_div=0.2, w_std=0.1, **kw)
    out = _tp_step(b, bounds)
    ref = run_oracle(b)
    assert np.abs(to64(out["logp"]) - ref["logp"]).max() <= TOL_LOGP_ABS
    assert np.abs(to64(out["lse"]) - ref["lse"]).max() <= TOL_LOGP_ABS
    assert abs(out["loss"].item() - ref["loss"]) <= TOL_LOSS_REL * max(abs(ref["loss"]), ref["abs_loss"])
    assert rel_l2(to64(out["coeff"]), ref["coeff"]) <= 1e-3
    assert rel_l2(to64(out["dH"]), ref["dH"]) <= TOL_GRAD_REL
    assert rel_l2(to64(out["dW"]), ref["dW"]) <= TOL_GRAD_REL
    np.testing.assert_allclose(to64(out["metrics"]), ref["metrics"], rtol=1e-4, atol=1e-3)
    # and against the unsharded CUDA path: same arithmetic up to where the vocab range is cut
    ctx = make_ctx(b, max_tokens=b.T, dhidden_fp32=1, bwd_chunk_tokens=1024)
    full = run_cuda(ctx, b)
    ctx.close()
    assert (out["logp"] - full["logp"]).abs().max().item() <= 2e-5
    assert rel_l2(to64(out["dH"]), to64(full["dH"])) <= 2e-3 and rel_l2(to64(out["dW"]), to64(full["dW"])) <= 2e-3
    assert to64(out["metrics"])[3] == to64(full["metrics"])[3]


ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _tp_batch():
    return make_config(1, device="cuda", seed=11, variant="1b", n_groups=4, G=4, d=128, V=3000, len_div=0.2, w_std=0.1,
                       mask_frac=0.2, bad_target_frac=0.1, kl_beta=0.02)


def _tp_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2606_26997_b200.dp import GrpoVocabParallel
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    b = _tp_batch()                                                     # replicated batch, as the TP body leaves it
    vp = GrpoVocabParallel(b.d, b.V, max_tokens=b.T, eps_std=b.eps_std, clip_lo=b.clip_lo, clip_hi=b.clip_hi,
                           kl_beta=b.kl_beta, loss_agg=b.loss_agg, group_size=b.G, bwd_chunk_tokens=1024)
    W_shard = vp.shard_rows(b.W)
    dW_shard = torch.zeros(vp.v1 - vp.v0, b.d, dtype=torch.float32, device="cuda")
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")
    metrics = torch.zeros(4, dtype=torch.float32, device="cuda")
    f = vp.step(b.hidden, W_shard, b.targets, b.cu_seqlens, b.rewards, b.G, b.old_logp, b.ref_logp, b.mask,
                dW_shard_accum=dW_shard, loss_accum=loss, metrics_accum=metrics)
    torch.cuda.synchronize()
    assert vp.ctx.grpo_check_errors_sync() == 0
    q.put((rank, vp.v0, vp.v1, dW_shard.cpu().numpy(), f["dH"].cpu().numpy(), f["logp"].cpu().numpy(),
           f["coeff"].cpu().numpy(), float(loss.item()), metrics.cpu().numpy()))
    vp.close()
    dist.barrier()
    dist.destroy_process_group()


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_tp_ranks_run_the_exchange():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_tp_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=600) for _ in range(world)), key=lambda r: r[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    b = _tp_batch()
    ref = run_oracle(b)
    assert [(r[1], r[2]) for r in res] == [(0, 1496), (1496, 3000)]
    dW = np.concatenate([r[3] for r in res])                            # dW stays sharded by rows
    assert rel_l2(dW, ref["dW"]) <= TOL_GRAD_REL
    for rank, v0, v1, dW_r, dH, logp, coeff, loss, metrics in res:
        assert rel_l2(dW_r, ref["dW"][v0:v1]) <= TOL_GRAD_REL
        assert rel_l2(dH, ref["dH"]) <= TOL_GRAD_REL                    # the all-reduced, full dHidden
        assert np.abs(logp - ref["logp"]).max() <= TOL_LOGP_ABS
        assert rel_l2(coeff, ref["coeff"]) <= 1e-3
        assert abs(loss - ref["loss"]) <= TOL_LOSS_REL * max(abs(ref["loss"]), ref["abs_loss"])   # replicated, not summed
        np.testing.assert_allclose(metrics, ref["metrics"], rtol=1e-4, atol=1e-3)
    for k in (4, 5, 6, 8):                                              # every rank ends with the same bits
        np.testing.assert_array_equal(res[0][k], res[1][k])
    assert res[0][7] == res[1][7]
