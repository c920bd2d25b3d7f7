"""Data parallelism over complete groups with the REAL kernels: two ranks, both on
cuda:0 (one GPU is all this build can reach; NCCL refuses two ranks on one device, so the ranks reduce through
gloo), each trains the groups `GrpoDataParallel` deals it through grpo_enqueue_groups with the denominator of the
whole update; after ONE sum all-reduce of dW / loss at the update boundary every rank must hold the single-rank
full-batch gradient (P12) - compared with rank 0's own full-batch run and with the float64 oracle.  The ranks'
kernels never wait on one another."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _batch():
    from workloads.synth import make_config
    return make_config(5, device="cuda", d=128, V=3000, n_groups=6, len_div=25.0, w_std=0.08, old_sigma=0.3,
                       kl_beta=0.002)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2606_26997_b200.dp import GrpoDataParallel
    from tests.parity_util import make_ctx, run_cuda
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dp = GrpoDataParallel()
    b = _batch()
    order = [int(g) for g in b.arrival_order]                          # FIFO order of the update's 6 groups
    mine = [order[k] for k in dp.local_positions(len(order))]
    toks = {g: int(b.seqlens[g * b.G:(g + 1) * b.G].sum()) for g in order}
    denom = dp.global_denominator(sum(toks[g] for g in mine))
    assert denom == b.T
    ctx = make_ctx(b, groups_per_update=len(mine), max_tokens=sum(toks[g] for g in mine), bwd_chunk_tokens=1024)
    dW, loss, metrics = dp.buffers(b.V, b.d)
    dH = torch.zeros(b.T, b.d, dtype=torch.bfloat16, device="cuda")
    descs = []
    for g in mine:
        t0, t1 = b.group_token_range(g)
        descs.append(ctx.make_group_desc(g, b.seqlens[g * b.G:(g + 1) * b.G], b.hidden[t0:t1], b.targets[t0:t1],
                                         b.old_logp[t0:t1], b.rewards[g * b.G:(g + 1) * b.G].contiguous(),
                                         b.ref_logp[t0:t1], None, dH[t0:t1], None))
    consumed, boundary = ctx.grpo_enqueue_groups(descs, b.W, dW, loss, metrics, loss_denom=denom)
    assert boundary and consumed == len(mine)
    # the boundary reduction: through gloo, so on host copies (NCCL + NVLink on a multi-GPU box: same call)
    torch.cuda.synchronize()
    dW_h, loss_h, met_h = dW.cpu(), loss.cpu(), metrics.cpu()
    dp.reduce_boundary(dW_h, loss_h, met_h).wait()
    full = None
    if rank == 0:                                                      # the single-rank full-batch step
        ctx2 = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=1024)
        f = run_cuda(ctx2, b, loss_denom=float(b.T))
        ctx2.close()
        full = (f["dW"].cpu().numpy(), float(f["loss"].item()), f["dH"].float().cpu().numpy())
    rows = torch.cat([torch.arange(*b.group_token_range(g)) for g in mine])
    q.put((rank, dW_h.numpy(), float(loss_h), met_h.numpy(), rows.numpy(), dH[rows.cuda()].float().cpu().numpy(), full))
    ctx.close()
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_sum_to_the_full_batch_step():
    from tests.parity_util import TOL_GRAD_REL, TOL_LOSS_REL, rel_l2, run_oracle
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=600) for _ in range(world)), key=lambda r: r[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    full_dW, full_loss, full_dH = res[0][6]
    b = _batch()
    ref = run_oracle(b, loss_denom=float(b.T))
    for rank, dW, loss, met, rows, dH_rows, _ in res:
        assert rel_l2(dW, full_dW) <= 1e-5                              # sum over ranks == full batch
        np.testing.assert_allclose(loss, full_loss, rtol=1e-5)
        assert rel_l2(dW, ref["dW"]) <= TOL_GRAD_REL
        assert abs(loss - ref["loss"]) <= TOL_LOSS_REL * max(abs(ref["loss"]), ref["abs_loss"])
        assert met[0] == b.T
        np.testing.assert_array_equal(dH_rows, full_dH[rows])          # batch invariance: same bits as the full batch
    np.testing.assert_array_equal(res[0][1], res[1][1])
