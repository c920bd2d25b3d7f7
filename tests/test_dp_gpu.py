"""Data parallelism over complete groups with the REAL kernels: two ranks, both on
cuda:0 (one GPU is all this build can reach; NCCL refuses two ranks on one device, so the ranks reduce through
gloo), each trains the groups `GrpoDataParallel` deals it through grpo_enqueue_groups with the denominator of the
whole update (token count for loss_agg 0; sequence count through grpo_set_seq_denom for loss_agg 1); after ONE sum
all-reduce of dW / loss at the update boundary every rank must hold the single-rank full-batch gradient (P12) -
compared with rank 0's own full-batch run and with the float64 oracle.  The reduction runs on the CUDA tensors
themselves (gloo stages them through the host), so `reduce_boundary`'s side stream, event wait and `done_event` and
`BoundaryHandle.wait(stream)` execute; the update is trained twice, back to back, into the two alternating buffer
sets of `buffers()` with the first reduction still outstanding.  The ranks' kernels never wait on one another."""
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


def _batch(loss_agg=0):
    from workloads.synth import make_config
    return make_config(5, device="cuda", d=128, V=3000, n_groups=6, len_div=25.0, w_std=0.08, old_sigma=0.3,
                       kl_beta=0.002, loss_agg=loss_agg)


def _worker(rank, world, port, q, loss_agg):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2606_26997_b200.dp import GrpoDataParallel
    from tests.parity_util import make_ctx, run_cuda
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dp = GrpoDataParallel()
    b = _batch(loss_agg)
    order = [int(g) for g in b.arrival_order]                          # FIFO order of the update's 6 groups
    mine = [order[k] for k in dp.local_positions(len(order))]
    toks = {g: int(b.seqlens[g * b.G:(g + 1) * b.G].sum()) for g in order}
    denom = dp.global_denominator(sum(toks[g] for g in mine))
    assert denom == b.T
    ctx = make_ctx(b, groups_per_update=len(mine), max_tokens=sum(toks[g] for g in mine), bwd_chunk_tokens=1024)
    if loss_agg == 1:                                                  # per-sequence mean over the WHOLE update
        S_all = dp.global_sequences(len(mine) * b.G)
        assert S_all == b.S
        ctx.grpo_set_seq_denom(S_all)
    dH = torch.zeros(b.T, b.d, dtype=torch.bfloat16, device="cuda")
    descs = lambda: [ctx.make_group_desc(g, b.seqlens[g * b.G:(g + 1) * b.G], b.hidden[slice(*b.group_token_range(g))],
                                         b.targets[slice(*b.group_token_range(g))],
                                         b.old_logp[slice(*b.group_token_range(g))],
                                         b.rewards[g * b.G:(g + 1) * b.G].contiguous(),
                                         b.ref_logp[slice(*b.group_token_range(g))], None,
                                         dH[slice(*b.group_token_range(g))], None) for g in mine]
    compute = torch.cuda.current_stream()
    sets, handles = [], []
    for it in range(2):                                                # two updates, alternating accumulator sets
        dW, loss, metrics = dp.buffers(b.V, b.d)
        assert not sets or dW.data_ptr() != sets[0][0].data_ptr()
        consumed, boundary = ctx.grpo_enqueue_groups(descs(), b.W, dW, loss, metrics, loss_denom=denom)
        assert boundary and consumed == (it + 1) * len(mine)
        # the boundary reduction on the device tensors: enqueued behind the update's launches on the side stream,
        # returns at once (NCCL + NVLink on a multi-GPU box: the same call)
        handles.append(dp.reduce_boundary(dW, loss, metrics, compute_stream=compute))
        assert handles[-1].done_event is not None
        sets.append((dW, loss, metrics))
    for h in handles:
        h.wait(compute)
    torch.cuda.synchronize()
    for k in range(3):
        assert torch.equal(sets[0][k], sets[1][k])                     # the same update, reduced twice: same bits
    dW_h, loss_h, met_h = (t.cpu() for t in sets[0])
    full = None
    if rank == 0:                                                      # the single-rank full-batch step
        ctx2 = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=1024)
        f = run_cuda(ctx2, b, loss_denom=float(b.T) if loss_agg == 0 else 0.0)
        ctx2.close()
        full = (f["dW"].cpu().numpy(), float(f["loss"].item()), f["dH"].float().cpu().numpy())
    rows = torch.cat([torch.arange(*b.group_token_range(g)) for g in mine])
    q.put((rank, dW_h.numpy(), float(loss_h), met_h.numpy(), rows.numpy(), dH[rows.cuda()].float().cpu().numpy(), full))
    ctx.close()
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("loss_agg", [0, 1])
def test_two_ranks_sum_to_the_full_batch_step(loss_agg):
    from tests.parity_util import TOL_GRAD_REL, TOL_LOSS_REL, rel_l2, run_oracle
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q, loss_agg)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=600) for _ in range(world)), key=lambda r: r[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    full_dW, full_loss, full_dH = res[0][6]
    b = _batch(loss_agg)
    ref = run_oracle(b, loss_denom=float(b.T) if loss_agg == 0 else None)
    for rank, dW, loss, met, rows, dH_rows, _ in res:
        assert rel_l2(dW, full_dW) <= 1e-5                              # sum over ranks == full batch
        np.testing.assert_allclose(loss, full_loss, rtol=1e-5)
        assert rel_l2(dW, ref["dW"]) <= TOL_GRAD_REL
        assert abs(loss - ref["loss"]) <= TOL_LOSS_REL * max(abs(ref["loss"]), ref["abs_loss"])
        assert met[0] == b.T
        np.testing.assert_array_equal(dH_rows, full_dH[rows])          # batch invariance: same bits as the full batch
    np.testing.assert_array_equal(res[0][1], res[1][1])


def _nccl_worker(port, q):
    """A one-rank NCCL group on cuda:0: every CUDA / NCCL branch of dp.py runs (the collectives are identities)."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1")
    sys.path.insert(0, ROOT)
    from paper_2606_26997_b200.dp import GrpoDataParallel, StitchedGradient
    from tests.parity_util import make_ctx, run_cuda
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda:0"))
    dp = GrpoDataParallel(always_reduce=True)
    assert dist.get_backend() == "nccl" and dp.world == 1
    b = _batch(1)
    assert dp.global_denominator(b.T) == float(b.T)                     # .cuda() + NCCL all-reduce of a float64 scalar
    assert dp.global_sequences(b.S) == b.S
    ctx = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=1024)
    ref = run_cuda(ctx, b)                                              # plain accumulators, no reduction
    compute = torch.cuda.current_stream()
    outs = []
    for it in range(2):                                                 # alternating sets, reductions left in flight
        dW, loss, metrics = dp.buffers(b.V, b.d)
        adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
        f = ctx.grpo_fused_logprob_loss_fwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp, b.mask,
                                            loss_accum=loss, metrics_accum=metrics)
        ctx.grpo_fused_logprob_loss_bwd(b.hidden, b.W, b.targets, f["lse"], f["coeff"], dW_accum=dW, want_dhidden=False)
        h = dp.reduce_boundary(dW, loss, metrics, compute_stream=compute)      # side stream, event wait, NCCL
        assert h.done_event is not None and not h.works
        outs.append((dW, loss, metrics, h))
    side = torch.cuda.Stream()
    for dW, loss, metrics, h in outs:
        h.wait(side)                                                    # a consumer stream waits on done_event
    side.synchronize()
    ok = all(torch.equal(o[0], ref["dW"]) and torch.equal(o[1], ref["loss"]) and torch.equal(o[2], ref["metrics"])
             for o in outs)
    # the stitched accumulator through its dp path (export, descriptor exchange of a one-rank group, map)
    sg = StitchedGradient(ctx, b.V, b.d, dp)
    adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
    f = ctx.grpo_fused_logprob_loss_fwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp, b.mask)
    ctx.grpo_fused_logprob_loss_bwd(b.hidden, b.W, b.targets, f["lse"], f["coeff"], dW_accum=sg.full, want_dhidden=False)
    sg.barrier()
    ok_sg = torch.equal(sg.full, ref["dW"]) and sg.local_rows == (0, b.V)
    sg.close()
    ctx.close()
    # the vocab-parallel exchange on NCCL: all_gather_into_tensor of the [3, T] partials, all-reduce of dHidden
    from paper_2606_26997_b200.dp import GrpoVocabParallel
    vp = GrpoVocabParallel(b.d, b.V, always_reduce=True, max_tokens=b.T, eps_std=b.eps_std, clip_lo=b.clip_lo,
                           clip_hi=b.clip_hi, kl_beta=b.kl_beta, loss_agg=b.loss_agg, group_size=b.G,
                           bwd_chunk_tokens=1024)
    dW_vp = torch.zeros(b.V, b.d, dtype=torch.float32, device="cuda")
    g = vp.step(b.hidden, vp.shard_rows(b.W), b.targets, b.cu_seqlens, b.rewards, b.G, b.old_logp, b.ref_logp, b.mask,
                dW_shard_accum=dW_vp)
    torch.cuda.synchronize()
    ok_vp = (vp.v0, vp.v1) == (0, b.V) and (g["logp"] - ref["logp"]).abs().max().item() <= 2e-5 and \
        ((dW_vp - ref["dW"]).norm() / ref["dW"].norm()).item() <= 2e-3
    vp.close()
    ok_sg = ok_sg and ok_vp
    q.put((ok, ok_sg))
    dist.destroy_process_group()


def test_nccl_and_cuda_branches_run_in_a_one_rank_group():
    """NCCL refuses two ranks on one GPU but accepts a group of one: with `always_reduce` the data-parallel boundary
    runs its real code path - `.cuda()` scalars, side-stream all-reduce behind an event, `done_event`, consumer-stream
    wait, alternating buffers, StitchedGradient's export / exchange / map - and must leave the gradients unchanged."""
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    p = ctx.Process(target=_nccl_worker, args=(port, q))
    p.start()
    ok, ok_sg = q.get(timeout=600)
    p.join(timeout=120)
    assert p.exitcode == 0
    assert ok and ok_sg
