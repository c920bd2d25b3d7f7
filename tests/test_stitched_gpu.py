"""NEXT-3: the dW accumulator stitched from per-rank shards with CUDA virtual memory management
(include/grpo.h grpo_shard_* / grpo_stitch_*; paper_2606_26997_b200/dp.py StitchedGradient), which turns the A6
epilogue's TMA reduce-adds into the data-parallel reduce-scatter.

One GPU is reachable, so: (1) one process stitches three chunks of its own GPU and runs the ordinary backward into the
stitched range - the contraction kernel, unchanged, must produce the same dW as into a plain buffer, across the
chunk boundaries; (2) two processes on cuda:0 each own one chunk, exchange the descriptors over Unix sockets, map
both, and accumulate their groups' gradients into the shared range CONCURRENTLY: after a barrier each rank's own
rows must hold the full-batch gradient (the reduce-scatter happened inside the GEMMs).  Over NVLink the only
difference is where the chunks physically live.  The ranks' kernels never wait on one another."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2606_26997_b200.build import build
    build()


def _batch():
    from workloads.synth import make_config
    # d = 2048: one 2 MiB allocation granule is 256 fp32 rows, so V = 3000 spans several shards
    return make_config(5, device="cuda", d=2048, V=3000, n_groups=4, len_div=60.0, w_std=0.02, old_sigma=0.3,
                       kl_beta=0.002)


def test_backward_into_a_range_stitched_from_three_chunks():
    from paper_2606_26997_b200.dp import StitchedGradient
    from tests.parity_util import TOL_GRAD_REL, make_ctx, rel_l2, run_cuda, run_oracle, to64
    b = _batch()
    ctx = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=512)
    plain = run_cuda(ctx, b)
    sg = StitchedGradient(ctx, b.V, b.d, n_local_shards=3)
    assert sg.rows_per_shard == 1024 and sg.full.shape == (b.V, b.d) and sg.full.is_contiguous()
    adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
    f = ctx.grpo_fused_logprob_loss_fwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp)
    ctx.grpo_fused_logprob_loss_bwd(b.hidden, b.W, b.targets, f["lse"], f["coeff"], dW_accum=sg.full, want_dhidden=False)
    sg.barrier()
    dW = sg.full.clone()
    sg.close()
    ctx.close()
    assert rel_l2(to64(dW), to64(plain["dW"])) <= 1e-6                     # same kernel, same tiles: atomics order only
    assert rel_l2(to64(dW), run_oracle(b)["dW"]) <= TOL_GRAD_REL


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2606_26997_b200.dp import GrpoDataParallel, StitchedGradient
    from tests.parity_util import make_ctx
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dp = GrpoDataParallel()
    b = _batch()
    mine = dp.local_positions(b.n_groups)
    toks = sum(int(b.seqlens[g * b.G:(g + 1) * b.G].sum()) for g in mine)
    denom = dp.global_denominator(toks)
    ctx = make_ctx(b, groups_per_update=len(mine), max_tokens=toks, bwd_chunk_tokens=512)
    sg = StitchedGradient(ctx, b.V, b.d, dp)                               # own chunk + the peer's, in rank order
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")
    descs = []
    for g in mine:
        t0, t1 = b.group_token_range(g)
        descs.append(ctx.make_group_desc(g, b.seqlens[g * b.G:(g + 1) * b.G], b.hidden[t0:t1], b.targets[t0:t1],
                                         b.old_logp[t0:t1], b.rewards[g * b.G:(g + 1) * b.G].contiguous(),
                                         b.ref_logp[t0:t1]))
    consumed, boundary = ctx.grpo_enqueue_groups(descs, b.W, sg.full, loss, loss_denom=denom)
    assert boundary and consumed == len(mine)
    sg.barrier()                                                           # both ranks' A6 launches are complete
    r0, r1 = sg.local_rows
    q.put((rank, r0, r1, sg.local[:r1 - r0].cpu().numpy(), denom))
    dist.barrier()
    sg.close()
    ctx.close()
    dist.destroy_process_group()


def test_two_ranks_reduce_scatter_inside_the_gemm():
    from tests.parity_util import TOL_GRAD_REL, make_ctx, rel_l2, run_cuda, run_oracle, to64
    world, port = 2, _free_port()
    mpctx = mp.get_context("spawn")
    q = mpctx.Queue()
    procs = [mpctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=600) for _ in range(world)), key=lambda r: r[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    b = _batch()
    ctx = make_ctx(b, max_tokens=b.T, bwd_chunk_tokens=512)
    full = to64(run_cuda(ctx, b, loss_denom=float(b.T))["dW"])
    ctx.close()
    ref = run_oracle(b, loss_denom=float(b.T))["dW"]
    assert (res[0][1], res[0][2], res[1][1], res[1][2]) == (0, 1536, 1536, 3000) and res[0][4] == b.T
    for rank, r0, r1, rows, _ in res:
        assert rel_l2(rows, full[r0:r1]) <= 1e-5                           # the rank's rows hold BOTH ranks' contributions
        assert rel_l2(rows, ref[r0:r1]) <= TOL_GRAD_REL
