"""world_size-2 `gloo` test (CPU) of the data-parallel boundary (P12 additivity):
each rank trains the groups `GrpoDataParallel` deals it, with the denominator of the WHOLE update, and one sum
all-reduce of dW / loss at the update boundary gives every rank the single-rank full-batch step.  The per-rank
compute here is the float64 oracle (the CUDA kernels need a GPU: tests/test_dp_gpu.py runs the same protocol with
them); what is under test is the host logic: group -> rank assignment, global denominators, asynchronous reduction,
alternating buffers."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q, loss_agg):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from oracle.grpo_oracle import OracleConfig, grpo_step
    from paper_2606_26997_b200.dp import GrpoDataParallel
    from workloads.synth import make_config, slice_groups
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dp = GrpoDataParallel()
    b = make_config(1, seed=3, variant="1b", n_groups=5, G=4, d=32, V=200, loss_agg=loss_agg)    # same batch on both ranks
    cfg = OracleConfig(kl_beta=b.kl_beta, clip_lo=b.clip_lo, clip_hi=b.clip_hi, loss_agg=loss_agg)
    mine = dp.local_positions(b.n_groups)                       # the update = all 5 groups, dealt 3 / 2
    sub = slice_groups(b, mine)
    denom = dp.global_denominator(sub.T)                        # token mean over the WHOLE update
    S_all = dp.global_sequences(sub.S)
    x = sub.numpy_f64()
    out = grpo_step(x["H"], x["W"], x["y"], x["cu_seqlens"], x["rewards"], x["old_logp"], x["ref_logp"], cfg=cfg,
                    G=b.G, loss_denom=denom)
    scale = sub.S / S_all if loss_agg == 1 else 1.0             # per-sequence mean: 1/S_update instead of 1/S_local
    dW, loss, _ = dp.buffers(b.V, b.d, device="cpu")
    dW2, _, _ = dp.buffers(b.V, b.d, device="cpu")
    dW3, _, _ = dp.buffers(b.V, b.d, device="cpu")
    assert dW2.data_ptr() != dW.data_ptr() and dW3.data_ptr() == dW.data_ptr()      # two sets, alternating
    dW.copy_(torch.from_numpy(out["dW"] * scale).float())
    loss.fill_(out["loss"] * scale)
    h = dp.reduce_boundary(dW, loss)
    h.wait()
    q.put((rank, mine, denom, S_all, dW.double().numpy(), float(loss)))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("loss_agg", [0, 1])
def test_sum_over_ranks_equals_the_full_batch_step(loss_agg):
    sys.path.insert(0, ROOT)
    from oracle.grpo_oracle import OracleConfig, grpo_step
    from workloads.synth import make_config
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q, loss_agg)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=240) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    b = make_config(1, seed=3, variant="1b", n_groups=5, G=4, d=32, V=200, loss_agg=loss_agg)
    x = b.numpy_f64()
    full = grpo_step(x["H"], x["W"], x["y"], x["cu_seqlens"], x["rewards"], x["old_logp"], x["ref_logp"],
                     cfg=OracleConfig(kl_beta=b.kl_beta, clip_lo=b.clip_lo, clip_hi=b.clip_hi, loss_agg=loss_agg), G=b.G)
    assert res[0][1] == [0, 2, 4] and res[1][1] == [1, 3]
    for rank, mine, denom, S_all, dW, loss in res:
        assert denom == b.T and S_all == b.S
        np.testing.assert_allclose(dW, full["dW"], rtol=1e-5, atol=1e-9)       # fp32 buffers
        np.testing.assert_allclose(loss, full["loss"], rtol=1e-5)
    np.testing.assert_array_equal(res[0][4], res[1][4])                        # every rank holds the same sum


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    from paper_2606_26997_b200.dp import GrpoDataParallel, assign_groups
    dp = GrpoDataParallel()
    assert dp.world == 1 and dp.local_positions(3) == [0, 1, 2] and dp.global_denominator(17) == 17.0
    t = torch.ones(4, 2)
    dp.reduce_boundary(t, torch.ones(1)).wait()
    assert torch.equal(t, torch.ones(4, 2))
    assert [assign_groups(7, 3, r) for r in range(3)] == [[0, 3, 6], [1, 4], [2, 5]]


def _node_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2606_26997_b200.dp import GrpoDataParallel, _require_one_node
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dp = GrpoDataParallel()
    _require_one_node(dp, device=-1)                              # both ranks really are on this machine
    try:
        _require_one_node(dp, identity=f"node-{rank}", device=-1)  # pretend they are not
        q.put((rank, "no error"))
    except RuntimeError as e:
        q.put((rank, str(e)))
    dist.barrier()
    dist.destroy_process_group()


def test_stitched_gradient_refuses_ranks_on_different_nodes():
    """The stitched accumulator passes shard handles as file descriptors over Unix sockets: one machine only.  Ranks
    on different machines get a clear error on EVERY rank instead of a hang in connect()."""
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_node_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        assert "one node" in res[r] and "spans 2 nodes" in res[r]
