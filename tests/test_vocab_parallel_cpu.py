"""world_size-2 `gloo` test (CPU) of the vocab-parallel exchange (TP = 4 in the paper's
trainer): shard bounds, shard-local targets, the ONE all-gather of the [3, T] partials into the
[n_shards, T] layout grpo_loss_from_partials reads, and the sum all-reduce of the partial dHidden.  The per-rank
compute here is float64 numpy written out in the test (the CUDA kernels need a GPU: tests/test_vocab_parallel_gpu.py
runs `GrpoVocabParallel.step` with them); what is under test is `dp.py`'s buffer plumbing."""
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


@pytest.mark.parametrize("V,world", [(151936, 4), (3000, 3), (17, 2), (8, 8), (1000, 1)])
def test_shard_bounds_cover_the_vocabulary_once(V, world):
    from paper_2606_26997_b200.dp import vocab_shard_bounds
    b = vocab_shard_bounds(V, world)
    assert len(b) == world + 1 and b[0] == 0 and b[-1] == V
    assert all(b[i] < b[i + 1] for i in range(world))                      # no empty shard
    if V >= 16 * world:
        assert all(x % 8 == 0 for x in b[1:-1])
        sizes = np.diff(b)
        assert sizes.max() - sizes.min() <= 16                             # balanced
    with pytest.raises(ValueError):
        vocab_shard_bounds(3, 4)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2606_26997_b200.dp import GrpoVocabParallel
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(5)                                         # the same batch on both ranks
    T, d, V = 37, 16, 203
    H, W = rng.standard_normal((T, d)), rng.standard_normal((V, d)) * 0.5
    y = rng.integers(0, V, T).astype(np.int32)
    y[3] = -100                                                            # an ignored token
    vp = GrpoVocabParallel(d, V, make_context=False)
    assert (vp.v0, vp.v1) == ((0, 96), (96, 203))[rank]
    y_loc = vp.local_targets(torch.from_numpy(y)).numpy()
    assert y_loc[3] == -1 and np.array_equal(np.delete(y_loc, 3), np.delete(y, 3) - vp.v0)
    Ws = vp.shard_rows(torch.from_numpy(W)).numpy()
    z2 = (H @ Ws.T) * np.log2(np.e)                                        # this shard's logits, log2 domain
    m2 = z2.max(axis=1)
    s2 = np.exp2(z2 - m2[:, None]).sum(axis=1)
    here = (y_loc >= 0) & (y_loc < vp.v1 - vp.v0)
    zy = np.where(here, (H @ Ws.T)[np.arange(T), np.clip(y_loc, 0, vp.v1 - vp.v0 - 1)], 0.0)
    f32 = lambda a: torch.from_numpy(a.astype(np.float32))
    m2g, s2g, zyg = vp.gather_partials(f32(m2), f32(s2), f32(zy))
    assert m2g.shape == (world, T) and m2g.is_contiguous() and s2g.is_contiguous() and zyg.is_contiguous()
    assert torch.equal(m2g[rank], f32(m2)) and torch.equal(s2g[rank], f32(s2)) and torch.equal(zyg[rank], f32(zy))
    dH_part = f32(np.full((T, d), float(rank + 1)) + H)                    # any per-rank partial
    dH = vp.reduce_dhidden(dH_part.clone())
    q.put((rank, m2g.double().numpy(), s2g.double().numpy(), zyg.double().numpy(), dH.double().numpy()))
    dist.barrier()
    dist.destroy_process_group()


def test_gathered_partials_combine_to_the_full_log_sum_exp():
    from scipy.special import logsumexp
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=120) for _ in range(world)), key=lambda r: r[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    rng = np.random.default_rng(5)
    T, d, V = 37, 16, 203
    H, W = rng.standard_normal((T, d)), rng.standard_normal((V, d)) * 0.5
    y = rng.integers(0, V, T).astype(np.int32)
    y[3] = -100
    z = H @ W.T
    for rank, m2g, s2g, zyg, dH in res:
        M = m2g.max(axis=0)                                                # the combine of grpo_loss_from_partials
        lse = (M + np.log2((s2g * np.exp2(m2g - M)).sum(axis=0))) * np.log(2.0)
        np.testing.assert_allclose(lse, logsumexp(z, axis=1), rtol=0, atol=2e-6)
        zy = zyg.sum(axis=0)                                               # exactly one shard holds the target column
        ok = y >= 0
        np.testing.assert_allclose(zy[ok], z[np.arange(T), np.clip(y, 0, V - 1)][ok], rtol=0, atol=2e-6)
        assert zy[3] == 0.0
        np.testing.assert_allclose(dH, 2 * H + 3.0, rtol=0, atol=1e-5)     # (H + 1) + (H + 2)
    for k in range(1, 5):
        np.testing.assert_array_equal(res[0][k], res[1][k])                # replicated after the exchange
