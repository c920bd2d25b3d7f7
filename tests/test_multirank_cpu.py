"""world_size-2 `gloo` tests (CPU) of the only multi-rank logic this build has (the path does not
shard through a collective; `bench.py --gpus N` runs one independent complete group per rank):
the whole-job reduction (MAX of the timed regions, SUM of tokens), the per-rank workload assignment, and
the reference arm's "rank 0 alone prints" rule."""
import os
import socket
import subprocess
import sys

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


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "measured" (ms, e2e seconds, tokens) = (10 + 5 r, 0.02 + 0.01 r, 1000 + 7 r)
    ms, e2e, toks = bench.reduce_over_ranks(10.0 + 5.0 * rank, 0.02 + 0.01 * rank, 1000 + 7 * rank, world,
                                            torch.device("cpu"))
    from workloads.synth import make_config
    b = make_config(2, seed=bench.rank_seed(rank), d=64, V=512, len_div=64.0)
    tlist = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(tlist, torch.tensor([b.T], dtype=torch.int64))
    q.put((rank, ms, e2e, toks, [int(t) for t in tlist], float(b.hidden.float().abs().sum())))
    dist.barrier()
    dist.destroy_process_group()


def test_whole_job_reduction_and_per_rank_groups_gloo_world2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, e2e, toks, Ts, _ in res:
        assert ms == 15.0 and e2e == pytest.approx(0.03) and toks == 2007.0     # MAX, MAX, SUM on every rank
    # every rank drew its OWN complete group (different seeds => different lengths / hidden states)
    assert res[0][4] == res[1][4] and res[0][5] != res[1][5]
    # value = tokens all ranks processed / max time
    steps = 4
    assert toks * steps / (ms * 1e-3) == pytest.approx(2007 * 4 / 0.015)


def test_single_rank_reduction_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(12.5, 0.5, 321, 1, None) == (12.5, 0.5, 321.0)


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_ours_arm_fails_loudly_without_cuda():
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "1"],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "no CUDA device" in (r.stderr + r.stdout)


def test_dp_arm_deals_the_update_by_fifo_position():
    """bench.py --dp: one logical update of world x k groups, dealt k mod world like GrpoDataParallel; every position
    is trained by exactly one rank."""
    sys.path.insert(0, ROOT)
    import bench
    U, plan = bench.dp_update_plan(2, 3)
    assert U == 6 and plan == [[0, 2, 4], [1, 3, 5]]
    U, plan = bench.dp_update_plan(8, 2)
    assert U == 16 and sorted(p for r in plan for p in r) == list(range(16)) and all(len(r) == 2 for r in plan)
    assert bench.dp_update_plan(1, 2) == (2, [[0, 1]])
