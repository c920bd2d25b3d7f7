"""CPU-only checks of the C ABI: the library loads, exports every symbol include/grpo.h declares,
and the pure-host CGP planner follows the paper's FIFO / feasible-prefix rules.  No compute calls."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_26997_b200.build import build
    build()
    from paper_2606_26997_b200.binding import load_library
    return load_library()


def test_every_declared_symbol_is_exported(lib):
    header = open(os.path.join(ROOT, "include", "grpo.h")).read()
    declared = set(re.findall(r"^(?:int32_t|const char\*)\s+(grpo_[a-z_0-9]+)\s*\(", header, flags=re.M))
    assert {"grpo_group_advantage", "grpo_fused_logprob_loss_fwd", "grpo_fused_logprob_loss_bwd",
            "grpo_enqueue_groups"} <= declared
    for name in sorted(declared):
        assert hasattr(lib, name), name
    from paper_2606_26997_b200.binding import EXPORTS
    assert declared == set(EXPORTS)


def test_default_config_and_struct_layout(lib):
    from paper_2606_26997_b200.binding import GrpoConfig
    cfg = GrpoConfig()
    assert lib.grpo_default_config(C.byref(cfg)) == 0
    assert cfg.eps_std == pytest.approx(1e-6) and cfg.clip_lo == pytest.approx(0.2)
    assert cfg.clip_hi == pytest.approx(0.28) and cfg.groups_per_update == 1 and cfg.bwd_chunk_tokens == 9472
    assert lib.grpo_default_config(None) != 0
    assert b"NULL" in lib.grpo_last_error()


def test_create_without_gpu_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2606_26997_b200.binding import GrpoConfig
    cfg = GrpoConfig()
    lib.grpo_default_config(C.byref(cfg))
    cfg.d, cfg.V = 64, 1000
    h = C.c_void_p()
    st = lib.grpo_create(C.byref(cfg), C.byref(h))
    assert st == 5 and h.value is None            # GRPO_ERR_CUDA: no silent fallback
    cfg.d = 60                                    # d % 8 != 0 is a shape error before any CUDA call
    assert lib.grpo_create(C.byref(cfg), C.byref(h)) == 2


# ---- CGP planner: PAPER.md:92 (earliest U dispatched), :187 (largest prefix of whole groups within the
# token budget; an over-budget group is taken alone), :111 (update boundary every U groups)
def test_plan_waits_for_U_groups():
    from paper_2606_26997_b200 import grpo_cgp_plan
    assert grpo_cgp_plan([100], U=2) == []                      # group 0 waits for group 1
    assert grpo_cgp_plan([100, 200], U=2) == [2]
    assert grpo_cgp_plan([100, 200, 300], U=2) == [2]           # only the earliest U
    assert grpo_cgp_plan([100], U=2, flush=True) == [1]
    assert grpo_cgp_plan([], U=2, flush=True) == []


def test_plan_feasible_prefix_whole_groups():
    from paper_2606_26997_b200 import grpo_cgp_plan
    toks = [4000, 3000, 5000, 1000]
    assert grpo_cgp_plan(toks, U=4, token_budget=8000) == [2, 2]     # 4000+3000 | 5000+1000
    assert grpo_cgp_plan(toks, U=4, token_budget=6000) == [1, 1, 2]
    assert grpo_cgp_plan(toks, U=4, token_budget=100) == [1, 1, 1, 1]  # over-budget groups taken alone
    assert grpo_cgp_plan(toks, U=4, token_budget=0) == [4]
    assert sum(grpo_cgp_plan(toks, U=3, token_budget=7000)) == 3


def test_plan_property_prefix_is_maximal():
    import random
    from paper_2606_26997_b200 import grpo_cgp_plan
    rnd = random.Random(0)
    for _ in range(200):
        n = rnd.randint(1, 12)
        toks = [rnd.randint(1, 9000) for _ in range(n)]
        U = rnd.randint(1, n)
        budget = rnd.randint(1, 20000)
        sizes = grpo_cgp_plan(toks, U=U, token_budget=budget)
        assert sum(sizes) == U and all(s >= 1 for s in sizes)
        pos = 0
        for s in sizes:
            tot = sum(toks[pos:pos + s])
            assert s == 1 or tot <= budget                           # fits unless a lone over-budget group
            if pos + s < U:
                assert tot + toks[pos + s] > budget                  # could not have taken one more
            pos += s
