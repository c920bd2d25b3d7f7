#!/usr/bin/env python
"""bench.py — GRPO loss fwd+bwd tokens/s at d=2048, V=151936 on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

One "step" is one pass of the whole hot path (group advantage, LM-head
contraction + online log-sum-exp, loss epilogue, backward recompute + dZ, dH, dW accumulation) over one
batch of synthetic input.  At N=1 the workload is BASELINE.json configs[1]: one complete group, G=8
responses of 512..4096 tokens, d=2048, V=151936 (Qwen3-1.7B LM-head shape), on-policy old log-probs,
no KL.  With N>1 (torchrun, one rank per GPU) every rank runs its own complete group (weak scaling over
independent groups; the path has no collective — DESIGN.md §7); the only torch.distributed traffic is
the barrier and the max/sum of the measurements.

Output: ONE JSON line on rank 0 (keys documented in DESIGN.md §6).  The headline `value` is always the north_star
path (forward, then the backward that recomputes the logits chunk by chunk); `other_variant` times the
3-contraction variant beside it.  Informational switches: `--stash` (make that variant the step),
`--config 3|4|5` (the other BASELINE configs, device-resident), `--cgp-mode per_group|batch4` (configs[4] streamed
through grpo_enqueue_groups), `--no-tile-skip`, `--no-drift-gate`, `--cta-group 1`, `--bwd-chunk N`, `--max-ctas N` (A/B runs).
`--impl reference` times the float64 CPU oracle (oracle/) on the host cores, on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "GRPO loss fwd+bwd tokens/sec at d=2048,V=151936; % of B200 BF16 tensor peak"
UNIT = "tokens/s"
# Oracle samples: configs[1] with response lengths / div at full d and V.  The cpu_baseline leg times ONE
# oracle step (~10-20 s of CPU work); the --impl reference arm times steps+warmup of them, so its sample is
# smaller (~3 s per step) to keep the whole run within a few minutes.
SAMPLE_LEN_DIV = 8.0           # cpu_baseline leg: T ~ 2.3k tokens
REF_SAMPLE_LEN_DIV = 32.0      # --impl reference arm: T ~ 580 tokens per step
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r03_traffic.txt")
KERNEL_SOURCES = ("gemm_sm100.cuh", "ptx_sm100.cuh", "token_kernels.cuh", "grpo_api.cu")


def kernel_source_hash():
    """sha256 over the CUDA sources: identifies the build an ncu capture belongs to."""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2606_26997_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def load_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of each contraction kernel, from the committed
    `ncu --set full` capture (profiles/r03_traffic.txt: `key value` lines, written from the capture's raw page).
    The capture names the source hash of the build it profiled; a capture of ANOTHER build is not reported as this
    build's traffic: the figure is dropped (null) and the mismatch is said on stderr and in the JSON line."""
    if not os.path.exists(TRAFFIC_FILE):
        return {}, "no ncu capture committed for this build"
    vals = {}
    with open(TRAFFIC_FILE) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) == 2:
                vals[line[0]] = line[1]
    have = kernel_source_hash()
    if vals.get("kernel_source_hash") != have:
        msg = (f"profiles/r03_traffic.txt is a capture of build {vals.get('kernel_source_hash')}, this build is {have}: "
               "roofline.traffic dropped (re-run the ncu capture)")
        print("bench.py: " + msg, file=sys.stderr)
        return {}, msg
    return {k: float(v) for k, v in vals.items() if k.startswith("gemm_")}, "profiles/r03_traffic.txt"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    d = dict(FALLBACK_PEAKS)
    d["_source"] = "fallback"
    return d


class ClockSampler:
    """Samples SM clock and clock-event reasons of one GPU with NVML while the timed region runs."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting",
               0x10: "sync_boost"}

    def __init__(self, torch_index: int, period_s: float = 0.02):
        self.period = period_s
        self.samples = []
        self.mask = 0
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        self.h = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                uuid = "GPU-" + str(torch.cuda.get_device_properties(torch_index).uuid)
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode())
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(torch_index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:      # NVML missing: report that, never fake a clock
            self.err = repr(e)

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1e3)
                except Exception:
                    pass
                try:
                    self.mask |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    self.mask |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            except Exception:
                pass
            self._stop.wait(self.period)

    def energy_mj(self):
        """NVML total energy counter of the board in millijoules (None if unavailable)."""
        try:
            return int(self.nv.nvmlDeviceGetTotalEnergyConsumption(self.h))
        except Exception:
            return None

    def start(self):
        if self.h is not None:
            self.power = []
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr is not None:
            self._stop.set()
            self._thr.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        reasons = [name for bit, name in self.REASONS.items() if self.mask & bit]
        out = {"sm_mhz": int(statistics.median(self.samples)), "sm_max_mhz": self.max_mhz,
               "sm_min_mhz": min(self.samples), "samples": len(self.samples), "reasons": reasons}
        if getattr(self, "power", None):
            out["power_w_median"] = round(statistics.median(self.power), 1)
        return out


def cublas_anchor(torch_index: int, seconds: float = 1.0):
    """Same-run, same-box anchor for the roofline fraction: ~`seconds` of back-to-back torch.matmul (cuBLAS) bf16
    8192 x 8192 x 2048 with N(0,1) operands on this device, outside every timed region, with its own clock sample.
    MEASURED_PEAKS.json was taken on another lease (other clocks under the same power cap); this is the library's
    rate on THIS board at THIS moment, so kernel TFLOP/s divided by it does not move with the box."""
    import torch
    dev = torch.device("cuda", torch_index)
    M = N = 8192
    K = 2048
    gen = torch.Generator(device=dev)
    gen.manual_seed(7)
    A = torch.randn(M, K, generator=gen, device=dev, dtype=torch.float32).to(torch.bfloat16)
    B = torch.randn(N, K, generator=gen, device=dev, dtype=torch.float32).to(torch.bfloat16)
    C = torch.empty(M, N, device=dev, dtype=torch.bfloat16)
    fn = lambda: torch.matmul(A, B.t(), out=C)
    for _ in range(20):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(20):
        fn()
    e1.record()
    torch.cuda.synchronize()
    n = max(20, int(seconds * 1e3 / (e0.elapsed_time(e1) / 20)))
    sampler = ClockSampler(torch_index)
    sampler.start()
    e0.record()
    for _ in range(n):
        fn()
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1) / n
    return {"tflops": 2.0 * M * N * K / ms / 1e9, "shape": [M, N, K], "calls": n, "seconds": ms * n * 1e-3,
            "api": "torch.matmul bf16 (cuBLAS), N(0,1) operands", "clocks": clocks}


# ----------------------------------------------------------------------------------------- oracle legs
def oracle_sample(device="cpu", len_div=SAMPLE_LEN_DIV):
    """Bounded sample of the timed workload for the CPU oracle: configs[1] with lengths / len_div."""
    from workloads.synth import make_config
    b = make_config(2, seed=0, device=device, len_div=len_div)
    return b.to("cpu") if device != "cpu" else b


def time_oracle_step(b):
    """One fwd+bwd of the oracle as it stands on sample `b`; returns seconds."""
    from oracle.grpo_oracle import OracleConfig, grpo_step
    x = b.numpy_f64()
    cfg = OracleConfig(eps_std=b.eps_std, clip_lo=b.clip_lo, clip_hi=b.clip_hi, kl_beta=b.kl_beta, loss_agg=b.loss_agg)
    t0 = time.perf_counter()
    out = grpo_step(x["H"], x["W"], x["y"], x["cu_seqlens"], x["rewards"], x["old_logp"], x["ref_logp"],
                    mask=x["mask"], cfg=cfg, G=b.G)
    dt = time.perf_counter() - t0
    assert out["dW"].shape == x["W"].shape
    return dt


def oracle_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 0) for p in threadpool_info() if p.get("user_api") == "blas"]
        if n:
            return int(max(n))
    except Exception:
        pass
    return os.cpu_count() or 1


def sample_desc(b, len_div=SAMPLE_LEN_DIV):
    return (f"configs[1] with response lengths/{len_div:g}: 1 group x G={b.G}, T={b.T} tokens, d={b.d}, "
            f"V={b.V}; one oracle fwd+bwd (float64, numpy/OpenBLAS) per step")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    b = oracle_sample("cpu", REF_SAMPLE_LEN_DIV)
    for _ in range(args.warmup):
        time_oracle_step(b)
    times = [time_oracle_step(b) for _ in range(args.steps)]
    total = sum(times)
    value = b.T * args.steps / total
    cores = oracle_threads()
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[1]: one complete group G=8, lengths U[512,4096], d=2048, V=151936 "
                               "(bounded sample, see cpu_baseline.sample)", "tokens_per_step": b.T},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": sample_desc(b, REF_SAMPLE_LEN_DIV)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------------------- CUDA arm
def rank_seed(rank: int) -> int:
    """Rank r times its own complete group (weak scaling over independent groups)."""
    return int(rank)


def reduce_over_ranks(ms_total: float, e2e_s: float, tokens: int, world: int, device):
    """Whole-job figures: the timed regions' MAX over ranks and the SUM of the tokens all ranks processed.
    The only torch.distributed traffic of the benchmark besides the barriers (the path has no collective)."""
    if world <= 1:
        return float(ms_total), float(e2e_s), float(tokens)
    import torch
    import torch.distributed as dist
    stats = torch.tensor([ms_total, e2e_s], dtype=torch.float64, device=device)
    toks = torch.tensor([float(tokens)], dtype=torch.float64, device=device)
    dist.all_reduce(stats, op=dist.ReduceOp.MAX)
    dist.all_reduce(toks, op=dist.ReduceOp.SUM)
    ms, e2e = stats.tolist()
    return ms, e2e, toks.item()


# north_star: the throughput "sits next to ... the paper's rollout-to-train-end reductions ... quoted with the hardware the
# paper states, as context only".  The paper has no number for this path: vs_baseline stays null.
PAPER_CONTEXT = {
    "rollout_to_train_end_reduction_vs_slime": "30.7 %-42.3 % (CGP+FGD over 12 settings; PAPER.md:9, 220)",
    "trainer_waiting_ratio": "Slime 47-52 %, CGP+FGD 14-33 % (PAPER.md:46, 236)",
    "hardware": "policy Qwen3-1.7B; trainer 8x RTX 4090 24 GB (TP=4, DP=2), rollout 2x A100 40 GB PCIe (TP=2) (PAPER.md:197)",
    "note": "whole-system times of the paper's Slime/SGLang/Megatron stack on other hardware: context only, not a "
            "target and not comparable with this line's tokens/s of the loss step alone",
}
GEMM_KINDS = ("gemm_lse", "gemm_dz", "gemm_dh", "gemm_dw")
WORKLOADS = {
    2: "configs[1]: one complete group G=8, lengths U[512,4096], d=2048, V=151936, on-policy old log-probs, "
       "no KL; one such group per GPU",
    3: "configs[2] (informational): 4 groups x G=8, lognormal lengths, zero-variance groups kept, KL beta=0.001",
    4: "configs[3] (informational): 8 groups x G=16, lognormal long-tail lengths, Beta-Bernoulli rewards, no KL",
    5: "configs[4] as ONE full-batch step (informational): 32 groups x G=8, geometric lengths, no KL",
}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_26997_b200 import GrpoContext
    from paper_2606_26997_b200.build import build
    from workloads.synth import make_config

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback (use --impl reference "
                         "for the oracle baseline)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if local == 0:
        build()
    if world > 1:
        dist.barrier()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.dp:
        return run_dp(args, dev, rank, world, local)
    if args.power_study:
        assert world == 1, "--power-study is a one-GPU informational run"
        return run_power_study(args, dev)
    if args.sweep_T:
        assert world == 1, "--sweep-T is a one-GPU informational run"
        return run_sweep_T(args, dev)
    # ---- workload: BASELINE.json configs[1]; rank r draws its own complete group (seed r)
    gen_kw = dict(old_sigma=0.3, mask_frac=0.1) if args.off_policy else {}
    if args.d:
        gen_kw["d"] = args.d
    if args.V:
        gen_kw["V"] = args.V
    args.informational = bool(args.off_policy or args.d or args.V or args.prenorm or args.fp8 or args.config != 2)
    b = make_config(args.config, seed=rank_seed(rank), device=dev, prenorm=args.prenorm, **gen_kw)
    if args.cgp_mode != "full":
        return run_cgp_stream(args, b, dev, world)
    T, d, V = b.T, b.d, b.V
    extra = {}
    if args.no_tile_skip:
        extra["bwd_skip_zero_tiles"] = -1
    if args.no_drift_gate:
        extra["gemm_drift_epoch_kb"] = -1
    elif args.drift_epoch:
        extra["gemm_drift_epoch_kb"] = args.drift_epoch
    if args.fp8:
        extra["fp8_logits"] = 1
    if args.max_ctas:
        extra["gemm_max_ctas"] = args.max_ctas
    if args.stash:
        extra["stash_logits"] = 1           # grpo_step_host (the e2e leg) then uses the same variant
    ctx = GrpoContext(d, V, max_tokens=T, group_size=b.G, kl_beta=b.kl_beta, clip_lo=b.clip_lo, clip_hi=b.clip_hi,
                      gemm_cta_group=args.cta_group, **extra, **({"bwd_chunk_tokens": args.bwd_chunk} if args.bwd_chunk else {}))
    dW = torch.zeros(V, d, dtype=torch.float32, device=dev)
    loss = torch.zeros(1, dtype=torch.float32, device=dev)
    dH = torch.empty(T, d, dtype=torch.bfloat16, device=dev)

    def step_recompute():       # north_star: forward, then backward with the logits recomputed chunk by chunk
        adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
        f = ctx.grpo_fused_logprob_loss_fwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp,
                                            b.mask, loss_accum=loss)
        ctx.grpo_fused_logprob_loss_bwd(b.hidden, b.W, b.targets, f["lse"], f["coeff"], dW_accum=dW, dhidden_out=dH)

    dgamma = torch.zeros(d, dtype=torch.float32, device=dev)

    def step_prenorm():         # NEXT-4 (informational): final RMSNorm -> north_star path -> dx, dgamma, dW
        Hn, rstd = ctx.grpo_rmsnorm_fwd(b.x_prenorm, b.gamma, b.eps_rms)
        adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
        f = ctx.grpo_fused_logprob_loss_fwd(Hn, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp, b.mask,
                                            loss_accum=loss)
        ctx.grpo_fused_logprob_loss_bwd_prenorm(b.x_prenorm, b.gamma, rstd, Hn, b.W, b.targets, f["lse"], f["coeff"],
                                                dgamma, dW_accum=dW)

    def step_stash():           # 3-contraction variant: logits stashed per chunk
        adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
        ctx.grpo_fused_logprob_loss_fwd_bwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp,
                                            b.mask, loss_accum=loss, dW_accum=dW, dhidden_out=dH)

    step = step_prenorm if args.prenorm else (step_stash if args.stash else step_recompute)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    assert ctx.grpo_check_errors_sync() == 0
    dW.zero_()
    loss.zero_()

    # ---- timed region (the headline): K steps, CUDA events on the launch stream; the library's per-kernel
    # profiling events are OFF here
    sampler = ClockSampler(local)
    n0 = ctx.grpo_kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    barrier()
    ms_total = e0.elapsed_time(e1)
    n1 = ctx.grpo_kernel_launches()
    launches = sum(n1.values()) - sum(n0.values())
    loss_val = loss.item()
    assert loss_val == loss_val, "loss is NaN"

    # ---- end to end through the C ABI with HOST buffers (grpo_step_host): H2D + compute + D2H per step.  Timed
    # right after the headline region so that both see the same thermal / power state of the board.
    e2e_s, h2d, d2h = 0.0, 0, 0
    if not args.informational:
        pin = lambda t: None if t is None else t.cpu().pin_memory()
        h_hidden, h_targets, h_cu, h_rewards, h_old = (pin(b.hidden), pin(b.targets), pin(b.cu_seqlens), pin(b.rewards),
                                                       pin(b.old_logp))
        h_logp = torch.empty(T, dtype=torch.float32).pin_memory()
        h_dh = torch.empty(T, d, dtype=torch.bfloat16).pin_memory()
        h_loss = torch.zeros(1, dtype=torch.float32).pin_memory()

        def step_host():
            ctx.grpo_step_host(h_hidden, h_targets, h_cu, h_rewards, h_old, b.n_groups, b.G, b.W, dW, loss_h=h_loss,
                               logp_h=h_logp, dhidden_h=h_dh)

        for _ in range(2):
            step_host()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            step_host()                     # synchronises its stream before returning: the host has the results
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
        barrier()
        h2d = sum(t.numel() * t.element_size() for t in (h_hidden, h_targets, h_cu, h_rewards, h_old))
        d2h = sum(t.numel() * t.element_size() for t in (h_logp, h_dh, h_loss))


    # ---- the same K steps once more with a CUDA event pair around every kernel launch (recorded by the library on
    # the launch stream): per-kernel times for the roofline; the pass's own total is reported beside the headline
    ctx.grpo_bwd_row_stats_sync()           # clear
    ctx.grpo_profile_enable(True)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    p0.record()
    for _ in range(args.steps):
        step()
    p1.record()
    torch.cuda.synchronize()
    barrier()
    args.profiled_ms_per_step = p0.elapsed_time(p1) / args.steps
    prof = ctx.grpo_profile_read_sync()
    ctx.grpo_profile_enable(False)
    rows_walked, rows_total = ctx.grpo_bwd_row_stats_sync()
    args.bwd_active_frac = rows_walked / rows_total if rows_total > 0 else 1.0
    args.bwd_rows = {"walked": rows_walked, "total": rows_total}

    # ---- energy: NVML's board energy counter around a >= 2 s run of the same step (the counter is too coarse
    # for the 0.35 s headline region); joules per step, mean power, tokens per joule
    args.energy = None
    if world == 1 and not args.no_energy:
        n_e = max(args.steps, int(2000.0 / max(ms_total / args.steps, 1e-3)) + 1)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        mj0 = sampler.energy_mj() if sampler.h is not None else None
        g0.record()
        for _ in range(n_e):
            step()
        g1.record()
        torch.cuda.synchronize()
        mj1 = sampler.energy_mj() if sampler.h is not None else None
        if mj0 is not None and mj1 is not None and mj1 > mj0:
            sec = g0.elapsed_time(g1) * 1e-3
            joules = (mj1 - mj0) * 1e-3
            args.energy = {"joules_per_step": joules / n_e, "mean_power_w": joules / sec, "tokens_per_joule": T * n_e / joules,
                           "steps": n_e, "tokens_per_s": T * n_e / sec, "source": "nvmlDeviceGetTotalEnergyConsumption"}

    # ---- the other variant of the step, timed the same way (reported beside the headline, never as it)
    args.other_variant = None
    if not args.no_variants and not args.prenorm and not args.fp8:
        other = step_recompute if args.stash else step_stash
        for _ in range(3):
            other()
        barrier()
        v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        v0.record()
        for _ in range(args.steps):
            other()
        v1.record()
        torch.cuda.synchronize()
        barrier()
        v_ms, _, v_tok = reduce_over_ranks(v0.elapsed_time(v1), 0.0, T, world, dev)
        args.other_variant = {"variant": "recompute (north_star)" if args.stash else "stash_logits (3 contractions)",
                              "value": v_tok * args.steps / (v_ms * 1e-3), "unit": UNIT,
                              "ms_per_step": v_ms / args.steps}

    # ---- same-run cuBLAS anchor (outside every timed region): the roofline fraction against the library's rate on
    # this board, now
    args.cublas_anchor = None
    if world == 1 and not args.no_anchor:
        args.cublas_anchor = cublas_anchor(local)

    # ---- informational runs (--config 3/4/5, --prenorm) are device-resident: no e2e / cpu_baseline legs
    if args.informational:
        ms_total, _, tokens_all = reduce_over_ranks(ms_total, 0.0, T, world, dev)
        if rank == 0:
            line = build_line(args, b, world, tokens_all * args.steps / (ms_total * 1e-3), ms_total, None, 0, 0,
                              launches, prof, clocks, load_peaks(), tokens_all, loss_val)
            print(json.dumps(line), flush=True)
        ctx.close()
        if world > 1:
            dist.destroy_process_group()
        return 0
    # ---- reduce over ranks: max time, sum tokens
    ms_total, e2e_s, tokens_all = reduce_over_ranks(ms_total, e2e_s, T, world, dev)
    value = tokens_all * args.steps / (ms_total * 1e-3)
    e2e_value = tokens_all * args.steps / e2e_s

    if rank == 0:
        peaks = load_peaks()
        line = build_line(args, b, world, value, ms_total, e2e_value, h2d, d2h, launches, prof, clocks, peaks,
                          tokens_all, loss_val)
        if world == 1 and not args.no_cpu_baseline:
            sb = oracle_sample(dev)
            dt = time_oracle_step(sb)
            line["cpu_baseline"] = {"value": sb.T / dt, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle",
                                    "sample": sample_desc(sb), "seconds": dt}
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


SWEEP_T = (2000, 4000, 8000, 10000, 16000, 18701, 24000, 33000)


def run_sweep_T(args, dev):
    """Informational (one JSON line): tokens/s of ONE complete group per launch at T ~ 2k .. 33k tokens - the range
    configs[1] draws from (8 responses of 512..4096 tokens) and the regime CGP feeds, one launch per arriving group
    (PAPER.md:92).  Same recipe as configs[1] with the response lengths rescaled; device-resident; north_star path
    and the 3-contraction variant."""
    import torch
    from paper_2606_26997_b200 import GrpoContext
    from workloads.synth import make_config
    rows = []
    ctx = None
    for T_target in SWEEP_T:
        b = make_config(2, seed=0, device=dev, len_div=18701.0 / T_target)
        if ctx is None:
            ctx = GrpoContext(b.d, b.V, max_tokens=int(max(SWEEP_T) * 1.1), group_size=b.G, kl_beta=b.kl_beta,
                              clip_lo=b.clip_lo, clip_hi=b.clip_hi)
        dW = torch.zeros(b.V, b.d, dtype=torch.float32, device=dev)
        loss = torch.zeros(1, dtype=torch.float32, device=dev)
        dH = torch.empty(b.T, b.d, dtype=torch.bfloat16, device=dev)

        def step_recompute():
            adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
            f = ctx.grpo_fused_logprob_loss_fwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp,
                                                b.mask, loss_accum=loss)
            ctx.grpo_fused_logprob_loss_bwd(b.hidden, b.W, b.targets, f["lse"], f["coeff"], dW_accum=dW, dhidden_out=dH)

        def step_stash():
            adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
            ctx.grpo_fused_logprob_loss_fwd_bwd(b.hidden, b.W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp,
                                                b.mask, loss_accum=loss, dW_accum=dW, dhidden_out=dH)

        row = {"T": b.T}
        for name, fn in (("recompute", step_recompute), ("stash", step_stash)):
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            n = max(args.steps, int(300.0 * 18701 / b.T / 35.0) + 1)      # ~0.3 s per point
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(n):
                fn()
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / n
            row[name] = {"tokens_per_s": b.T / (ms * 1e-3), "ms_per_step": ms, "steps": n}
        rows.append(row)
        del dW, dH, b
    ref = next(r for r in rows if abs(r["T"] - 18701) < 200)
    for r in rows:
        r["recompute"]["vs_T18701"] = r["recompute"]["tokens_per_s"] / ref["recompute"]["tokens_per_s"]
        r["stash"]["vs_T18701"] = r["stash"]["tokens_per_s"] / ref["stash"]["tokens_per_s"]
    print(json.dumps({"metric": METRIC, "unit": UNIT, "informational": "sweep_T", "n_gpus": 1, "dtype": "bf16",
                      "data": "synthetic", "config": {"workload": "configs[1] recipe, one complete group G=8 per launch, "
                      "response lengths rescaled to T tokens; d=2048, V=151936"}, "sweep_T": rows}), flush=True)
    ctx.close()
    return 0


def run_power_study(args, dev):
    """Informational (one JSON line): how much of the 1000 W board cap the OPERAND DATA costs.  The north_star step of
    configs[1] is timed for >= 1.5 s on its synthetic operands and again with H and W replaced by zeros (same
    launches, same tiles, same bytes moved: only the bits that toggle in the tensor-core datapath differ), and
    cuBLAS (torch.matmul bf16 8192^3, the shape MEASURED_PEAKS.json was taken on) with N(0,1) and with zero
    operands beside it.  DESIGN.md section 5, "Where the power goes"."""
    import torch
    from paper_2606_26997_b200 import GrpoContext
    from workloads.synth import make_config
    b = make_config(2, seed=0, device=dev)
    T, d, V = b.T, b.d, b.V
    # dense backward: with zero operands every ratio leaves the clip range and the row compaction would drop the rows
    ctx = GrpoContext(d, V, max_tokens=T, group_size=b.G, kl_beta=b.kl_beta, clip_lo=b.clip_lo, clip_hi=b.clip_hi,
                      bwd_skip_zero_tiles=-1)
    dW = torch.zeros(V, d, dtype=torch.float32, device=dev)
    loss = torch.zeros(1, dtype=torch.float32, device=dev)
    dH = torch.empty(T, d, dtype=torch.bfloat16, device=dev)

    def sustained(fn, seconds, flops):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); fn(); e1.record(); torch.cuda.synchronize()
        n = max(3, int(seconds * 1e3 / e0.elapsed_time(e1)))
        sampler = ClockSampler(dev.index or 0)
        sampler.start()
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        clocks = sampler.stop()
        ms = e0.elapsed_time(e1) / n
        return {"ms": ms, "tflops": flops / ms / 1e9, "sm_mhz": clocks.get("sm_mhz"),
                "power_w": clocks.get("power_w_median"), "reasons": clocks.get("reasons"), "calls": n}

    rows = {}
    for name in ("synthetic", "zeros"):
        H, W = (b.hidden, b.W) if name == "synthetic" else (torch.zeros_like(b.hidden), torch.zeros_like(b.W))

        def step():
            adv = ctx.grpo_group_advantage(b.rewards, G=b.G)
            f = ctx.grpo_fused_logprob_loss_fwd(H, W, b.targets, b.cu_seqlens, adv, b.old_logp, b.ref_logp, b.mask,
                                                loss_accum=loss)
            ctx.grpo_fused_logprob_loss_bwd(H, W, b.targets, f["lse"], f["coeff"], dW_accum=dW, dhidden_out=dH)

        r = sustained(step, 1.5, 8.0 * T * V * d)
        r["tokens_per_s"] = T / (r["ms"] * 1e-3)
        rows["grpo_step_" + name] = r
        del H, W
    n = 8192
    for name in ("randn", "zeros"):
        A = (torch.randn if name == "randn" else torch.zeros)(n, n, device=dev, dtype=torch.bfloat16)
        B = (torch.randn if name == "randn" else torch.zeros)(n, n, device=dev, dtype=torch.bfloat16)
        C = torch.empty(n, n, device=dev, dtype=torch.bfloat16)
        rows["cublas_8192_" + name] = sustained(lambda: torch.matmul(A, B, out=C), 1.5, 2.0 * n ** 3)
    # Which input of the multipliers the energy follows: ONE operand random, the other constant, both ways round,
    # through cuBLAS and through this library's contraction kernel (grpo_debug_gemm: the production kernel with a
    # plain fp32 epilogue; layout 0: A [M, K] and B [N, K] both K-major, like A2 / A4).  K = 2048 so that both
    # operands stay in L2 and DRAM traffic is out of the picture.  torch.matmul(A, B^T) hands row-major operands to
    # a column-major library, which swaps their roles: its expensive side is the other one.
    K2 = 2048
    mk = {"randn": lambda: torch.randn(n, K2, device=dev, dtype=torch.bfloat16),
          "zeros": lambda: torch.zeros(n, K2, device=dev, dtype=torch.bfloat16),
          "ones": lambda: torch.ones(n, K2, device=dev, dtype=torch.bfloat16)}
    Cf = torch.empty(n, n, device=dev, dtype=torch.float32)
    Cb = torch.empty(n, n, device=dev, dtype=torch.bfloat16)
    for ka, kb in (("randn", "randn"), ("randn", "zeros"), ("zeros", "randn"), ("randn", "ones"), ("ones", "randn"),
                   ("zeros", "zeros")):
        A, B = mk[ka](), mk[kb]()
        rows[f"grpo_gemm_A_{ka}_B_{kb}"] = sustained(lambda: ctx.grpo_debug_gemm(0, A, B, n, n, K2, C_out=Cf), 0.8,
                                                     2.0 * n * n * K2)
        rows[f"cublas_A_{ka}_B_{kb}"] = sustained(lambda: torch.matmul(A, B.t(), out=Cb), 0.8, 2.0 * n * n * K2)
    print(json.dumps({"metric": METRIC, "unit": UNIT, "informational": "power_study", "n_gpus": 1, "dtype": "bf16",
                      "data": "synthetic", "config": {"workload": "configs[1], north_star step; operands as drawn vs "
                      "all-zero H and W; torch.matmul bf16 8192^3 beside it"}, "power_study": rows}), flush=True)
    ctx.close()
    return 0


def run_cgp_stream(args, b, dev, world):
    """configs[4] (informational): the 32 complete groups are handed to grpo_enqueue_groups one at a time in their
    seeded arrival order, as CGP delivers them: `per_group` = U = 1, one launch per group on one
    stream; `batch4` = U = 4, 4-group launches round-robin on 4 streams.  Gradients accumulate in fp32 across
    launches; the denominator is the whole batch's token count (R10)."""
    import torch
    from paper_2606_26997_b200 import GrpoContext
    assert world == 1 and args.config == 5, "--cgp-mode per_group|batch4 needs --config 5 on one GPU"
    U, n_streams = (1, 1) if args.cgp_mode == "per_group" else (4, 4)
    order = [int(g) for g in b.arrival_order]
    gtok = [b.group_token_range(g)[1] - b.group_token_range(g)[0] for g in order]
    max_launch = max(sum(gtok[i:i + U]) for i in range(0, len(order), U))
    ctx = GrpoContext(b.d, b.V, max_tokens=max_launch, n_slots=n_streams, group_size=b.G, kl_beta=b.kl_beta,
                      clip_lo=b.clip_lo, clip_hi=b.clip_hi, groups_per_update=U, groups_per_round=len(order),
                      **({"stash_logits": 1} if args.stash else {}))
    streams = [torch.cuda.Stream() for _ in range(n_streams)]
    dW = torch.zeros(b.V, b.d, dtype=torch.float32, device=dev)
    loss = torch.zeros(1, dtype=torch.float32, device=dev)
    dH = torch.empty(b.T, b.d, dtype=torch.bfloat16, device=dev)
    descs = []
    for g in order:
        t0, t1 = b.group_token_range(g)
        descs.append(ctx.make_group_desc(g, b.seqlens[g * b.G:(g + 1) * b.G], b.hidden[t0:t1], b.targets[t0:t1],
                                         b.old_logp[t0:t1], b.rewards[g * b.G:(g + 1) * b.G].contiguous(),
                                         None if b.ref_logp is None else b.ref_logp[t0:t1], None, dH[t0:t1], None))

    def step():
        for d_ in descs:
            ctx.grpo_enqueue_groups([d_], b.W, dW, loss, loss_denom=float(b.T), streams=streams)
        if ctx.grpo_queue_state()["pending_groups"]:
            ctx.grpo_flush(b.W, dW, loss, loss_denom=float(b.T), streams=streams)
        ctx.grpo_reset_round()

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    assert ctx.grpo_check_errors_sync() == 0
    sampler = ClockSampler(dev.index or 0)
    n0 = ctx.grpo_kernel_launches()
    sampler.start()
    cur = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(cur)
    for s_ in streams:
        s_.wait_event(e0)
    for _ in range(args.steps):
        step()
    for s_ in streams:
        cur.wait_stream(s_)
    e1.record(cur)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    n1 = ctx.grpo_kernel_launches()
    line = {"metric": METRIC, "value": b.T * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": WORKLOADS[5].replace("as ONE full-batch step", f"streamed through "
                       f"grpo_enqueue_groups: {args.cgp_mode} (U={U}, {n_streams} stream(s))"),
                       "tokens_per_step": b.T, "groups": len(order), "variant": "stash_logits" if args.stash else "recompute"},
            "e2e": None, "gpu_launches": sum(n1.values()) - sum(n0.values()), "clocks": clocks,
            "executed_tflops": (2.0 * b.T * b.V * b.d * (3 if args.stash else 4)) * args.steps / (ms * 1e-3) / 1e12,
            "note": "dense FLOP basis (zero-coefficient tiles are skipped, so this is an upper bound on executed FLOPs)"}
    print(json.dumps(line), flush=True)
    ctx.close()
    return 0


def dp_update_plan(world: int, groups_per_rank: int):
    """The logical update of the --dp arm: world x groups_per_rank complete groups in FIFO order, dealt by position
    (k mod world) as GrpoDataParallel does; returns per rank the update positions it trains (host logic, unit-tested
    under gloo in tests/test_multirank_cpu.py)."""
    from paper_2606_26997_b200.dp import assign_groups
    U = world * groups_per_rank
    return U, [assign_groups(U, world, r) for r in range(world)]


def run_dp(args, dev, rank, world, local):
    """--dp allreduce|stitched (informational): ONE logical update of
    world x k complete groups (configs[1] groups: G = 8, lengths U[512, 4096]) dealt to the ranks by
    GrpoDataParallel; every rank trains its k groups through grpo_enqueue_groups with the update's global
    denominator, then the update boundary reduces dW / loss / metrics over the ranks.  tokens/s INCLUDES the
    reduction: `allreduce` = asynchronous NCCL all-reduce on a side stream into alternating buffer sets (the next
    update's contractions overlap it; --dp-max-ctas leaves SMs to it), `stitched` = the A6 reduce-adds go straight
    into the rank-sharded accumulator (StitchedGradient) and the boundary is a barrier.  With one rank the
    collectives are still issued (always_reduce), so the line measures their fixed cost, not NVLink."""
    import torch
    import torch.distributed as dist
    from paper_2606_26997_b200 import GrpoContext
    from paper_2606_26997_b200.dp import GrpoDataParallel, StitchedGradient
    from workloads.synth import make_config
    k = args.dp_groups
    if world == 1 and not dist.is_initialized():          # a one-rank NCCL group: the real collective calls still run
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29517")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
    U, plan = dp_update_plan(world, k)
    b = make_config(2, seed=rank_seed(rank), device=dev, n_groups=k)      # this rank's k groups of the update
    dp = GrpoDataParallel(always_reduce=True)
    gtok = [b.group_token_range(g)[1] - b.group_token_range(g)[0] for g in range(k)]
    denom = dp.global_denominator(b.T)                                      # token mean over the WHOLE update
    extra = {"gemm_max_ctas": args.dp_max_ctas} if args.dp_max_ctas else {}
    ctx = GrpoContext(b.d, b.V, max_tokens=max(gtok), group_size=b.G, kl_beta=b.kl_beta, clip_lo=b.clip_lo,
                      clip_hi=b.clip_hi, groups_per_update=k, token_budget=max(gtok), **extra)
    dH = torch.empty(b.T, b.d, dtype=torch.bfloat16, device=dev)

    def descs():
        out = []
        for g in range(k):
            t0, t1 = b.group_token_range(g)
            out.append(ctx.make_group_desc(plan[rank][g], b.seqlens[g * b.G:(g + 1) * b.G], b.hidden[t0:t1],
                                           b.targets[t0:t1], b.old_logp[t0:t1],
                                           b.rewards[g * b.G:(g + 1) * b.G].contiguous(),
                                           None if b.ref_logp is None else b.ref_logp[t0:t1], None, dH[t0:t1], None))
        return out

    compute = torch.cuda.current_stream()
    sg = StitchedGradient(ctx, b.V, b.d, dp) if args.dp == "stitched" else None
    loss_s = torch.zeros(1, dtype=torch.float32, device=dev)
    pending = []

    def step():
        if sg is not None:
            loss_s.zero_()
            _, boundary = ctx.grpo_enqueue_groups(descs(), b.W, sg.full, loss_s, loss_denom=denom)
            assert boundary
            sg.barrier()                                   # every rank's reduce-adds have landed: rows are final
            sg.local.zero_()                               # (the optimizer would consume them here)
            return
        dW, loss, metrics = dp.buffers(b.V, b.d, device=dev)
        if len(pending) == 2:                              # the set's previous reduction must have finished
            pending.pop(0).wait(compute)
        dW.zero_(); loss.zero_(); metrics.zero_()
        _, boundary = ctx.grpo_enqueue_groups(descs(), b.W, dW, loss, metrics, loss_denom=denom)
        assert boundary
        pending.append(dp.reduce_boundary(dW, loss, metrics, compute_stream=compute))

    def drain():
        while pending:
            pending.pop(0).wait(compute)

    for _ in range(max(args.warmup, 3)):
        step()
    drain()
    torch.cuda.synchronize()
    dist.barrier()
    assert ctx.grpo_check_errors_sync() == 0
    sampler = ClockSampler(local)
    n0 = ctx.grpo_kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    e0.record()
    for _ in range(args.steps):
        step()
    drain()
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    dist.barrier()
    n1 = ctx.grpo_kernel_launches()
    ms, _, tokens_all = reduce_over_ranks(e0.elapsed_time(e1), 0.0, b.T, world, dev)
    if rank == 0:
        line = {"metric": METRIC, "value": tokens_all * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "informational": "dp",
                "config": {"workload": f"one logical update of U = {U} configs[1]-style complete groups (G = 8, lengths "
                                       f"U[512, 4096], d = {b.d}, V = {b.V}) dealt {k} per rank; boundary reduction "
                                       "INSIDE the timed region",
                           "parallelism": f"dp{world} {args.dp}" + (f", gemm_max_ctas={args.dp_max_ctas}" if args.dp_max_ctas else ""),
                           "tokens_per_step": int(tokens_all), "tokens_rank0": b.T, "groups_per_rank": k,
                           "boundary_bytes_per_rank": 4 * b.V * b.d,
                           "l2": "inputs larger than L2 (W 622 MB, dW 1.2 GB); no flush needed"},
                "e2e": None, "gpu_launches": sum(n1.values()) - sum(n0.values()), "clocks": clocks,
                "note": "world 1: the collectives run in a one-rank NCCL group (fixed cost only); nothing here has "
                        "been timed on more than one GPU" if world == 1 else "max over ranks, device-timed"}
        print(json.dumps(line), flush=True)
    if sg is not None:
        sg.close()
    ctx.close()
    dist.destroy_process_group()
    return 0


def build_line(args, b, world, value, ms_total, e2e_value, h2d, d2h, launches, prof, clocks, peaks, tokens_all,
               loss_val):
    T, d, V = b.T, b.d, b.V
    steps = args.steps
    flops_per_gemm_step = 2.0 * T * V * d                 # each of A2, A4, A5, A6 (rank 0's tokens)
    # the kernels are timed inside a long step (hundreds of ms of back-to-back tensor work), so the
    # denominator is the SUSTAINED measured bf16 matmul rate; the burst figure is reported beside it
    peak = float(peaks.get("bf16_tflops_sustained") or peaks["bf16_tflops"])
    peak_burst = float(peaks["bf16_tflops"])
    kernels = {}
    # executed FLOPs: the backward contractions walk only token tiles with a non-zero coefficient
    act = getattr(args, "bwd_active_frac", 1.0)
    kind_flops = {k: flops_per_gemm_step * (1.0 if k == "gemm_lse" else act) * (prof[k]["launches"] > 0)
                  for k in GEMM_KINDS}
    for k, v in prof.items():
        if v["launches"] == 0:
            continue
        e = {"ms_per_step": v["ms"] / steps, "launches_per_step": v["launches"] / steps}
        if k in GEMM_KINDS:
            e["tflops"] = kind_flops[k] * steps / (v["ms"] * 1e-3) / 1e12
            # --fp8: A2 / A4 run on e4m3 operands; their peak is the measured bf16 peak x the nominal fp8 : bf16
            # ratio of 2 (4.5 vs 2.25 PFLOP/s dense, B200_PROFILING.md)
            k_peak = peak * (2.0 if getattr(args, "fp8", False) and k in ("gemm_lse", "gemm_dz") else 1.0)
            e["frac_of_peak"] = e["tflops"] / k_peak
        if k == "loss" and world == 1 and args.config == 2 and not args.stash:
            # A3 reads / writes >= 56 B per token (one LSE split); launch-latency bound at this size
            e["gbps_at_least"] = 56.0 * T * steps / (v["ms"] * 1e-3) / 1e9
        if k == "stash_dz":     # HBM-bound: 2 B read + 2 B written per logit of the walked rows
            e["gbps"] = 4.0 * T * V * act * steps / (v["ms"] * 1e-3) / 1e9
            e["frac_of_hbm_peak"] = e["gbps"] / float(peaks["hbm_gbs"])
        kernels[k] = e
    gemm_ms = sum(prof[k]["ms"] for k in GEMM_KINDS)
    traffic, traffic_src = load_traffic()
    dom = max(GEMM_KINDS, key=lambda k: prof[k]["ms"])
    dom_tflops = kernels[dom]["tflops"]
    exec_flops = sum(kind_flops.values())
    path_tflops = exec_flops * steps / (gemm_ms * 1e-3) / 1e12
    step_tflops = exec_flops * steps / (ms_total * 1e-3) / 1e12 if world == 1 else None
    prof_total = getattr(args, "profiled_ms_per_step", None)
    gemm_share = gemm_ms / (prof_total * steps) if prof_total else gemm_ms / ms_total
    roofline = {
        "bound": "tensor", "kernel": dom, "achieved": dom_tflops, "peak": peak, "unit": "TFLOP/s",
        "frac": dom_tflops / peak, "traffic": traffic.get(dom), "traffic_source": traffic_src,
        "peak_source": f"{peaks['_source']} bf16_tflops_sustained (MEASURED_PEAKS.json); burst {peak_burst:g}",
        "frac_of_burst": dom_tflops / peak_burst,
        "flops_per_launch": kind_flops[dom] / kernels[dom]["launches_per_step"],
        "all_gemms": {"achieved": path_tflops, "frac": path_tflops / peak, "share_of_step": gemm_share},
        "whole_step": None if step_tflops is None else {"achieved": step_tflops, "frac": step_tflops / peak,
                                                        "flops_basis": "executed: 2*T*V*d (A2) + 2*T_walked*V*d per backward "
                                                                       "contraction (3 recompute / 2 stash); 8*T*V*d for "
                                                                       "the north_star path when no tile is skipped"},
    }
    anchor = getattr(args, "cublas_anchor", None)
    if anchor:
        roofline["same_run_cublas_tflops"] = anchor["tflops"]
        roofline["frac_of_same_run_cublas"] = dom_tflops / anchor["tflops"]
        roofline["all_gemms"]["frac_of_same_run_cublas"] = path_tflops / anchor["tflops"]
        if roofline["whole_step"] is not None:
            roofline["whole_step"]["frac_of_same_run_cublas"] = step_tflops / anchor["tflops"]
        roofline["same_run_cublas"] = anchor
    return {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_total / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "e4m3 (A2, A4 operands) + bf16" if getattr(args, "fp8", False) else "bf16", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config] + (" (informational: --off-policy, old log-prob noise 0.3, "
                                                         "10 % of the tokens masked)" if args.off_policy else "")
                               + (f" (informational: d = {d}, V = {V} instead of the Qwen3-1.7B head)"
                                  if (args.d or args.V) else ""),
                   "variant": "fp8_logits (informational PRECISION STUDY, NEXT-4: e4m3 operands for A2 / A4; does not meet "
                   "north_star's log-prob tolerance)" if args.fp8 else "prenorm (informational, NEXT-4): RMSNorm fwd + north_star path + RMSNorm bwd fused behind A5"
                   if args.prenorm else "stash_logits (3 contractions, DESIGN.md section 11)" if args.stash
                   else "recompute (north_star: 4 contractions)",
                   "tokens_per_step": int(tokens_all), "tokens_rank0": T, "d": d, "V": V, "G": b.G,
                   "parallelism": f"replicas x{world}: independent complete groups, no collective",
                   "l2": "inputs larger than L2 (W 622 MB, dW 1.2 GB, dZ chunk 2.9 GB vs 126 MB L2); no flush needed",
                   "bwd_chunk_tokens": args.bwd_chunk or "library default"},
        "e2e": None if e2e_value is None else {
            "value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
            "api": "grpo_step_host (C ABI, pinned host buffers; W and dW resident on the device)"},
        "bwd_rows": getattr(args, "bwd_rows", None),
        "profiled_ms_per_step": getattr(args, "profiled_ms_per_step", None),
        "energy": getattr(args, "energy", None),
        "other_variant": getattr(args, "other_variant", None),
        "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "kernels": kernels,
        "loss_after_steps": loss_val,
        "paper_context": PAPER_CONTEXT,
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--cta-group", type=int, default=0, choices=[0, 1, 2],
                    help="grpo_config.gemm_cta_group: 0 = library default (CTA pairs), 1 = single-CTA tiles")
    ap.add_argument("--config", type=int, default=2, choices=[2, 3, 4, 5],
                    help="workload = workloads.synth.make_config index (2 = BASELINE configs[1], the headline; "
                         "3-5 are informational device-resident runs without the e2e / cpu_baseline legs)")
    ap.add_argument("--cgp-mode", choices=["full", "per_group", "batch4"], default="full",
                    help="--config 5 only: stream the 32 groups through grpo_enqueue_groups one launch per group "
                         "(per_group) or in 4-group launches on 4 streams (batch4) instead of one full-batch step")
    ap.add_argument("--stash", action="store_true",
                    help="time grpo_fused_logprob_loss_fwd_bwd (3-contraction variant) as the step instead of the "
                         "north_star forward + recomputing backward")
    ap.add_argument("--prenorm", action="store_true",
                    help="informational (NEXT-4): the step starts from pre-norm activations (grpo_rmsnorm_fwd, forward, "
                         "grpo_fused_logprob_loss_bwd_prenorm); no e2e / cpu_baseline legs")
    ap.add_argument("--fp8", action="store_true",
                    help="informational precision study (NEXT-4): grpo_config.fp8_logits = 1 (e4m3 operands for the two "
                         "logit contractions); no e2e / cpu_baseline legs")
    ap.add_argument("--d", type=int, default=0, help="informational: another hidden width (the workload's recipe otherwise)")
    ap.add_argument("--V", type=int, default=0, help="informational: another vocabulary size")
    ap.add_argument("--off-policy", action="store_true",
                    help="informational: the workload in the off-policy regime of config 1b (old log-prob noise 0.3: "
                         "20-40 %% of the tokens clipped; 10 %% masked; no KL), whose zero-coefficient rows the backward "
                         "compacts away (DESIGN.md section 10); no e2e / cpu_baseline legs")
    ap.add_argument("--no-variants", action="store_true", help="do not time the other variant beside the headline")
    ap.add_argument("--no-tile-skip", action="store_true", help="bwd_skip_zero_tiles = off (A/B runs)")
    ap.add_argument("--no-drift-gate", action="store_true", help="gemm_drift_epoch_kb = off (A/B runs)")
    ap.add_argument("--drift-epoch", type=int, default=0, help="gemm_drift_epoch_kb (A/B runs; 0 = library default 32)")
    ap.add_argument("--max-ctas", type=int, default=0, help="grpo_config.gemm_max_ctas (A/B runs; 0 = every SM)")
    ap.add_argument("--bwd-chunk", type=int, default=0, help="grpo_config.bwd_chunk_tokens (0 = library default)")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg (profiling runs)")
    ap.add_argument("--no-energy", action="store_true", help="skip the >= 2 s NVML energy leg (profiling runs)")
    ap.add_argument("--dp", choices=["allreduce", "stitched"], default=None,
                    help="informational multi-GPU arm: one logical update of N x k complete groups dealt by "
                         "GrpoDataParallel, tokens/s including the boundary reduction (DESIGN.md section 7)")
    ap.add_argument("--dp-groups", type=int, default=2, help="--dp: complete groups per rank and update (k)")
    ap.add_argument("--dp-max-ctas", type=int, default=0,
                    help="--dp: gemm_max_ctas of the contraction kernels (leave SMs to the collective); 0 = all SMs")
    ap.add_argument("--no-anchor", action="store_true",
                    help="skip the ~1 s same-run cuBLAS bf16 matmul leg (roofline.same_run_cublas_tflops)")
    ap.add_argument("--power-study", action="store_true",
                    help="informational: the step and cuBLAS on their operands vs all-zero operands (what the data costs "
                         "under the board power cap)")
    ap.add_argument("--sweep-T", action="store_true",
                    help="informational: single-group launches (configs[1] recipe, lengths rescaled) at "
                         "T ~ 2k .. 33k tokens, the range CGP feeds one complete group at a time (PAPER.md:92)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and world == 1 and "RANK" not in os.environ:
        # `python bench.py --gpus N` without a launcher: start one rank per GPU ourselves (the same command the
        # driver uses) and let rank 0 print the line
        import subprocess
        port = 29500 + (os.getpid() % 2000)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        return subprocess.call(cmd)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
