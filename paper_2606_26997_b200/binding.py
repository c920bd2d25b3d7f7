"""ctypes binding of include/grpo.h — argument marshalling only.

Every step of the path runs in libgrpo_b200.so's CUDA kernels.  PyTorch is used for device
memory and streams.  If the library is missing this module raises; there is no fallback.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import torch

from .build import LIB_PATH

GRPO_OK = 0
STATUS_NAMES = {0: "GRPO_OK", 1: "GRPO_ERR_INVALID_ARG", 2: "GRPO_ERR_SHAPE", 3: "GRPO_ERR_WORKSPACE",
                4: "GRPO_ERR_ARCH", 5: "GRPO_ERR_CUDA", 6: "GRPO_ERR_INCOMPLETE_GROUP", 7: "GRPO_ERR_QUEUE_FULL"}

EXPORTS = [
    "grpo_default_config", "grpo_create", "grpo_destroy", "grpo_last_error", "grpo_workspace_bytes",
    "grpo_set_workspace", "grpo_group_advantage", "grpo_fused_logprob_loss_fwd", "grpo_fused_logprob_loss_bwd",
    "grpo_fused_logprob_loss_fwd_bwd", "grpo_set_entropy_out", "grpo_set_seq_denom", "grpo_bwd_row_stats_sync",
    "grpo_rmsnorm_fwd", "grpo_rmsnorm_bwd", "grpo_fused_logprob_loss_bwd_prenorm", "grpo_debug_max_active_clusters",
    "grpo_vocab_shard_partials", "grpo_loss_from_partials", "grpo_loss_from_partials_static",
    "grpo_shard_granularity", "grpo_shard_create", "grpo_shard_import", "grpo_shard_release", "grpo_stitch_map",
    "grpo_stitch_unmap",
    "grpo_enqueue_groups", "grpo_flush", "grpo_queue_state", "grpo_reset_round", "grpo_cgp_plan",
    "grpo_check_errors_sync", "grpo_step_host", "grpo_debug_gemm", "grpo_kernel_launches",
    "grpo_profile_enable", "grpo_profile_read_sync",
]
KERNEL_KINDS = ["advantage", "token_count", "gemm_lse", "loss", "gemm_dz", "gemm_dh", "gemm_dw", "debug", "reserved_8", "stash_dz",
                "compact", "dh_reduce", "rmsnorm", "quantize"]


class GrpoError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


class GrpoConfig(C.Structure):
    _fields_ = [("d", C.c_int32), ("V", C.c_int32), ("eps_std", C.c_float), ("std_ddof", C.c_int32),
                ("clip_lo", C.c_float), ("clip_hi", C.c_float), ("kl_beta", C.c_float), ("loss_agg", C.c_int32),
                ("logit_scale", C.c_float), ("dhidden_fp32", C.c_int32), ("group_size", C.c_int32),
                ("groups_per_update", C.c_int32), ("groups_per_round", C.c_int32), ("token_budget", C.c_int64),
                ("bwd_chunk_tokens", C.c_int64), ("max_pending_groups", C.c_int32), ("gemm_cta_group", C.c_int32),
                ("gemm_drift_epoch_kb", C.c_int32), ("kl_type", C.c_int32), ("dual_clip", C.c_float),
                ("bwd_skip_zero_tiles", C.c_int32), ("stash_logits", C.c_int32), ("fp8_logits", C.c_int32),
                ("gemm_max_ctas", C.c_int32)]


class GroupDesc(C.Structure):
    _fields_ = [("group_order", C.c_int64), ("G", C.c_int32), ("seqlens_host", C.POINTER(C.c_int32)),
                ("hidden", C.c_void_p), ("targets", C.c_void_p), ("old_logp", C.c_void_p), ("ref_logp", C.c_void_p),
                ("mask", C.c_void_p), ("rewards", C.c_void_p), ("dhidden_out", C.c_void_p), ("logp_out", C.c_void_p)]


_LIB = None


def load_library() -> C.CDLL:
    global _LIB
    if _LIB is not None:
        return _LIB
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_26997_b200.build` "
                           "(or __graft_entry__.build()). There is no CPU or PyTorch fallback.")
    lib = C.CDLL(LIB_PATH)
    for name in EXPORTS:
        getattr(lib, name)          # AttributeError if a declared symbol is not exported
    lib.grpo_last_error.restype = C.c_char_p
    for name in EXPORTS:
        if name != "grpo_last_error":
            getattr(lib, name).restype = C.c_int32
    vp, i32, i64, f32, f64 = C.c_void_p, C.c_int32, C.c_int64, C.c_float, C.c_double
    lib.grpo_default_config.argtypes = [C.POINTER(GrpoConfig)]
    lib.grpo_create.argtypes = [C.POINTER(GrpoConfig), C.POINTER(vp)]
    lib.grpo_destroy.argtypes = [vp]
    lib.grpo_workspace_bytes.argtypes = [vp, i64, C.POINTER(i64)]
    lib.grpo_set_workspace.argtypes = [vp, vp, i64, i64, i32]
    lib.grpo_group_advantage.argtypes = [vp, vp, vp, i32, i32, vp, vp, vp]
    lib.grpo_fused_logprob_loss_fwd.argtypes = [vp, vp, vp, vp, vp, i32, i64, vp, vp, vp, vp, f64, vp, vp, vp, vp,
                                                vp, vp]
    lib.grpo_fused_logprob_loss_bwd.argtypes = [vp, vp, vp, vp, vp, vp, i64, f32, vp, vp, vp]
    lib.grpo_fused_logprob_loss_fwd_bwd.argtypes = [vp, vp, vp, vp, vp, i32, i64, vp, vp, vp, vp, f64, f32, vp, vp, vp,
                                                    vp, vp, vp, vp, vp]
    lib.grpo_enqueue_groups.argtypes = [vp, C.POINTER(GroupDesc), i32, vp, vp, vp, vp, f64, C.POINTER(vp), i32,
                                        C.POINTER(i32), C.POINTER(i32)]
    lib.grpo_flush.argtypes = [vp, vp, vp, vp, vp, f64, C.POINTER(vp), i32, C.POINTER(i32), C.POINTER(i32)]
    lib.grpo_queue_state.argtypes = [vp, C.POINTER(i32), C.POINTER(i64), C.POINTER(i32), C.POINTER(i32)]
    lib.grpo_reset_round.argtypes = [vp]
    lib.grpo_cgp_plan.argtypes = [C.POINTER(i64), i32, i32, i64, i32, C.POINTER(i32), i32, C.POINTER(i32)]
    lib.grpo_check_errors_sync.argtypes = [vp, C.POINTER(i32)]
    lib.grpo_step_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, i32, i64, vp, vp, f64, vp, vp, vp, vp]
    lib.grpo_debug_gemm.argtypes = [vp, i32, vp, vp, vp, i32, i32, i32, i32, vp]
    lib.grpo_kernel_launches.argtypes = [vp, C.POINTER(i64)]
    lib.grpo_profile_enable.argtypes = [vp, i32]
    lib.grpo_profile_read_sync.argtypes = [vp, C.POINTER(f64), C.POINTER(i64)]
    lib.grpo_set_entropy_out.argtypes = [vp, vp]
    lib.grpo_set_seq_denom.argtypes = [vp, i32]
    lib.grpo_shard_granularity.argtypes = [vp, C.POINTER(i64)]
    lib.grpo_shard_create.argtypes = [vp, i64, C.POINTER(vp), C.POINTER(i32)]
    lib.grpo_shard_import.argtypes = [vp, i32, i64, C.POINTER(vp)]
    lib.grpo_shard_release.argtypes = [vp, vp]
    lib.grpo_stitch_map.argtypes = [vp, C.POINTER(vp), i32, C.POINTER(vp)]
    lib.grpo_stitch_unmap.argtypes = [vp, vp]
    lib.grpo_vocab_shard_partials.argtypes = [vp, vp, vp, vp, i64, vp, vp, vp, vp]
    lib.grpo_loss_from_partials.argtypes = [vp, i32, vp, vp, vp, vp, i32, vp, i32, i64, vp, vp, vp, vp, f64, vp, vp, vp,
                                            vp, vp, vp]
    lib.grpo_loss_from_partials_static.argtypes = [C.POINTER(GrpoConfig), i32, vp, vp, vp, vp, i32, vp, i32, i32, i64,
                                                   vp, vp, vp, vp, f64, vp, vp, vp, vp, vp, vp, vp]
    lib.grpo_debug_max_active_clusters.argtypes = [vp, i32, C.POINTER(i32)]
    lib.grpo_rmsnorm_fwd.argtypes = [vp, vp, vp, f32, i64, vp, vp, vp]
    lib.grpo_rmsnorm_bwd.argtypes = [vp, vp, vp, vp, vp, i32, i64, vp, vp, vp]
    lib.grpo_fused_logprob_loss_bwd_prenorm.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, i64, f32, vp, vp, vp, vp]
    lib.grpo_bwd_row_stats_sync.argtypes = [vp, C.POINTER(i64), C.POINTER(i64)]
    _LIB = lib
    return lib


def _check(status: int):
    if status != GRPO_OK:
        raise GrpoError(status, load_library().grpo_last_error().decode())


def _dev(t: Optional[torch.Tensor], dtype, name: str, numel: Optional[int] = None):
    if t is None:
        return None
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise TypeError(f"{name}: need a contiguous CUDA tensor of {dtype}, got {t.dtype} on {t.device}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name}: expected {numel} elements, got {t.numel()}")
    return C.c_void_p(t.data_ptr())


def _host(t: Optional[torch.Tensor], dtype, name: str):
    if t is None:
        return None
    if t.is_cuda or not t.is_contiguous() or t.dtype != dtype:
        raise TypeError(f"{name}: need a contiguous CPU tensor of {dtype}")
    return C.c_void_p(t.data_ptr())


def _stream(stream) -> C.c_void_p:
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def grpo_cgp_plan(group_tokens: Sequence[int], U: int, token_budget: int = 0, flush: bool = False):
    """Pure-host planner: launch sizes (in groups) of the next logical update."""
    lib = load_library()
    n = len(group_tokens)
    arr = (C.c_int64 * max(n, 1))(*group_tokens)
    out = (C.c_int32 * max(n, 1))()
    nl = C.c_int32(0)
    _check(lib.grpo_cgp_plan(arr, n, U, token_budget, int(flush), out, max(n, 1), C.byref(nl)))
    return [out[i] for i in range(nl.value)]


STATIC_MAX_TOKENS = 1048576        # GRPO_STATIC_MAX_TOKENS / GRPO_STATIC_MAX_SEQUENCES of include/grpo.h
STATIC_MAX_SEQUENCES = 65536


def grpo_loss_from_partials_static(m2, s2, zy, targets, V_global: int, cu_seqlens, adv, old_logp, out, ref_logp=None,
                                   mask=None, loss_denom: float = 0.0, S_norm: int = 0, err_flags=None, stream=None,
                                   **switches):
    """A3 on gathered vocab-shard partials for callers that cannot allocate GPU memory where they need the loss
    (include/grpo.h, "A3 for callers that must not allocate"): no GrpoContext, no workspace - the kernel's scratch is
    an array built into libgrpo_b200.so - and this function creates no tensor either.  A framework that has given all
    of HBM to its own allocator, a step whose neighbouring streams must not be stalled by cudaMalloc's device
    synchronisation, or a loss-only rank without a vocab shard can call it with buffers it already owns.

    `out` holds the caller's buffers: logp / lse / coeff fp32 [T], loss fp32 [1] (ADDED to), optionally metrics
    fp32 [4] (ADDED to).  `switches` are grpo_config fields (clip_lo, clip_hi, kl_beta, kl_type, dual_clip, loss_agg).
    T <= STATIC_MAX_TOKENS and S <= STATIC_MAX_SEQUENCES, else GrpoError(GRPO_ERR_WORKSPACE).  All calls on one GPU
    share the built-in array: keep them ordered on one stream (or by events); calls that overlap on the GPU race."""
    lib = load_library()
    cfg = GrpoConfig()
    _check(lib.grpo_default_config(C.byref(cfg)))
    for k, v in switches.items():
        if not hasattr(cfg, k):
            raise AttributeError(f"grpo_config has no field {k}")
        setattr(cfg, k, v)
    n_shards, T = m2.shape
    S = cu_seqlens.numel() - 1
    _check(lib.grpo_loss_from_partials_static(
        C.byref(cfg), n_shards, _dev(m2, torch.float32, "m2", n_shards * T), _dev(s2, torch.float32, "s2", n_shards * T),
        _dev(zy, torch.float32, "zy", n_shards * T), _dev(targets, torch.int32, "targets", T), int(V_global),
        _dev(cu_seqlens, torch.int32, "cu_seqlens"), S, int(S_norm), T, _dev(adv, torch.float32, "adv", S),
        _dev(old_logp, torch.float32, "old_logp", T), _dev(ref_logp, torch.float32, "ref_logp", T),
        _dev(mask, torch.uint8, "mask", T), float(loss_denom), _dev(out["logp"], torch.float32, "logp", T),
        _dev(out["lse"], torch.float32, "lse", T), _dev(out["coeff"], torch.float32, "coeff", T),
        _dev(out["loss"], torch.float32, "loss", 1), _dev(out.get("metrics"), torch.float32, "metrics", 4),
        _dev(err_flags, torch.int32, "err_flags", 1), _stream(stream)))
    return out


class GrpoContext:
    """Owns a grpo_ctx and its torch-allocated workspace.  Method names mirror the C calls."""

    def __init__(self, d: int, V: int, *, max_tokens: int = 0, n_slots: int = 1, **overrides):
        self.lib = load_library()
        cfg = GrpoConfig()
        _check(self.lib.grpo_default_config(C.byref(cfg)))
        cfg.d, cfg.V = d, V
        for k, v in overrides.items():
            if not hasattr(cfg, k):
                raise AttributeError(f"grpo_config has no field {k}")
            setattr(cfg, k, v)
        self.cfg = cfg
        h = C.c_void_p()
        _check(self.lib.grpo_create(C.byref(cfg), C.byref(h)))
        self.h = h
        self.workspace = None
        self.max_tokens = 0
        self._keep = []                     # group descriptors queued in the library, FIFO order
        self._inflight = []                 # (events, descriptors) of consumed groups whose launches may still run
        self._consumed_seen = 0
        if max_tokens > 0:
            self.ensure_workspace(max_tokens, n_slots)

    def close(self):
        if getattr(self, "h", None):
            self.lib.grpo_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ workspace
    def workspace_bytes(self, max_T: int) -> int:
        out = C.c_int64(0)
        _check(self.lib.grpo_workspace_bytes(self.h, max_T, C.byref(out)))
        return out.value

    def ensure_workspace(self, max_T: int, n_slots: int = 1):
        if self.workspace is not None and max_T <= self.max_tokens and n_slots <= self.n_slots:
            return
        torch.cuda.synchronize()
        per = self.workspace_bytes(max_T)
        self.workspace = None
        self.workspace = torch.empty(per * n_slots + 256, dtype=torch.uint8, device="cuda")
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        _check(self.lib.grpo_set_workspace(self.h, C.c_void_p(base), per * n_slots, max_T, n_slots))
        self.max_tokens, self.n_slots = max_T, n_slots

    # ------------------------------------------------------------------ A1
    def grpo_group_advantage(self, rewards, G: int = 0, cu_groups=None, n_groups: Optional[int] = None,
                             want_zero_var: bool = False, stream=None):
        """A1 - Eq. 1: A_i = (r_i - mean_g) / (std_g + eps_std), one warp per group (include/grpo.h)."""
        S = rewards.numel()
        if n_groups is None:
            n_groups = (cu_groups.numel() - 1) if cu_groups is not None else S // G
        adv = torch.empty(S, dtype=torch.float32, device=rewards.device)
        zv = torch.empty(n_groups, dtype=torch.uint8, device=rewards.device) if want_zero_var else None
        _check(self.lib.grpo_group_advantage(self.h, _dev(rewards, torch.float32, "rewards"),
                                             _dev(cu_groups, torch.int32, "cu_groups"), n_groups, G,
                                             _dev(adv, torch.float32, "adv"), _dev(zv, torch.uint8, "zero_var"),
                                             _stream(stream)))
        return (adv, zv) if want_zero_var else adv

    # ------------------------------------------------------------------ A2 + A3
    def grpo_fused_logprob_loss_fwd(self, hidden, W, targets, cu_seqlens, adv, old_logp, ref_logp=None, mask=None,
                                    loss_denom: float = 0.0, loss_accum=None, metrics_accum=None, stream=None):
        """A2 + A3 - LM-head contraction with online log-sum-exp, clipped surrogate, optional KL,
        masked mean (loss mask): returns logp / lse / coeff [T] and the accumulated loss (include/grpo.h)."""
        T, d = hidden.shape
        S = cu_seqlens.numel() - 1
        self.ensure_workspace(T, 1)
        dev = hidden.device
        logp = torch.empty(T, dtype=torch.float32, device=dev)
        lse = torch.empty(T, dtype=torch.float32, device=dev)
        coeff = torch.empty(T, dtype=torch.float32, device=dev)
        if loss_accum is None:
            loss_accum = torch.zeros(1, dtype=torch.float32, device=dev)
        _check(self.lib.grpo_fused_logprob_loss_fwd(
            self.h, _dev(hidden, torch.bfloat16, "hidden", T * self.cfg.d), _dev(W, torch.bfloat16, "W", self.cfg.V * self.cfg.d),
            _dev(targets, torch.int32, "targets", T), _dev(cu_seqlens, torch.int32, "cu_seqlens"), S, T,
            _dev(adv, torch.float32, "adv", S), _dev(old_logp, torch.float32, "old_logp", T),
            _dev(ref_logp, torch.float32, "ref_logp", T), _dev(mask, torch.uint8, "mask", T), float(loss_denom),
            _dev(logp, torch.float32, "logp"), _dev(lse, torch.float32, "lse"), _dev(coeff, torch.float32, "coeff"),
            _dev(loss_accum, torch.float32, "loss_accum"), _dev(metrics_accum, torch.float32, "metrics_accum"),
            _stream(stream)))
        return dict(logp=logp, lse=lse, coeff=coeff, loss=loss_accum)

    # ------------------------------------------------------------------ NEXT-3(b): vocab-parallel forward
    def grpo_vocab_shard_partials(self, hidden, W_shard, targets_local, stream=None):
        T = hidden.shape[0]
        self.ensure_workspace(T, 1)
        out = [torch.empty(T, dtype=torch.float32, device=hidden.device) for _ in range(3)]
        _check(self.lib.grpo_vocab_shard_partials(
            self.h, _dev(hidden, torch.bfloat16, "hidden", T * self.cfg.d), _dev(W_shard, torch.bfloat16, "W_shard", self.cfg.V * self.cfg.d),
            _dev(targets_local, torch.int32, "targets_local", T), T, *[_dev(o, torch.float32, "out") for o in out],
            _stream(stream)))
        return tuple(out)

    def grpo_loss_from_partials(self, m2, s2, zy, targets, V_global: int, cu_seqlens, adv, old_logp, ref_logp=None,
                                mask=None, loss_denom: float = 0.0, loss_accum=None, metrics_accum=None, stream=None):
        n_shards, T = m2.shape
        S = cu_seqlens.numel() - 1
        self.ensure_workspace(T, 1)
        dev = m2.device
        logp, lse, coeff = [torch.empty(T, dtype=torch.float32, device=dev) for _ in range(3)]
        if loss_accum is None:
            loss_accum = torch.zeros(1, dtype=torch.float32, device=dev)
        _check(self.lib.grpo_loss_from_partials(
            self.h, n_shards, _dev(m2, torch.float32, "m2", n_shards * T), _dev(s2, torch.float32, "s2", n_shards * T),
            _dev(zy, torch.float32, "zy", n_shards * T), _dev(targets, torch.int32, "targets", T), int(V_global),
            _dev(cu_seqlens, torch.int32, "cu_seqlens"), S, T, _dev(adv, torch.float32, "adv", S),
            _dev(old_logp, torch.float32, "old_logp", T), _dev(ref_logp, torch.float32, "ref_logp", T),
            _dev(mask, torch.uint8, "mask", T), float(loss_denom), _dev(logp, torch.float32, "logp"),
            _dev(lse, torch.float32, "lse"), _dev(coeff, torch.float32, "coeff"), _dev(loss_accum, torch.float32, "loss_accum"),
            _dev(metrics_accum, torch.float32, "metrics_accum"), _stream(stream)))
        return dict(logp=logp, lse=lse, coeff=coeff, loss=loss_accum)

    # ------------------------------------------------------------------ A4 - A6
    def grpo_fused_logprob_loss_bwd(self, hidden, W, targets, lse, coeff, dW_accum=None, grad_scale: float = 1.0,
                                    want_dhidden: bool = True, dhidden_out=None, stream=None):
        """A4 - A6 - recompute the logits chunk by chunk, dZ = coeff (1[v=y] - p), dH = dZ W, dW += dZ^T H
        (north_star; accumulation until the update boundary: PAPER.md:111)."""
        T, d = hidden.shape
        self.ensure_workspace(T, 1)
        if want_dhidden and dhidden_out is None:
            dhidden_out = torch.empty(T, d, dtype=torch.float32 if self.cfg.dhidden_fp32 else torch.bfloat16,
                                      device=hidden.device)
        dh_ptr = None if dhidden_out is None else C.c_void_p(dhidden_out.data_ptr())
        _check(self.lib.grpo_fused_logprob_loss_bwd(
            self.h, _dev(hidden, torch.bfloat16, "hidden"), _dev(W, torch.bfloat16, "W"),
            _dev(targets, torch.int32, "targets", T), _dev(lse, torch.float32, "lse", T),
            _dev(coeff, torch.float32, "coeff", T), T, float(grad_scale), dh_ptr,
            _dev(dW_accum, torch.float32, "dW_accum", self.cfg.V * self.cfg.d), _stream(stream)))
        return dhidden_out

    # ------------------------------------------------------------------ NEXT-4: final RMSNorm in front of the path
    def grpo_rmsnorm_fwd(self, x, gamma, eps_rms: float = 1e-6, stream=None):
        T, d = x.shape
        H = torch.empty(T, d, dtype=torch.bfloat16, device=x.device)
        rstd = torch.empty(T, dtype=torch.float32, device=x.device)
        _check(self.lib.grpo_rmsnorm_fwd(self.h, _dev(x, torch.bfloat16, "x", T * self.cfg.d),
                                         _dev(gamma, torch.bfloat16, "gamma", self.cfg.d), float(eps_rms), T,
                                         _dev(H, torch.bfloat16, "H"), _dev(rstd, torch.float32, "rstd"), _stream(stream)))
        return H, rstd

    def _dx_like(self, x):
        return torch.empty(x.shape, dtype=torch.float32 if self.cfg.dhidden_fp32 else torch.bfloat16, device=x.device)

    def grpo_rmsnorm_bwd(self, x, gamma, rstd, dhidden, dgamma_accum, stream=None):
        T, d = x.shape
        dx = self._dx_like(x)
        if dhidden.dtype not in (torch.float32, torch.bfloat16) or not dhidden.is_contiguous():
            raise TypeError("dhidden: need a contiguous bf16 or fp32 CUDA tensor")
        _check(self.lib.grpo_rmsnorm_bwd(self.h, _dev(x, torch.bfloat16, "x", T * d), _dev(gamma, torch.bfloat16, "gamma", d),
                                         _dev(rstd, torch.float32, "rstd", T), C.c_void_p(dhidden.data_ptr()),
                                         int(dhidden.dtype == torch.float32), T, C.c_void_p(dx.data_ptr()),
                                         _dev(dgamma_accum, torch.float32, "dgamma_accum", d), _stream(stream)))
        return dx

    def grpo_fused_logprob_loss_bwd_prenorm(self, x, gamma, rstd, hidden, W, targets, lse, coeff, dgamma_accum,
                                            dW_accum=None, grad_scale: float = 1.0, stream=None):
        T, d = hidden.shape
        self.ensure_workspace(T, 1)
        dx = self._dx_like(x)
        _check(self.lib.grpo_fused_logprob_loss_bwd_prenorm(
            self.h, _dev(x, torch.bfloat16, "x", T * d), _dev(gamma, torch.bfloat16, "gamma", d),
            _dev(rstd, torch.float32, "rstd", T), _dev(hidden, torch.bfloat16, "hidden", T * d), _dev(W, torch.bfloat16, "W"),
            _dev(targets, torch.int32, "targets", T), _dev(lse, torch.float32, "lse", T),
            _dev(coeff, torch.float32, "coeff", T), T, float(grad_scale), C.c_void_p(dx.data_ptr()),
            _dev(dgamma_accum, torch.float32, "dgamma_accum", d),
            _dev(dW_accum, torch.float32, "dW_accum", self.cfg.V * self.cfg.d), _stream(stream)))
        return dx

    # ------------------------------------------------------------------ A2 - A6 in one call (3-contraction variant)
    def grpo_fused_logprob_loss_fwd_bwd(self, hidden, W, targets, cu_seqlens, adv, old_logp, ref_logp=None, mask=None,
                                        loss_denom: float = 0.0, grad_scale: float = 1.0, loss_accum=None,
                                        metrics_accum=None, dW_accum=None, want_dhidden: bool = True,
                                        dhidden_out=None, stream=None):
        T, d = hidden.shape
        S = cu_seqlens.numel() - 1
        self.ensure_workspace(T, 1)
        dev = hidden.device
        logp = torch.empty(T, dtype=torch.float32, device=dev)
        lse = torch.empty(T, dtype=torch.float32, device=dev)
        coeff = torch.empty(T, dtype=torch.float32, device=dev)
        if loss_accum is None:
            loss_accum = torch.zeros(1, dtype=torch.float32, device=dev)
        if want_dhidden and dhidden_out is None:
            dhidden_out = torch.empty(T, d, dtype=torch.float32 if self.cfg.dhidden_fp32 else torch.bfloat16,
                                      device=dev)
        dh_ptr = None if dhidden_out is None else C.c_void_p(dhidden_out.data_ptr())
        _check(self.lib.grpo_fused_logprob_loss_fwd_bwd(
            self.h, _dev(hidden, torch.bfloat16, "hidden", T * self.cfg.d), _dev(W, torch.bfloat16, "W", self.cfg.V * self.cfg.d),
            _dev(targets, torch.int32, "targets", T), _dev(cu_seqlens, torch.int32, "cu_seqlens"), S, T,
            _dev(adv, torch.float32, "adv", S), _dev(old_logp, torch.float32, "old_logp", T),
            _dev(ref_logp, torch.float32, "ref_logp", T), _dev(mask, torch.uint8, "mask", T), float(loss_denom),
            float(grad_scale), _dev(logp, torch.float32, "logp"), _dev(lse, torch.float32, "lse"),
            _dev(coeff, torch.float32, "coeff"), _dev(loss_accum, torch.float32, "loss_accum"),
            _dev(metrics_accum, torch.float32, "metrics_accum"), dh_ptr,
            _dev(dW_accum, torch.float32, "dW_accum", self.cfg.V * self.cfg.d), _stream(stream)))
        return dict(logp=logp, lse=lse, coeff=coeff, loss=loss_accum, dH=dhidden_out)

    # ------------------------------------------------------------------ A0 / A7
    def make_group_desc(self, order: int, seqlens, hidden, targets, old_logp, rewards, ref_logp=None, mask=None,
                        dhidden_out=None, logp_out=None) -> GroupDesc:
        G = len(seqlens)
        arr = (C.c_int32 * G)(*[int(x) for x in seqlens])
        g = GroupDesc()
        g.group_order, g.G = order, G
        g.seqlens_host = C.cast(arr, C.POINTER(C.c_int32))
        p = lambda t: None if t is None else t.data_ptr()
        g.hidden, g.targets, g.old_logp = p(hidden), p(targets), p(old_logp)
        g.ref_logp, g.mask, g.rewards = p(ref_logp), p(mask), p(rewards)
        g.dhidden_out, g.logp_out = p(dhidden_out), p(logp_out)
        g._keep = (arr, hidden, targets, old_logp, rewards, ref_logp, mask, dhidden_out, logp_out)
        return g

    def _streams(self, streams):
        if not streams:
            streams = [torch.cuda.current_stream()]
        arr = (C.c_void_p * len(streams))(*[s.cuda_stream for s in streams])
        return arr, len(streams)

    # Lifetime of the callers' tensors: a group's tensors must outlive the asynchronous launches that read them.
    # Descriptors wait in `_keep` (FIFO order, like the library's queue) until the library reports them consumed;
    # they then move to `_inflight` behind an event recorded on every launch stream and are dropped once it has
    # completed - so a long-running trainer does not accumulate references to every group it ever enqueued.
    def _retire(self, consumed_total: int, streams):
        n = consumed_total - self._consumed_seen
        self._consumed_seen = consumed_total
        if n > 0:
            done, self._keep = self._keep[:n], self._keep[n:]
            evs = []
            for s in (streams or [torch.cuda.current_stream()]):
                e = torch.cuda.Event()
                e.record(s)
                evs.append(e)
            self._inflight.append((evs, done))
        while self._inflight and all(e.query() for e in self._inflight[0][0]):
            self._inflight.pop(0)

    def grpo_enqueue_groups(self, groups: Sequence[GroupDesc], W, dW_accum, loss_accum, metrics_accum=None,
                            loss_denom: float = 0.0, streams=None):
        """A0 + A7 - append complete groups in arrival order and run one logical update of U groups when
        it is complete, cut into whole-group launches under the token budget; returns
        (groups consumed so far, update boundary reached)."""
        arr = (GroupDesc * max(len(groups), 1))(*groups)
        sarr, ns = self._streams(streams)
        consumed, boundary = C.c_int32(self._consumed_seen), C.c_int32(0)
        pending_before = self.grpo_queue_state()["pending_groups"]
        st = self.lib.grpo_enqueue_groups(self.h, arr, len(groups), _dev(W, torch.bfloat16, "W"),
                                          _dev(dW_accum, torch.float32, "dW_accum"),
                                          _dev(loss_accum, torch.float32, "loss_accum"),
                                          _dev(metrics_accum, torch.float32, "metrics_accum"), float(loss_denom),
                                          sarr, ns, C.byref(consumed), C.byref(boundary))
        # the groups were appended unless the call was rejected before the queue was touched
        if self.grpo_queue_state()["pending_groups"] + (consumed.value - self._consumed_seen) > pending_before:
            self._keep.extend(groups)
        self._retire(consumed.value, streams)
        _check(st)
        return consumed.value, bool(boundary.value)

    def grpo_flush(self, W, dW_accum, loss_accum, metrics_accum=None, loss_denom: float = 0.0, streams=None):
        """End of round: run what is pending (< U groups) as a final short update (Alg. 1 l.16-22)."""
        sarr, ns = self._streams(streams)
        consumed, boundary = C.c_int32(self._consumed_seen), C.c_int32(0)
        st = self.lib.grpo_flush(self.h, _dev(W, torch.bfloat16, "W"), _dev(dW_accum, torch.float32, "dW_accum"),
                                 _dev(loss_accum, torch.float32, "loss_accum"),
                                 _dev(metrics_accum, torch.float32, "metrics_accum"), float(loss_denom), sarr, ns,
                                 C.byref(consumed), C.byref(boundary))
        self._retire(consumed.value, streams)
        _check(st)
        return consumed.value, bool(boundary.value)

    def grpo_queue_state(self):
        pg, pt, cg, rc = C.c_int32(0), C.c_int64(0), C.c_int32(0), C.c_int32(0)
        _check(self.lib.grpo_queue_state(self.h, C.byref(pg), C.byref(pt), C.byref(cg), C.byref(rc)))
        return dict(pending_groups=pg.value, pending_tokens=pt.value, consumed_groups=cg.value,
                    round_complete=bool(rc.value))

    def grpo_reset_round(self):
        _check(self.lib.grpo_reset_round(self.h))
        self._keep.clear()                  # never launched: nothing reads them
        self._consumed_seen = 0             # the library's counter restarts with the round

    def grpo_check_errors_sync(self) -> int:
        f = C.c_int32(0)
        _check(self.lib.grpo_check_errors_sync(self.h, C.byref(f)))
        return f.value

    # ------------------------------------------------------------------ end to end over host buffers
    def grpo_step_host(self, hidden_h, targets_h, cu_seqlens_h, rewards_h, old_logp_h, n_groups: int, G: int, W,
                       dW_accum, ref_logp_h=None, mask_h=None, loss_denom: float = 0.0, loss_h=None, logp_h=None,
                       dhidden_h=None, stream=None):
        """A1 - A6 over HOST buffers in one C-ABI call (H2D, compute, D2H pipelined inside the library): what
        bench.py's e2e leg times."""
        T = hidden_h.shape[0]
        self.ensure_workspace(T, 1)
        if loss_h is None:
            loss_h = torch.zeros(1, dtype=torch.float32).pin_memory()
        dh_ptr = None if dhidden_h is None else C.c_void_p(dhidden_h.data_ptr())
        _check(self.lib.grpo_step_host(
            self.h, _host(hidden_h, torch.bfloat16, "hidden_h"), _host(targets_h, torch.int32, "targets_h"),
            _host(cu_seqlens_h, torch.int32, "cu_seqlens_h"), _host(rewards_h, torch.float32, "rewards_h"),
            _host(old_logp_h, torch.float32, "old_logp_h"), _host(ref_logp_h, torch.float32, "ref_logp_h"),
            _host(mask_h, torch.uint8, "mask_h"), n_groups, G, T, _dev(W, torch.bfloat16, "W"),
            _dev(dW_accum, torch.float32, "dW_accum"), float(loss_denom), _host(loss_h, torch.float32, "loss_h"),
            _host(logp_h, torch.float32, "logp_h"), dh_ptr, _stream(stream)))
        return loss_h

    # ------------------------------------------------------------------ accounting / profiling
    def grpo_kernel_launches(self) -> dict:
        arr = (C.c_int64 * len(KERNEL_KINDS))()
        _check(self.lib.grpo_kernel_launches(self.h, arr))
        return {k: arr[i] for i, k in enumerate(KERNEL_KINDS)}

    def grpo_profile_enable(self, on: bool = True):
        _check(self.lib.grpo_profile_enable(self.h, int(on)))

    def grpo_profile_read_sync(self) -> dict:
        ms = (C.c_double * len(KERNEL_KINDS))()
        n = (C.c_int64 * len(KERNEL_KINDS))()
        _check(self.lib.grpo_profile_read_sync(self.h, ms, n))
        return {k: dict(ms=ms[i], launches=n[i]) for i, k in enumerate(KERNEL_KINDS)}

    def grpo_set_entropy_out(self, entropy_out):
        """entropy_out: fp32 CUDA tensor [>= T of the later forward calls] or None (off)."""
        self._entropy_out = entropy_out          # keep it alive
        _check(self.lib.grpo_set_entropy_out(self.h, _dev(entropy_out, torch.float32, "entropy_out")))

    def grpo_set_seq_denom(self, n_sequences: int):
        _check(self.lib.grpo_set_seq_denom(self.h, int(n_sequences)))

    def grpo_bwd_row_stats_sync(self):
        a, t = C.c_int64(0), C.c_int64(0)
        _check(self.lib.grpo_bwd_row_stats_sync(self.h, C.byref(a), C.byref(t)))
        return a.value, t.value

    # ------------------------------------------------------------------ NEXT-3: stitched dW accumulator (CUDA VMM)
    def grpo_shard_granularity(self) -> int:
        g = C.c_int64(0)
        _check(self.lib.grpo_shard_granularity(self.h, C.byref(g)))
        return g.value

    def grpo_shard_create(self, nbytes: int, export: bool = True):
        sh, fd = C.c_void_p(), C.c_int32(-1)
        _check(self.lib.grpo_shard_create(self.h, int(nbytes), C.byref(sh), C.byref(fd) if export else None))
        return sh, fd.value

    def grpo_shard_import(self, fd: int, nbytes: int):
        sh = C.c_void_p()
        _check(self.lib.grpo_shard_import(self.h, int(fd), int(nbytes), C.byref(sh)))
        return sh

    def grpo_shard_release(self, shard):
        _check(self.lib.grpo_shard_release(self.h, shard))

    def grpo_stitch_map(self, shards) -> int:
        arr = (C.c_void_p * len(shards))(*[s.value for s in shards])
        ptr = C.c_void_p()
        _check(self.lib.grpo_stitch_map(self.h, arr, len(shards), C.byref(ptr)))
        return ptr.value

    def grpo_stitch_unmap(self, ptr: int):
        _check(self.lib.grpo_stitch_unmap(self.h, C.c_void_p(ptr)))

    def grpo_debug_max_active_clusters(self, cluster_size: int) -> int:
        n = C.c_int32(0)
        _check(self.lib.grpo_debug_max_active_clusters(self.h, int(cluster_size), C.byref(n)))
        return n.value

    # ------------------------------------------------------------------ test hook
    def grpo_debug_gemm(self, layout: int, A, B, M: int, N: int, K: int, C_out=None, accumulate: bool = False,
                        stream=None):
        if C_out is None:
            C_out = torch.zeros(M, N, dtype=torch.float32, device=A.device)
        _check(self.lib.grpo_debug_gemm(self.h, layout, _dev(A, torch.bfloat16, "A"), _dev(B, torch.bfloat16, "B"),
                                        _dev(C_out, torch.float32, "C"), M, N, K, int(accumulate), _stream(stream)))
        return C_out
