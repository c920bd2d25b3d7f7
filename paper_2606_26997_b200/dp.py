"""Data parallelism over complete groups.

Complete groups are independent units of work, and the paper's trainer ran DP = 2.
A logical update of U groups is dealt to the ranks by arrival position (group k of the update ->
rank k mod world); every rank runs A1-A6 on its groups through ``grpo_enqueue_groups`` with the denominator of the
WHOLE update (R10: ``loss_denom=global_denominator(...)`` for the token mean; for ``loss_agg = 1``
``ctx.grpo_set_seq_denom(global_sequences(...))`` before enqueueing), accumulating into its local fp32 ``dW`` / loss; at the update boundary ONE sum
all-reduce of ``dW`` (1.245 GB at the Qwen3-1.7B head) plus the scalars gives every rank the full-update gradient:
by the additivity of the step over groups (P12) the result equals the single-rank full-batch step up to fp32
summation order.

The all-reduce is issued on a side stream behind an event of the compute stream and returns immediately, so it
overlaps with the next update's contractions, which accumulate into the OTHER of two gradient buffers
(``buffers()`` hands them out alternately).  ``torch.distributed`` is plumbing only (NCCL over NVLink 5 on the GPU
box; gloo in the CPU tests): no arithmetic of the method lives here.  Every branch has run on ONE GPU (a one-rank
NCCL group, tests/test_dp_gpu.py); nothing in this module has run or been timed on more than one GPU (none is
reachable from this build); DESIGN.md section 7 says so.
"""
from __future__ import annotations

import math
import os
import socket
import threading
import uuid
from dataclasses import dataclass, field
from typing import List, Optional

import torch
import torch.distributed as dist


def assign_groups(n_groups_in_update: int, world: int, rank: int) -> List[int]:
    """Positions (within the update, in FIFO order) of the groups rank `rank` trains: k with k mod world == rank."""
    return [k for k in range(n_groups_in_update) if k % world == rank]


@dataclass
class BoundaryHandle:
    """Outstanding reduction of one logical update's accumulators."""
    works: list = field(default_factory=list)
    done_event: Optional["torch.cuda.Event"] = None

    def wait(self, stream: Optional["torch.cuda.Stream"] = None):
        """Make `stream` (default: the current stream) wait for the reduced gradients; on CPU, block."""
        for w in self.works:
            w.wait()
        if self.done_event is not None:
            (stream or torch.cuda.current_stream()).wait_event(self.done_event)


class GrpoDataParallel:
    """always_reduce: issue the collectives even when the group has ONE rank (they are then identities).  A single
    GPU can host a one-rank NCCL group, so this is how the CUDA / NCCL branches below are executed where no second
    GPU is reachable (tests/test_dp_gpu.py); leave it off in production."""

    def __init__(self, process_group=None, comm_stream: Optional["torch.cuda.Stream"] = None,
                 always_reduce: bool = False):
        self.pg = process_group
        self.always_reduce = always_reduce
        self.world = dist.get_world_size(process_group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(process_group) if dist.is_initialized() else 0
        self._comm_stream = comm_stream
        self._buf = None
        self._turn = 0

    # ------------------------------------------------------------------ work split
    def local_positions(self, n_groups_in_update: int) -> List[int]:
        return assign_groups(n_groups_in_update, self.world, self.rank)

    def global_denominator(self, local_loss_tokens: int) -> float:
        """Loss-bearing tokens of the WHOLE update (token-mean denominator, R10): sum over ranks of the
        local counts (host integers: the sequence lengths are host data in the CGP handoff)."""
        if self.world == 1 and not self.always_reduce:
            return float(local_loss_tokens)
        t = torch.tensor([float(local_loss_tokens)], dtype=torch.float64)
        if dist.get_backend(self.pg) == "nccl":
            t = t.cuda()
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.pg)
        return float(t.item())

    def global_sequences(self, local_sequences: int) -> int:
        """Sequences of the whole update (loss_agg = 1 divides by it; ``GrpoContext.grpo_set_seq_denom``)."""
        return int(round(self.global_denominator(local_sequences)))

    # ------------------------------------------------------------------ double-buffered accumulators
    def buffers(self, V: int, d: int, device="cuda"):
        """(dW, loss, metrics) of the update about to be trained; alternates between two sets so that the previous
        update's all-reduce can still be in flight.  The caller zeroes a set after consuming it."""
        if self._buf is None:
            mk = lambda: (torch.zeros(V, d, dtype=torch.float32, device=device),
                          torch.zeros(1, dtype=torch.float32, device=device),
                          torch.zeros(4, dtype=torch.float32, device=device))
            self._buf = (mk(), mk())
        out = self._buf[self._turn]
        self._turn ^= 1
        return out

    # ------------------------------------------------------------------ the collective
    def reduce_boundary(self, dW_accum: torch.Tensor, loss_accum: torch.Tensor,
                        metrics_accum: Optional[torch.Tensor] = None,
                        compute_stream: Optional["torch.cuda.Stream"] = None) -> BoundaryHandle:
        """Sum `dW_accum`, `loss_accum` (and `metrics_accum`) over the ranks, in place, asynchronously.

        CUDA tensors: the collectives are enqueued on the side stream behind an event recorded on `compute_stream`
        (default: current), so everything the update's launches enqueued is reduced, and the call returns at once:
        the next update's kernels run concurrently.  CPU tensors (gloo tests): asynchronous works."""
        tensors = [t for t in (dW_accum, loss_accum, metrics_accum) if t is not None]
        h = BoundaryHandle()
        if self.world == 1 and not self.always_reduce:
            return h
        if dW_accum.is_cuda:
            if self._comm_stream is None:
                self._comm_stream = torch.cuda.Stream()
            ev = torch.cuda.Event()
            ev.record(compute_stream or torch.cuda.current_stream())
            with torch.cuda.stream(self._comm_stream):
                self._comm_stream.wait_event(ev)
                for t in tensors:
                    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.pg)
                h.done_event = torch.cuda.Event()
                h.done_event.record(self._comm_stream)
        else:
            for t in tensors:
                h.works.append(dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.pg, async_op=True))
        return h


# ---------------------------------------------------------------------- vocab (tensor) parallel
def vocab_shard_bounds(V: int, world: int, multiple: int = 8) -> List[int]:
    """Row bounds [v_0 = 0, v_1, ..., v_world = V] of the vocab shards: as even as possible, every inner bound a
    multiple of `multiple` rows (keeps every shard 16-byte aligned for TMA whatever d is)."""
    if world < 1 or V < world:
        raise ValueError(f"cannot cut V={V} rows into {world} shards")
    bounds = [0]
    for r in range(1, world):
        b = (V * r // world) // multiple * multiple
        bounds.append(max(b, bounds[-1] + 1))
    bounds.append(V)
    return bounds


class GrpoVocabParallel:
    """Vocab-parallel (tensor-parallel) GRPO step (the paper's trainer ran TP = 4,
    PAPER.md:197, which cuts the LM head by vocabulary rows).  Rank r owns rows [v0, v1) of W and of dW and a context
    created with V = v1 - v0.  EVERY rank holds the same packed batch (hidden, targets, rewards, ...) - with TP the
    transformer body's output is replicated - and after ``step`` every rank holds the same loss, metrics, logp and
    the full dHidden; dW stays sharded by rows.

    The exchange is two collectives per step: ONE all-gather of the per-token partials ([3, T] fp32 per rank:
    running max, sum of 2^(z - max), target logit) and ONE sum all-reduce of the partial dHidden ([T, d] fp32).
    Everything else runs in the library's kernels; this class only moves buffers (torch.distributed: NCCL on a GPU
    box, gloo in the tests).  The loss / metrics accumulators are REPLICATED, never summed over the TP group.  Not
    run or timed on more than one GPU."""

    def __init__(self, d: int, V_global: int, process_group=None, make_context: bool = True,
                 always_reduce: bool = False, **ctx_kw):
        self.pg = process_group
        self.always_reduce = always_reduce            # issue the collectives even in a one-rank group (tests)
        self.world = dist.get_world_size(process_group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(process_group) if dist.is_initialized() else 0
        self.d, self.V_global = d, V_global
        self.bounds = vocab_shard_bounds(V_global, self.world)
        self.v0, self.v1 = self.bounds[self.rank], self.bounds[self.rank + 1]
        self.ctx = None
        if make_context:
            from .binding import GrpoContext
            ctx_kw.setdefault("dhidden_fp32", 1)          # the partial dHidden is summed over ranks: keep it fp32
            if not ctx_kw["dhidden_fp32"]:
                raise ValueError("GrpoVocabParallel sums partial dHidden over ranks and needs dhidden_fp32=1")
            self.ctx = GrpoContext(d, self.v1 - self.v0, **ctx_kw)

    def close(self):
        if self.ctx is not None:
            self.ctx.close()
            self.ctx = None

    # ------------------------------------------------------------------ buffer plumbing
    def shard_rows(self, W_full: torch.Tensor) -> torch.Tensor:
        """This rank's rows of a full [V, d] matrix (a copy, contiguous)."""
        return W_full[self.v0:self.v1].contiguous()

    def local_targets(self, targets: torch.Tensor) -> torch.Tensor:
        """Shard-local target ids: y - v0; ignored tokens (y < 0) stay ignored in every shard.  Ids that land outside
        [0, v1 - v0) simply have no one-hot entry in this shard (include/grpo.h)."""
        shifted = targets - self.v0
        return torch.where(targets < 0, torch.full_like(targets, -1), shifted).contiguous()

    def gather_partials(self, m2: torch.Tensor, s2: torch.Tensor, zy: torch.Tensor):
        """ONE all-gather of this rank's [3, T] partials -> three contiguous [world, T] arrays in shard order, the
        layout grpo_loss_from_partials reads."""
        T = m2.numel()
        mine = torch.stack((m2, s2, zy)).contiguous()                                # [3, T]
        if self.world == 1 and not self.always_reduce:
            everyone = mine.unsqueeze(0)
        else:
            flat = torch.empty(self.world * 3, T, dtype=mine.dtype, device=mine.device)    # ranks concatenated on dim 0
            dist.all_gather_into_tensor(flat, mine, group=self.pg)
            everyone = flat.view(self.world, 3, T)
        by_kind = everyone.permute(1, 0, 2).contiguous()                             # [3, world, T]
        return by_kind[0], by_kind[1], by_kind[2]

    def reduce_dhidden(self, dH_partial: torch.Tensor) -> torch.Tensor:
        """Sum of the ranks' partial dHidden, in place."""
        if self.world > 1 or self.always_reduce:
            dist.all_reduce(dH_partial, op=dist.ReduceOp.SUM, group=self.pg)
        return dH_partial

    # ------------------------------------------------------------------ the step
    def step(self, hidden, W_shard, targets, cu_seqlens, rewards, G: int, old_logp, ref_logp=None, mask=None,
             dW_shard_accum=None, loss_accum=None, metrics_accum=None, loss_denom: float = 0.0,
             grad_scale: float = 1.0):
        """A1 -> A2 on the shard -> all-gather -> A3 -> A4-A6 on the shard -> all-reduce of dHidden.
        targets are GLOBAL ids.  Returns logp / lse / coeff / loss (replicated), dH (full, fp32) and adds the
        shard's rows of dW into dW_shard_accum ([v1 - v0, d] fp32)."""
        ctx = self.ctx
        y_loc = self.local_targets(targets)
        m2, s2, zy = ctx.grpo_vocab_shard_partials(hidden, W_shard, y_loc)
        m2g, s2g, zyg = self.gather_partials(m2, s2, zy)
        adv = ctx.grpo_group_advantage(rewards, G=G)
        f = ctx.grpo_loss_from_partials(m2g, s2g, zyg, targets, self.V_global, cu_seqlens, adv, old_logp, ref_logp,
                                        mask, loss_denom=loss_denom, loss_accum=loss_accum,
                                        metrics_accum=metrics_accum)
        dH = ctx.grpo_fused_logprob_loss_bwd(hidden, W_shard, y_loc, f["lse"], f["coeff"], dW_accum=dW_shard_accum,
                                             grad_scale=grad_scale)
        f["dH"] = self.reduce_dhidden(dH)
        f["adv"] = adv
        return f


# ---------------------------------------------------------------------- fused GEMM -> reduce-scatter (stitched dW)
class _RawCudaBuffer:
    """A raw device range exposed through __cuda_array_interface__ so that torch can alias it."""

    def __init__(self, ptr: int, n_float32: int):
        self.__cuda_array_interface__ = {"shape": (n_float32,), "typestr": "<f4", "data": (ptr, False), "version": 2}


def _node_identity() -> str:
    """Something every process on one machine agrees on, containers included (the kernel's boot id), else the
    hostname."""
    try:
        with open("/proc/sys/kernel/random/boot_id") as f:
            return f.read().strip()
    except OSError:
        return socket.gethostname()


def _require_one_node(dp: "GrpoDataParallel", identity: Optional[str] = None, device: Optional[int] = None):
    """The stitched accumulator needs (1) every rank on ONE machine - shard handles travel as file descriptors over
    Unix sockets - and (2) peer access between the ranks' GPUs, since the A6 reduce-adds are NVLink stores into the
    peers' memory.  Raises on EVERY rank (the facts are all-gathered) instead of hanging in connect() or faulting in
    the kernel.  GPUs hidden behind per-rank CUDA_VISIBLE_DEVICES all read as device 0 here and cannot be checked:
    cuMemSetAccess in grpo_stitch_map then reports the missing access."""
    if device is None:
        device = torch.cuda.current_device() if torch.cuda.is_available() else -1
    me = (identity if identity is not None else _node_identity(), int(device))
    everyone = [None] * dp.world
    dist.all_gather_object(everyone, me, group=dp.pg)
    nodes = sorted({n for n, _ in everyone})
    if len(nodes) > 1:
        raise RuntimeError(f"StitchedGradient needs all {dp.world} ranks on one node (shard handles are POSIX file "
                           f"descriptors passed over Unix sockets); the group spans {len(nodes)} nodes. Use "
                           "GrpoDataParallel.reduce_boundary (all-reduce) across nodes.")
    if me[1] >= 0:
        for r, (_, dev_r) in enumerate(everyone):
            if r != dp.rank and dev_r >= 0 and dev_r != me[1] and not torch.cuda.can_device_access_peer(me[1], dev_r):
                raise RuntimeError(f"StitchedGradient: GPU {me[1]} (rank {dp.rank}) has no peer access to GPU {dev_r} "
                                   f"(rank {r}); the stitched accumulator needs NVLink / P2P between all ranks.")


def _exchange_fds(own_fd: int, dp: "GrpoDataParallel") -> List[int]:
    """Every rank's exported shard descriptor, by rank (own at dp.rank).  POSIX file descriptors only cross process
    boundaries as SCM_RIGHTS ancillary data: every rank serves its descriptor on a Unix socket, then fetches the
    others'.  One node only: checked first (_require_one_node)."""
    if dp.world == 1:
        return [own_fd]
    _require_one_node(dp)
    tag = [uuid.uuid4().hex if dp.rank == 0 else None]
    dist.broadcast_object_list(tag, src=0, group=dp.pg)
    path = lambda r: f"/tmp/grpo_stitch_{tag[0]}_{r}.sock"
    srv = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
    srv.bind(path(dp.rank))
    srv.listen(dp.world)

    def serve():
        for _ in range(dp.world - 1):
            conn, _ = srv.accept()
            socket.send_fds(conn, [b"fd"], [own_fd])
            conn.close()

    th = threading.Thread(target=serve, daemon=True)
    th.start()
    dist.barrier(group=dp.pg)                      # every socket is listening
    fds = []
    for r in range(dp.world):
        if r == dp.rank:
            fds.append(own_fd)
            continue
        c = socket.socket(socket.AF_UNIX, socket.SOCK_STREAM)
        c.connect(path(r))
        _, got, _, _ = socket.recv_fds(c, 16, 1)
        c.close()
        fds.append(got[0])
    th.join()
    srv.close()
    os.unlink(path(dp.rank))
    return fds


class StitchedGradient:
    """fp32 [V, d] gradient accumulator whose row range r R .. (r+1) R physically lives on rank r's GPU
    (include/grpo.h: grpo_shard_* / grpo_stitch_*).  Passed as ``dW_accum`` it makes the A6 epilogue's reduce-adds
    the data-parallel reduce-scatter: no collective follows the GEMM.  ``full`` is the [V, d] view every rank
    accumulates into, ``local`` the rank's own (fully reduced after ``barrier()``) rows, ``local_rows`` their range.

    n_local_shards > 0 builds the same layout from that many chunks of THIS process's GPU (one-GPU emulation)."""

    def __init__(self, ctx, V: int, d: int, dp: Optional[GrpoDataParallel] = None, n_local_shards: int = 0):
        self.ctx, self.dp = ctx, dp
        n = n_local_shards if n_local_shards > 0 else (dp.world if dp else 1)
        rank = 0 if n_local_shards > 0 or dp is None else dp.rank
        gran, row_bytes = ctx.grpo_shard_granularity(), 4 * d
        unit = gran * row_bytes // math.gcd(gran, row_bytes) // row_bytes      # rows per shard come in these units
        self.rows_per_shard = -(-(-(-V // n)) // unit) * unit
        nbytes = self.rows_per_shard * row_bytes
        if n_local_shards > 0:
            self._shards = [ctx.grpo_shard_create(nbytes, export=False)[0] for _ in range(n)]
        else:
            own, fd = ctx.grpo_shard_create(nbytes)
            fds = _exchange_fds(fd, dp) if dp else [fd]
            self._shards = [own if r == rank else ctx.grpo_shard_import(fds[r], nbytes) for r in range(n)]
            for f in set(fds):
                os.close(f)
        self._ptr = ctx.grpo_stitch_map(self._shards)
        flat = torch.as_tensor(_RawCudaBuffer(self._ptr, n * self.rows_per_shard * d), device="cuda")
        self._all = flat.view(n * self.rows_per_shard, d)
        self.full = self._all[:V]
        self.local_rows = (rank * self.rows_per_shard, min(V, (rank + 1) * self.rows_per_shard))
        self.local = self._all[rank * self.rows_per_shard:(rank + 1) * self.rows_per_shard]
        self.local.zero_() if n_local_shards == 0 else self._all.zero_()
        self.barrier()

    def barrier(self):
        """All ranks' launches into the accumulator have completed (device + host barrier)."""
        torch.cuda.synchronize()
        if self.dp is not None and self.dp.world > 1:
            dist.barrier(group=self.dp.pg)

    def close(self):
        if getattr(self, "_ptr", None):
            self.full = self.local = self._all = None
            self.ctx.grpo_stitch_unmap(self._ptr)
            for s in self._shards:
                self.ctx.grpo_shard_release(s)
            self._ptr = None
