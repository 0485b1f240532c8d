"""ParameterServerStep: device buffers + the two calls of one step (plumbing only, no arithmetic).

Holds theta / ema / optimizer state, the kept[] / status / t_Nth outputs of the selection kernel and
the device pointer table of the gradient buffers, and enqueues the selection followed by the fused update
(psync_step_device) on one stream with no host synchronisation in between (Alg. 4).

Gradients come either as W flat buffers (set_gradients) or as W*M per-(worker, server) slices -- what each parameter
server receives (set_gradient_slices); per_server=True runs Alg. 4 literally per server j (arrival times [M][W], one
kept row per server).
"""
from __future__ import annotations

from collections import deque
from typing import Optional, Sequence

import numpy as np
import torch

from . import binding as B


class ParameterServerStep:
    def __init__(self, shard_off, N: int, b: int, theta: torch.Tensor, ema: Optional[torch.Tensor],
                 state0: Optional[torch.Tensor], state1: Optional[torch.Tensor], opt: int, ema_mode: int,
                 alpha: float = 0.0, mu: float = 0.0, rho: float = 0.0, eps: float = 0.0, grid_ctas: int = 0,
                 variant: int = 0, per_server: bool = False):
        dev = theta.device
        self.shard_off = np.ascontiguousarray(shard_off, dtype=np.int64)
        self.N, self.b, self.W = N, b, N + b
        self.theta, self.ema, self.state0, self.state1 = theta, ema, state0, state1
        self.opt, self.ema_mode = opt, ema_mode
        self.alpha, self.mu, self.rho, self.eps = alpha, mu, rho, eps
        self.grid_ctas, self.variant = grid_ctas, variant
        self.per_server = bool(per_server)
        self.M = self.shard_off.size - 1
        rows = self.M if per_server else 1
        self.d_kept = torch.full((rows, N) if per_server else (N,), -1, dtype=torch.int32, device=dev)
        self.d_status = torch.full((rows,), B.PSYNC_ECUDA, dtype=torch.int32, device=dev)
        self.d_t_nth = torch.zeros(rows, dtype=torch.float32, device=dev)
        self.d_shard_off = torch.from_numpy(self.shard_off).to(dev)   # the shard-aware kernels read it on the device
        self._d_tiles = {}                                            # work list per gradient dtype, built on demand
        self.layout = B.PSYNC_GRADS_FLAT
        self.table: Optional[B.GradTable] = None
        # A fused kernel in flight stages its pointers from the table it was launched with for its whole lifetime
        # (each CTA reads it at its own start).  Tables replaced by set_gradients() are therefore kept alive for a few
        # steps instead of going straight back to torch's caching allocator, and step() also records the launch stream
        # on the table AND on every gradient tensor it points to (GradTable.record_stream), so a step enqueued on a
        # side stream can never see a block reused under it, however many steps are in flight.
        self._retired = deque(maxlen=4)
        self._step = None
        self._keep = None
        self.d_kept_timeout = None
        self._tstep = None

    def set_gradients(self, buffers: Sequence[torch.Tensor]) -> None:
        if len(buffers) != self.W:
            raise ValueError(f"need W = {self.W} gradient buffers")
        if self.table is not None:
            self._retired.append((self.table, self._keep))
        self.table = B.make_grad_table(buffers)
        self.layout = B.PSYNC_GRADS_FLAT
        self._step = None

    def set_gradient_slices(self, slices: Sequence[Sequence[Optional[torch.Tensor]]]) -> None:
        """slices[k][j] = worker k's G_k[j] (len_j elements, its own tensor; None where server j does not keep worker k)."""
        if len(slices) != self.W or any(len(row) != self.M for row in slices):
            raise ValueError(f"need W = {self.W} rows of M = {self.M} slices")
        if self.table is not None:
            self._retired.append((self.table, self._keep))
        self.table = B.make_slice_table(slices, self.shard_off)
        self.layout = B.PSYNC_GRADS_SLICES
        self._step = None

    def _tiles(self, grad_dtype: int) -> torch.Tensor:
        if grad_dtype not in self._d_tiles:
            self._d_tiles[grad_dtype] = B.psync_shard_worklist(self.d_shard_off, grad_dtype)
        return self._d_tiles[grad_dtype]

    def _build(self, gamma_t: float):
        sharded = self.per_server or self.layout == B.PSYNC_GRADS_SLICES   # the (server, tile) work-list kernel
        self._step, self._keep = B.make_step(
            self.shard_off, self.N, self.W, self.table.grad_dtype, self.theta, self.ema, self.state0, self.state1,
            opt=self.opt, ema_mode=self.ema_mode, gamma_t=gamma_t, alpha=self.alpha, mu=self.mu, rho=self.rho,
            eps=self.eps, d_grads=self.table.d_ptrs, d_kept=self.d_kept, d_status=self.d_status,
            grid_ctas=self.grid_ctas, variant=self.variant, per_shard=self.per_server,
            d_shard_off=self.d_shard_off if sharded else None, grad_layout=self.layout,
            d_tile_start=self._tiles(self.table.grad_dtype) if sharded else None)
        return self._step

    def geometry(self, gamma_t: float = 0.0) -> dict:
        return B.psync_launch_geometry(self._build(gamma_t))

    def step(self, d_arrival: torch.Tensor, gamma_t: float, d_step_tag: Optional[torch.Tensor] = None, t: int = 0,
             stream=None) -> None:
        """Enqueue selection + fused update for one iteration; returns without synchronising.
        d_arrival is [W], or [M][W] with per_server=True (the times at which each server received each gradient)."""
        if self.table is None:
            raise RuntimeError("set_gradients() first")
        if self._step is None or self._step.gamma_t != np.float32(gamma_t):
            self._build(gamma_t)
        self.table.record_stream(stream)    # a side stream reads the pointer table and every gradient tensor
        B.psync_step_device(self._step, d_arrival, self.d_t_nth, d_step_tag, t, stream)   # K1 + K2, one C call

    def aggregate_only(self, gamma_t: float, stream=None) -> None:
        if self._step is None or self._step.gamma_t != np.float32(gamma_t):
            self._build(gamma_t)
        B.psync_aggregate_update(self._step, stream)

    def step_timeout(self, d_arrival: torch.Tensor, timeout: float, gamma_t: float, min_keep: int = 1,
                     d_step_tag: Optional[torch.Tensor] = None, t: int = 0, stream=None) -> None:
        """The time-out rule instead of backup workers: keep every eligible worker that arrived within
        `timeout` seconds, divide by the number kept (per server with per_server=True).  Kept rows land in
        self.d_kept_timeout [rows][W] (first self.d_n_kept[r] entries), status in self.d_status."""
        if self.table is None:
            raise RuntimeError("set_gradients() first")
        rows = self.M if self.per_server else 1
        if getattr(self, "d_kept_timeout", None) is None:
            dev = self.theta.device
            self.d_kept_timeout = torch.full((rows, self.W), -1, dtype=torch.int32, device=dev)
            self.d_n_kept = torch.zeros(rows, dtype=torch.int32, device=dev)
            self._tstep = None
        if self._tstep is None or self._tstep[0].gamma_t != np.float32(gamma_t) or self._tstep[2] is not self.table:
            sharded = self.per_server or self.layout == B.PSYNC_GRADS_SLICES
            st, keep = B.make_step(
                self.shard_off, 1, self.W, self.table.grad_dtype, self.theta, self.ema, self.state0, self.state1,
                opt=self.opt, ema_mode=self.ema_mode, gamma_t=gamma_t, alpha=self.alpha, mu=self.mu, rho=self.rho,
                eps=self.eps, d_grads=self.table.d_ptrs, d_kept=self.d_kept_timeout, d_status=self.d_status,
                per_shard=self.per_server, kept_stride=self.W, d_shard_off=self.d_shard_off if sharded else None,
                d_n_kept=self.d_n_kept, grad_layout=self.layout,
                d_tile_start=self._tiles(self.table.grad_dtype) if sharded else None)
            self._tstep = (st, keep, self.table)
        self.table.record_stream(stream)    # a side stream reads the pointer table and every gradient tensor
        B.psync_select_timeout(d_arrival, self.W, timeout, self.d_kept_timeout, self.d_n_kept, self.d_status, rows=rows,
                               min_keep=min_keep, d_step_tag=d_step_tag, t=t, stream=stream)
        B.psync_aggregate_update(self._tstep[0], stream)


class AsyncServerStep:
    """The Async-SGD parameter server (Alg. 2, L78-89): device buffers + the calls of one batch of arrivals.

    apply(d_arrival) enqueues, with no host synchronisation: the arrival order (per server with per_server=True,
    d_arrival [M][W]), optionally the global-norm clip factors (clip > 0: the norm is over the whole gradient of a
    worker, all of its slices, L313), optionally the learning rates of this batch's iterations (lr = (gamma0, beta, s):
    gamma0 * beta^((t + i) s), L315, with t = the number of gradients applied so far, counted on the device in
    d_t_sched -- a batch in which K < W gradients arrived advances it by K; apply(t0=...) restarts it), the one-pass application of the arrivals, and with track_staleness=True Table 1's
    bookkeeping (per server with per_server=True).  Plumbing only, no arithmetic."""

    def __init__(self, shard_off, W: int, theta: torch.Tensor, ema: Optional[torch.Tensor],
                 state0: Optional[torch.Tensor], state1: Optional[torch.Tensor], opt: int, ema_mode: int = B.PSYNC_EMA_PRE,
                 alpha: float = 0.0, mu: float = 0.0, rho: float = 0.0, eps: float = 0.0, per_server: bool = False,
                 clip: float = 0.0, lr=None, track_staleness: bool = False, lag: int = 0):
        dev = theta.device
        self.shard_off = np.ascontiguousarray(shard_off, dtype=np.int64)
        self.M, self.W = self.shard_off.size - 1, W
        self.theta, self.ema, self.state0, self.state1 = theta, ema, state0, state1
        self.opt, self.ema_mode = opt, ema_mode
        self.alpha, self.mu, self.rho, self.eps = alpha, mu, rho, eps
        self.per_server, self.clip, self.lr, self.lag = bool(per_server), float(clip), lr, int(lag)
        rows = self.M if per_server else 1
        self.d_order = torch.full((rows, W), -1, dtype=torch.int32, device=dev)
        self.d_n_arrived = torch.zeros(rows, dtype=torch.int32, device=dev)
        self.d_shard_off = torch.from_numpy(self.shard_off).to(dev)
        self.d_gamma = torch.zeros(W, dtype=torch.float32, device=dev) if lr is not None else None
        self.d_gscale = torch.ones(W, dtype=torch.float32, device=dev) if clip > 0 else None
        self._d_clip_work = None
        # iterations applied so far, for the schedule (L315): a DEVICE counter, advanced before each batch by the number
        # of gradients the previous batch really applied (d_n_arrived), so a partial batch does not run the schedule ahead
        self.d_t_sched = torch.zeros(1, dtype=torch.int64, device=dev)
        self.track_staleness = bool(track_staleness)
        if track_staleness:               # one row per server with per_server=True: every server counts its own updates
            self.d_read_iter = torch.zeros((rows, W), dtype=torch.int64, device=dev)
            self.d_t = torch.zeros(rows, dtype=torch.int64, device=dev)
            self.d_staleness = torch.zeros((rows, W), dtype=torch.int64, device=dev)
            self.d_stale_stats = torch.zeros((rows, 6), dtype=torch.float64, device=dev)
            self.d_stale_status = torch.zeros(rows, dtype=torch.int32, device=dev)
        self._d_tiles = {}
        self.layout = B.PSYNC_GRADS_FLAT
        self.table: Optional[B.GradTable] = None
        self._retired = deque(maxlen=4)   # tables of batches that may still be in flight (ParameterServerStep's note)
        self._step = None
        self._keep = None

    def set_gradients(self, buffers: Sequence[torch.Tensor]) -> None:
        if len(buffers) != self.W:
            raise ValueError(f"need W = {self.W} gradient buffers")
        if self.table is not None:
            self._retired.append((self.table, self._keep))
        self.table, self.layout, self._step = B.make_grad_table(buffers), B.PSYNC_GRADS_FLAT, None

    def set_gradient_slices(self, slices: Sequence[Sequence[Optional[torch.Tensor]]]) -> None:
        if len(slices) != self.W or any(len(row) != self.M for row in slices):
            raise ValueError(f"need W = {self.W} rows of M = {self.M} slices")
        if self.clip > 0 and any(t is None and self.shard_off[j + 1] > self.shard_off[j]
                                 for row in slices for j, t in enumerate(row)):
            raise ValueError("global-norm clipping needs every slice of every worker (the norm is over all of them)")
        if self.table is not None:
            self._retired.append((self.table, self._keep))
        self.table, self.layout, self._step = B.make_slice_table(slices, self.shard_off), B.PSYNC_GRADS_SLICES, None

    def _build(self, gamma_t: float):
        sharded = self.per_server or self.layout == B.PSYNC_GRADS_SLICES
        gd = self.table.grad_dtype
        if sharded and gd not in self._d_tiles:
            self._d_tiles[gd] = B.psync_shard_worklist(self.d_shard_off, gd)
        self._step, self._keep = B.make_step(
            self.shard_off, self.W, self.W, gd, self.theta, self.ema, self.state0, self.state1, opt=self.opt,
            ema_mode=self.ema_mode, gamma_t=gamma_t, alpha=self.alpha, mu=self.mu, rho=self.rho, eps=self.eps,
            d_grads=self.table.d_ptrs, d_kept=self.d_order, per_shard=self.per_server,
            d_shard_off=self.d_shard_off if sharded else None, d_n_kept=self.d_n_arrived, kept_stride=self.W,
            grad_layout=self.layout, d_tile_start=self._d_tiles[gd] if sharded else None)
        return self._step

    def apply(self, d_arrival: torch.Tensor, gamma_t: float = 0.0, t0: Optional[int] = None, stream=None) -> None:
        """One batch: every gradient whose arrival time is finite is one iteration, in arrival order (L85-87).
        t0 (optional) restarts the schedule's iteration counter at that value for this batch."""
        if self.table is None:
            raise RuntimeError("set_gradients() first")
        if self._step is None or self._step.gamma_t != np.float32(gamma_t):
            self._build(gamma_t)
        self.table.record_stream(stream)    # a side stream reads the pointer table and every gradient tensor
        if self.clip > 0:                 # norms and rates do not depend on the order: they are enqueued first
            sliced = self.layout == B.PSYNC_GRADS_SLICES
            key = (sliced, self.table.grad_dtype)
            if self._d_clip_work is None or self._d_clip_work[0] != key:
                nbytes = (B.psync_clip_slices_workspace_bytes(self.W, self.shard_off, self.table.grad_dtype) if sliced
                          else B.psync_clip_workspace_bytes(self.W, self.theta.numel(), self.table.grad_dtype))
                self._d_clip_work = (key, torch.empty((nbytes + 7) // 8, dtype=torch.float64, device=self.theta.device))
            if sliced:
                B.psync_clip_scales_slices(self.table, self.shard_off, self.d_shard_off, self.clip, self.d_gscale,
                                           self._d_clip_work[1], stream)
            else:
                B.psync_clip_scales(self.table, self.clip, self.d_gscale, self._d_clip_work[1], stream)
        if self.lr is not None:
            gamma0, beta, s = self.lr
            B.psync_lr_schedule_counted(gamma0, beta, self.d_t_sched, self.W, s, self.d_gamma, d_n_add=self.d_n_arrived,
                                        t_set=-1 if t0 is None else int(t0), stream=stream)   # before this batch's order
        B.psync_async_step_device(self._step, d_arrival, self.d_gamma, stream, d_gscale=self.d_gscale)   # order + K iterations
        if self.track_staleness:
            B.psync_staleness_sharded(self.d_read_iter, self.d_order, self.d_t, self.d_staleness, self.d_stale_stats,
                                      self.d_stale_status, d_n_arrived=self.d_n_arrived, lag=self.lag, stream=stream)
