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
        # on the table, so a step enqueued on a side stream can never see its table's block reused under it.
        self._retired = deque(maxlen=4)
        self._step = None
        self._keep = None

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
        self.table = B.make_slice_table(slices)
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
        if stream is not None and hasattr(stream, "cuda_stream"):
            self.table.d_ptrs.record_stream(stream)
        B.psync_step_device(self._step, d_arrival, self.d_t_nth, d_step_tag, t, stream)   # K1 + K2, one C call

    def aggregate_only(self, gamma_t: float, stream=None) -> None:
        if self._step is None or self._step.gamma_t != np.float32(gamma_t):
            self._build(gamma_t)
        B.psync_aggregate_update(self._step, stream)
