"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json:configs; recipe in DESIGN.md).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: it only draws parameters, gradients, arrival times and shard cuts.  Both
sides always consume the same bytes (the oracle gets device-generated data by D2H copy), so
parity never depends on reproducing a random stream twice.

The paper measures on ImageNet/Inception, CIFAR-10/PixelCNN and MNIST (PAPER.md:L99, L223, L235,
L299).  None of those is available or needed: the parameter-server step is data-oblivious, so
gradients with the configs' shapes and distributions stand in for them, and the arrival times
stand in for the measured distribution of PAPER.md:L171-179 (tight lognormal body, rare long tail).
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Optional

import numpy as np
import torch

MASTER_SEED = 170205800
STREAM_GRAD, STREAM_ARRIVAL, STREAM_INIT = 0, 1, 2

# enum values of include/psync.h (plain integers; no arithmetic here)
F32, BF16 = 0, 1
SGD, MOMENTUM, RMSPROP_MOM = 0, 1, 2
EMA_POST, EMA_PRE, EMA_OFF = 0, 1, 2


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config.  Notation follows the paper: N, b, M, gamma, alpha."""
    name: str
    cfg_id: int
    P: int
    M: int
    N: int
    b: int
    grad_dtype: int = F32
    theta_dist: tuple = ("normal", 0.02)      # ("normal", std) | ("uniform", half_width)
    grad_dist: tuple = ("normal", 1e-3)
    arrival_sigma: float = 0.25               # arrival = exp(sigma * z)
    delay_prob: float = 0.0                   # independent Bernoulli per worker per step
    delay_factor: float = 1.0
    opt: int = SGD
    gamma: float = 0.045
    alpha: float = 0.9999
    mu: float = 0.0
    rho: float = 0.0
    eps: float = 0.0
    ms0: float = 1.0                          # RMSProp second-moment initial value (reading R5)
    steps: int = 1
    ragged: bool = True                       # seeded uneven shard sizes; False -> equal cuts
    ema_mode: int = EMA_POST

    @property
    def W(self) -> int:
        return self.N + self.b

    @property
    def n_state(self) -> int:
        return {SGD: 0, MOMENTUM: 1, RMSPROP_MOM: 2}[self.opt]

    @property
    def grad_bytes(self) -> int:
        return 4 if self.grad_dtype == F32 else 2

    @property
    def bytes_per_element(self) -> int:
        """north_star's bytes model: N*sizeof(grad) + (theta + state + EMA) read and written."""
        n_arrays = 1 + self.n_state + (0 if self.ema_mode == EMA_OFF else 1)
        return self.N * self.grad_bytes + 8 * n_arrays

    @property
    def bytes_per_step(self) -> int:
        return self.P * self.bytes_per_element

    @property
    def footprint_bytes(self) -> int:
        return self.P * (self.W * self.grad_bytes + 4 * (2 + self.n_state))


TINY = Config(name="cfg1_tiny", cfg_id=1, P=4096, M=2, N=4, b=1, theta_dist=("uniform", 0.1),
              grad_dist=("uniform", 1.0), arrival_sigma=0.3, opt=SGD, gamma=0.1, alpha=0.999, steps=10,
              ragged=False)
INCEPTION_SGD = Config(name="cfg2_inception_sgd", cfg_id=2, P=25_165_824, M=20, N=50, b=5, arrival_sigma=0.25,
                       opt=SGD, gamma=0.045, alpha=0.9999, steps=20)
PAPER_RMSPROP = Config(name="cfg3_paper_rmsprop", cfg_id=3, P=25_165_824, M=20, N=100, b=6, arrival_sigma=0.25,
                       delay_prob=0.02, delay_factor=5.0, opt=RMSPROP_MOM, gamma=0.045, alpha=0.9999, mu=0.9,
                       rho=0.9, eps=1.0, steps=50)
MIXED_PRECISION = Config(name="cfg4_mixed_precision", cfg_id=4, P=100_000_000, M=50, N=100, b=8, grad_dtype=BF16,
                         arrival_sigma=0.3, delay_prob=0.05, delay_factor=3.0, opt=MOMENTUM, gamma=0.01,
                         alpha=0.999, mu=0.9, steps=20)

CONFIGS = {c.name: c for c in (TINY, INCEPTION_SGD, PAPER_RMSPROP, MIXED_PRECISION)}

SWEEP_P = tuple(m << 20 for m in (1, 4, 16, 64, 256))
SWEEP_M = (1, 64)
SWEEP_NB = ((8, 0), (16, 2), (50, 5), (100, 10))
HBM_LIMIT_BYTES = 170 * 10**9


def sweep_configs():
    """cfg5: the bandwidth sweep; cases above 170 GB of HBM are skipped (none is, rule kept)."""
    out = []
    for P in SWEEP_P:
        for M in SWEEP_M:
            for (N, b) in SWEEP_NB:
                c = Config(name=f"cfg5_P{P >> 20}Mi_M{M}_N{N}_b{b}", cfg_id=5, P=P, M=M, N=N, b=b,
                           theta_dist=("uniform", 0.1), grad_dist=("uniform", 1.0), arrival_sigma=0.3, opt=SGD,
                           gamma=0.01, alpha=0.999, steps=5, ragged=(M > 1))
                if c.footprint_bytes <= HBM_LIMIT_BYTES:
                    out.append(c)
    return out


def scaled(cfg: Config, P: int, name: Optional[str] = None) -> Config:
    """The same workload at a smaller P (parity cases the oracle finishes in seconds)."""
    return replace(cfg, P=P, name=name or f"{cfg.name}_P{P}")


def seed_for(cfg: Config, step: int, stream: int, worker: int = 0) -> int:
    return MASTER_SEED + 100_000 * cfg.cfg_id + 10 * step + stream + 1_000_003 * worker


def shard_offsets(cfg: Config) -> np.ndarray:
    """int64 [M+1] with off[0]=0, off[M]=P.  Ragged: w_j ~ U[0.5,1.5], len_j = floor(P w_j / sum w),
    remainder to the last shard (element-aligned only)."""
    if not cfg.ragged or cfg.M == 1:
        base = cfg.P // cfg.M
        lens = np.full(cfg.M, base, dtype=np.int64)
        lens[-1] += cfg.P - base * cfg.M
    else:
        rng = np.random.default_rng(seed_for(cfg, 0, STREAM_INIT) + 7)
        w = rng.uniform(0.5, 1.5, size=cfg.M)
        lens = np.floor(cfg.P * w / w.sum()).astype(np.int64)
        lens[-1] += cfg.P - int(lens.sum())
    off = np.zeros(cfg.M + 1, dtype=np.int64)
    off[1:] = np.cumsum(lens)
    assert off[-1] == cfg.P and (np.diff(off) >= 0).all()
    return off


def _draw(dist, n, gen, device):
    kind, scale = dist
    if kind == "normal":
        out = torch.empty(n, dtype=torch.float32, device=device)
        out.normal_(0.0, scale, generator=gen)
        return out
    if kind == "uniform":
        out = torch.empty(n, dtype=torch.float32, device=device)
        out.uniform_(-scale, scale, generator=gen)
        return out
    raise ValueError(kind)


def init_theta(cfg: Config, device="cpu") -> torch.Tensor:
    gen = torch.Generator(device=device)
    gen.manual_seed(seed_for(cfg, 0, STREAM_INIT))
    return _draw(cfg.theta_dist, cfg.P, gen, device)


def init_state(cfg: Config, device="cpu"):
    """(state0, state1): momentum v0 = 0; RMSProp ms0 = cfg.ms0, mom0 = 0 (reading R5)."""
    if cfg.opt == SGD:
        return None, None
    if cfg.opt == MOMENTUM:
        return torch.zeros(cfg.P, dtype=torch.float32, device=device), None
    return (torch.full((cfg.P,), cfg.ms0, dtype=torch.float32, device=device),
            torch.zeros(cfg.P, dtype=torch.float32, device=device))


def gradient(cfg: Config, step: int, worker: int, device="cpu", out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Worker `worker`'s gradient buffer for `step`: fp32 [P], or bf16 [P] rounded once (RN-even)."""
    gen = torch.Generator(device=device)
    gen.manual_seed(seed_for(cfg, step, STREAM_GRAD, worker))
    g = _draw(cfg.grad_dist, cfg.P, gen, device)
    if cfg.grad_dtype == BF16:
        g = g.to(torch.bfloat16)
    if out is not None:
        out.copy_(g)
        return out
    return g


def arrival_times(cfg: Config, step: int) -> np.ndarray:
    """fp32 [W] seconds since the step started: exp(sigma z) times delay_factor with probability
    delay_prob (independent per worker per step); computed in double, rounded once to fp32."""
    rng = np.random.default_rng(seed_for(cfg, step, STREAM_ARRIVAL))
    z = rng.standard_normal(cfg.W)
    t = np.exp(cfg.arrival_sigma * z)
    if cfg.delay_prob > 0.0:
        t = np.where(rng.random(cfg.W) < cfg.delay_prob, t * cfg.delay_factor, t)
    return t.astype(np.float32)


def arrival_times_per_server(cfg: Config, step: int, server_sigma: float = 0.05) -> np.ndarray:
    """fp32 [M][W]: the time worker k's gradient slice reaches parameter server j (Alg. 4 runs per server,
    PAPER.md:L134).  Recipe: the worker's own time (arrival_times) times an independent per-(server, worker)
    network jitter exp(server_sigma z_jk); computed in double, rounded once to fp32."""
    base = arrival_times(cfg, step).astype(np.float64)
    rng = np.random.default_rng(seed_for(cfg, step, STREAM_ARRIVAL) + 5)
    z = rng.standard_normal((cfg.M, cfg.W))
    return (base[None, :] * np.exp(server_sigma * z)).astype(np.float32)


def as_numpy_grad(g: torch.Tensor) -> np.ndarray:
    """Host view for the oracle: float32 array, or uint16 bit patterns for bf16."""
    g = g.detach().cpu().contiguous()
    if g.dtype == torch.bfloat16:
        return g.view(torch.int16).numpy().view(np.uint16)
    return g.numpy()
