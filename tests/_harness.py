"""Shared test plumbing: run the CUDA path and the CPU oracle on the same seeded bytes and compare.

The oracle always receives the device-generated inputs by D2H copy; no expected value ever comes
from the CUDA path.  Tolerances are north_star's (BASELINE.json): rtol 1e-5 / atol 1e-6 per step in
lock-step, rtol 1e-4 after a 100-step free run, rtol 2e-3 for bf16 gradients.
"""
from __future__ import annotations

import numpy as np
import torch

import oracle
import paper_1702_05800_b200 as psync
from paper_1702_05800_b200 import synth

RTOL_STEP, ATOL_STEP = 1e-5, 1e-6
RTOL_FREE_100 = 1e-4
RTOL_BF16 = 2e-3

STATE_NAMES = ("theta", "ema", "state0", "state1")


def assert_close(got, want, rtol, atol, what=""):
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    err = np.abs(got - want)
    bound = atol + rtol * np.abs(want)
    bad = err > bound
    if bad.any():
        i = int(np.argmax(err - bound))
        raise AssertionError(f"{what}: {int(bad.sum())} of {got.size} elements out of tolerance; worst at {i}: "
                             f"got {got.flat[i]!r} want {want.flat[i]!r} err {err.flat[i]:.3e} bound {bound.flat[i]:.3e}")


def to_np(t):
    return None if t is None else t.detach().cpu().numpy().copy()


class Pair:
    """The same parameter-server state on the GPU (product) and on the host (oracle)."""

    def __init__(self, cfg: synth.Config, device="cuda", shard_off=None, variant=0, grid_ctas=0, theta=None):
        self.cfg = cfg
        self.dev = device
        self.shard_off = synth.shard_offsets(cfg) if shard_off is None else np.asarray(shard_off, dtype=np.int64)
        th = synth.init_theta(cfg, device) if theta is None else theta
        s0, s1 = synth.init_state(cfg, device)
        ema = th.clone() if cfg.ema_mode != synth.EMA_OFF else None     # reading R4: ema(-1) = theta(0)
        self.ps = psync.ParameterServerStep(self.shard_off, cfg.N, cfg.b, th, ema, s0, s1, cfg.opt, cfg.ema_mode,
                                            alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps,
                                            grid_ctas=grid_ctas, variant=variant)
        self.host = {n: to_np(getattr(self.ps, n)) for n in STATE_NAMES}

    # ---- inputs -------------------------------------------------------------------------------
    def gradients(self, step):
        return [synth.gradient(self.cfg, step, k, self.dev) for k in range(self.cfg.W)]

    # ---- one step on both sides -----------------------------------------------------------------
    def gpu_step(self, grads, arrival, tags=None, t=0):
        self.ps.set_gradients(grads)
        d_arr = torch.from_numpy(arrival).to(self.dev)
        d_tags = None if tags is None else torch.from_numpy(tags).to(self.dev)
        self.ps.step(d_arr, self.cfg.gamma, d_tags, t)
        torch.cuda.synchronize()
        return int(self.ps.d_status.item()), self.ps.d_kept.cpu().numpy(), float(self.ps.d_t_nth.item())

    def oracle_step(self, grads, arrival, tags=None, t=0):
        cfg = self.cfg
        st, kept, t_nth = oracle.select_first_n(arrival, cfg.N, cfg.b, tags=tags, t=t)
        if st != oracle.OK:
            return st, None, None
        h = self.host
        rc = oracle.aggregate_update(self.shard_off, cfg.N, [synth.as_numpy_grad(g) for g in grads], kept,
                                     h["theta"], h["ema"], h["state0"], h["state1"], opt=cfg.opt,
                                     ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu,
                                     rho=cfg.rho, eps=cfg.eps)
        assert rc == oracle.OK
        return st, kept, t_nth

    def sync_host_from_gpu(self):
        """Lock-step: the oracle's next step starts from the GPU's stored state."""
        self.host = {n: to_np(getattr(self.ps, n)) for n in STATE_NAMES}

    def compare(self, rtol, atol, what=""):
        for n in STATE_NAMES:
            g = getattr(self.ps, n)
            if g is None:
                continue
            assert_close(to_np(g), self.host[n], rtol, atol, f"{what} {self.cfg.name} {n}")

    def run(self, steps, lockstep=True, rtol=RTOL_STEP, atol=ATOL_STEP, check_every=1):
        for s in range(steps):
            grads = self.gradients(s)
            arrival = synth.arrival_times(self.cfg, s)
            st_g, kept_g, tn_g = self.gpu_step(grads, arrival)
            st_o, kept_o, tn_o = self.oracle_step(grads, arrival)
            assert st_g == st_o == 0
            assert np.array_equal(kept_g, kept_o), f"kept set differs at step {s}"
            assert tn_g == tn_o
            if (s + 1) % check_every == 0 or s == steps - 1:
                self.compare(rtol, atol, f"step {s}")
            if lockstep:
                self.sync_host_from_gpu()
            del grads
