#!/usr/bin/env python
"""bench.py -- whole-job throughput of the parameter-server step (Alg. 4) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg1..cfg5] [--impl psync|reference]
                    [--mode first_n|per_server|timeout|async] [--layout flat|slices] [--variant 1|5|6|7] [--servers M]

The default run is the headline (cfg3, first_n, flat buffers); its JSON line also carries `also`: short
measurements of cfg2, cfg4, every other mode, the slices layout, many-server cuts and launch variants 5 / 6.
`--config cfg5` runs BASELINE.json's bandwidth sweep (one JSON line with every point, `--sweep-md` for the table).

A "step" is one pass of the whole hot path -- psync_select_first_n then the fused
psync_aggregate_update (sum of the N kept gradients, optimizer update, EMA) -- over one batch of
synthetic input (fresh arrival times every step, gradient buffers rotated over several resident
sets far larger than L2).  Prints ONE JSON line (rank 0).  Metric: aggregated gradient elements
per second = N * P * steps / time; GB/s uses north_star's bytes model
N*P*sizeof(grad) + P*8*(1 + n_state + 1).

Multi-GPU (--gpus N under torchrun): the step does not shard across GPUs (north_star: no
collectives) -> N independent replicas, weak scaling; value = units of all ranks / max-over-ranks
time.  `--impl reference` times the CPU oracle (oracle/) as it stands on the host cores on the full workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1702_05800_b200 import synth  # noqa: E402

METRIC = "aggregated gradient elements/s"
UNIT = "grad-elements/s"
WORKLOADS = {"cfg1": synth.TINY, "cfg2": synth.INCEPTION_SGD, "cfg3": synth.PAPER_RMSPROP,
             "cfg4": synth.MIXED_PRECISION}
DTYPE_NAME = {synth.F32: "f32", synth.BF16: "f32 accumulate of bf16 gradients"}
OPT_NAME = {synth.SGD: "sgd", synth.MOMENTUM: "momentum", synth.RMSPROP_MOM: "rmsprop_momentum"}


def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


# ------------------------------------------------------------------------------------ multi-rank glue
def aggregate_over_ranks(local_units: float, local_ms: float, dist=None):
    """Whole-job numbers from per-rank ones: units are summed, time is the MAX over ranks.
    Works on any backend (tests drive it with gloo on CPU)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_units, local_ms
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([local_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([local_units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(u.item()), float(t.item())


class ClockSampler:
    """Samples SM clock / throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.002):
        self.index, self.period = index, period_s
        self.samples, self.reasons, self.power = [], set(), []
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        self.ok = False
        if period_s < 0:
            self.err = "disabled"
            return
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            visible = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if visible:
                ids = [v for v in visible.split(",") if v.strip() != ""]
                if index < len(ids) and ids[index].strip().isdigit():
                    phys = int(ids[index])
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)

    def _loop(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                 "sw_thermal_slowdown": 0x20, "hw_power_brake": 0x80, "sync_boost": 0x10,
                 "applications_clocks_setting": 0x2}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:  # noqa: BLE001
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:  # noqa: BLE001
                pass
            time.sleep(self.period)

    def start(self):
        if self.ok:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self) -> dict:
        if self._thr is not None:
            self._stop.set()
            self._thr.join()
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": float(self.max_mhz),
                "reasons": sorted(self.reasons), "samples": len(self.samples),
                "power_w_max": max(self.power) if self.power else None}


def load_peaks():
    """Measured roofline denominators (driver-written), else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
    except Exception:  # noqa: BLE001
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# ------------------------------------------------------------------------------------ CPU oracle legs
def oracle_full(cfg, host_grads, seconds_budget=12.0, max_steps=2000, warmup=0, fixed_steps=None, wall_budget=90.0,
                first_step=0, form="streamed"):
    """Times the oracle AS IT STANDS (all host cores) on the FULL workload: all P parameters of the W gradient buffers in
    `host_grads` (numpy, host RAM; for the cpu_baseline leg the exact bytes of the GPU's gradient set 0, copied D2H before
    timing), fresh arrival times every step, continuing from the previous step's theta / state / ema.
      form = "streamed": oracle.select_first_n, then oracle.accumulate over the kept buffers one at
             a time in ascending worker order, then oracle.apply_sum;
      form = "whole"  : oracle.select_first_n + oracle.aggregate_update (element-major over the N kept streams).
    The two are the same arithmetic in the same order (bit-identical, pinned in tests/test_oracle_update.py).  Runs
    `fixed_steps` steps, else until `seconds_budget` seconds of oracle time (or `wall_budget` seconds of wall clock).
    Returns (grad-elements/s, info)."""
    import oracle  # the one place bench.py executes oracle/ (cpu_baseline / --impl reference)

    off = synth.shard_offsets(cfg)
    theta = synth.init_theta(cfg).numpy().copy()
    s0, s1 = synth.init_state(cfg)
    s0 = None if s0 is None else s0.numpy().copy()
    s1 = None if s1 is None else s1.numpy().copy()
    ema = theta.copy()
    S = np.zeros(cfg.P, np.float64) if form == "streamed" else None
    hp = dict(opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
    t_begin = time.perf_counter()
    times = []
    total_steps = (fixed_steps + warmup) if fixed_steps is not None else max_steps
    for s in range(total_steps):
        arrival = synth.arrival_times(cfg, first_step + s)
        t0 = time.perf_counter()
        st, kept, _ = oracle.select_first_n(arrival, cfg.N, cfg.b)
        if form == "streamed":
            S[:] = 0.0
            for k in kept:
                rc = oracle.accumulate(S, host_grads[k])
            rc = rc or oracle.apply_sum(off, cfg.N, S, theta, ema, s0, s1, **hp)
        else:
            rc = oracle.aggregate_update(off, cfg.N, host_grads, kept, theta, ema, s0, s1, **hp)
        t1 = time.perf_counter()
        assert st == 0 and rc == 0
        if s >= warmup:
            times.append(t1 - t0)
        if fixed_steps is None and times and (sum(times) > seconds_budget or t1 - t_begin > wall_budget):
            break
    sec = float(np.sum(times))
    value = cfg.N * cfg.P * len(times) / sec
    how = ("kept buffers accumulated one at a time in ascending worker order (oracle.accumulate), then oracle.apply_sum"
           if form == "streamed" else "oracle.aggregate_update, element-major over the N kept streams")
    info = {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "note": "the oracle as it stands, never tuned: double arithmetic, " + how,
            "sample": f"the FULL workload: all P={cfg.P} parameters of the W={cfg.W} gradient buffers of one resident "
                      f"gradient set held in host RAM, N={cfg.N} b={cfg.b}, fresh arrival times per step, "
                      f"{len(times)} steps, {sec:.2f} s of oracle time (select + aggregate/update/EMA; input "
                      f"generation and device-to-host copies excluded)",
            "ms_per_step": 1e3 * sec / len(times),
            "gbps": cfg.bytes_per_step * len(times) / sec / 1e9}
    return value, info


def host_gradient_set(cfg, device="cpu", set_id=0):
    """The W gradient buffers of one set in host RAM (numpy): drawn on `device` with the workload's seeds."""
    out = []
    for k in range(cfg.W):
        out.append(synth.as_numpy_grad(synth.gradient(cfg, set_id, k, device)).copy())
    return out


def host_ram_ok(cfg) -> bool:
    need = cfg.W * cfg.P * cfg.grad_bytes + 6 * 4 * cfg.P + (2 << 30)
    try:
        import psutil
        return psutil.virtual_memory().available > need
    except Exception:  # noqa: BLE001
        return True


def run_reference(args, cfg, rank):
    """--impl reference: the oracle on the host cores, K steps of the FULL workload (no GPU is touched: the
    gradient set is drawn by torch's CPU generator with the workload's seeds and distribution), same metric."""
    if rank != 0:
        return None
    run_cfg = cfg if args.ref_sample_elems <= 0 else synth.scaled(cfg, int(min(args.ref_sample_elems, cfg.P)),
                                                                   name=cfg.name)
    if run_cfg is cfg and not host_ram_ok(cfg):        # a host without room for one gradient set: bounded sample
        run_cfg = synth.scaled(cfg, 1 << 22, name=cfg.name)
    grads = host_gradient_set(run_cfg)
    value, info = oracle_full(run_cfg, grads, warmup=args.warmup, fixed_steps=args.steps)
    if run_cfg is not cfg:
        info["sample"] = f"first {run_cfg.P} of P={cfg.P} parameters of every buffer; " + info["sample"]
    return {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": info["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64 arithmetic on f32 storage", "data": "synthetic",
            "config": workload_config(cfg, "first_n", "flat"),
            "cpu_baseline": {k: info[k] for k in ("value", "unit", "cores", "kind", "sample", "note")},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def workload_config(cfg, mode="first_n", layout="flat"):
    """The `config` object: names the workload; identical for the CUDA arm and the reference arm."""
    return {"workload": f"{cfg.name}: P={cfg.P} fp32 params in M={cfg.M} ragged shards, N={cfg.N}, b={cfg.b}, "
                        f"{'bf16' if cfg.grad_dtype == synth.BF16 else 'fp32'} gradients, {OPT_NAME[cfg.opt]}, EMA",
            "P": cfg.P, "M": cfg.M, "N": cfg.N, "b": cfg.b, "optimizer": OPT_NAME[cfg.opt],
            "grad_dtype": "bf16" if cfg.grad_dtype == synth.BF16 else "fp32", "gamma": cfg.gamma, "alpha": cfg.alpha,
            "bytes_per_step_model": cfg.bytes_per_step, "parallelism": "replicas only (no sharding across GPUs)",
            "mode": mode, "grad_layout": layout,
            "l2": f"no flush: each step streams {cfg.bytes_per_step / 1e9:.2f} GB (>> 126 MB L2) and the gradient "
                  f"buffers rotate over several resident sets"}


# ------------------------------------------------------------------------------------ the CUDA arm
L2_BYTES = 126 * 10**6


class Workload:
    """Device-resident data of one config: `n_sets` gradient sets (flat buffers or per-(worker, server) slices), the
    pointer tables, theta / state / ema, the shard table and the (server, tile) work list."""

    def __init__(self, psync, cfg, dev, n_sets, layout="flat", state_first=False):
        self.cfg, self.dev, self.layout = cfg, dev, layout
        self.off = synth.shard_offsets(cfg)
        tdt = torch.float32 if cfg.grad_dtype == synth.F32 else torch.bfloat16
        set_bytes = cfg.W * cfg.P * cfg.grad_bytes
        free, _ = torch.cuda.mem_get_info()
        self.n_sets = int(max(1, min(n_sets, (0.7 * free) // max(set_bytes, 1))))
        self.tables, self.sets = [], []
        if layout == "flat":
            for r in range(self.n_sets):     # gradient sets are allocated before theta / state (DESIGN.md s.5)
                bufs = [torch.empty(cfg.P, dtype=tdt, device=dev) for _ in range(cfg.W)]
                for k in range(cfg.W):
                    synth.gradient(cfg, r, k, dev, out=bufs[k])
                self.sets.append(bufs)
                self.tables.append(psync.make_grad_table(bufs))
        elif cfg.M <= 64:                    # every (worker, server) slice is its own allocation
            tmp = torch.empty(cfg.P, dtype=tdt, device=dev)
            for r in range(self.n_sets):
                slices = []
                for k in range(cfg.W):
                    synth.gradient(cfg, r, k, dev, out=tmp)
                    row = []
                    for j in range(cfg.M):
                        lo, hi = int(self.off[j]), int(self.off[j + 1])
                        t = torch.empty(hi - lo, dtype=tdt, device=dev)
                        t.copy_(tmp[lo:hi])
                        row.append(t)
                    slices.append(row)
                self.sets.append(slices)
                self.tables.append(psync.make_slice_table(slices))
            del tmp
            self.slices_how = "every slice its own torch allocation"
        else:
            # Thousands of servers: W*M separate tensors cost minutes of Python, so each worker's slices are carved
            # from one arena at 256-byte boundaries (the alignment a separate cudaMalloc would give each of them);
            # the kernel sees the same thing either way -- W*M unrelated base pointers in a table.
            lens = np.diff(self.off)
            esz = cfg.grad_bytes
            starts = np.zeros(cfg.M, dtype=np.int64)      # arena offset of slice j, in elements
            pos = 0
            for j in range(cfg.M):
                starts[j] = pos
                pos = -(-(pos + int(lens[j])) * esz // 256) * 256 // esz
            arena_elems = max(pos, 1)
            pad = torch.from_numpy(starts - self.off[:-1]).to(dev)
            dst = torch.arange(cfg.P, dtype=torch.int64, device=dev) + torch.repeat_interleave(
                pad, torch.from_numpy(lens).to(dev))
            tmp = torch.empty(cfg.P, dtype=tdt, device=dev)
            for r in range(self.n_sets):
                arenas = []
                ptrs = np.empty((cfg.W, cfg.M), dtype=np.int64)
                for k in range(cfg.W):
                    synth.gradient(cfg, r, k, dev, out=tmp)
                    arena = torch.zeros(arena_elems, dtype=tdt, device=dev)
                    arena.index_copy_(0, dst, tmp)
                    arenas.append(arena)
                    ptrs[k] = arena.data_ptr() + starts * esz
                self.sets.append(arenas)
                self.tables.append(psync.binding.GradTable(torch.from_numpy(ptrs.reshape(-1)).to(dev), arenas,
                                                           psync.PSYNC_F32 if esz == 4 else psync.PSYNC_BF16))
            del tmp, dst
            self.arena_starts = starts
            self.slices_how = "slices carved at 256-byte boundaries from one arena per worker"
        self.theta = synth.init_theta(cfg, dev)
        self.s0, self.s1 = synth.init_state(cfg, dev)
        self.ema = self.theta.clone()
        self.d_off = torch.from_numpy(self.off).to(dev)
        self.d_tiles = psync.psync_shard_worklist(self.d_off, cfg.grad_dtype)

    def break_worklist(self, psync):
        """--fault worklist: the list of the OTHER gradient dtype (another tile count): the kernel must refuse it."""
        self.d_tiles = psync.psync_shard_worklist(self.d_off, 1 - self.cfg.grad_dtype)

    def with_servers(self, psync, M):
        """The same resident flat gradient sets and state cut into M ragged servers (only the tables change)."""
        from dataclasses import replace
        other = object.__new__(Workload)
        other.__dict__.update(self.__dict__)
        other.cfg = replace(self.cfg, M=M, name=f"{self.cfg.name}_M{M}")
        other.off = synth.shard_offsets(other.cfg)
        other.d_off = torch.from_numpy(other.off).to(self.dev)
        other.d_tiles = psync.psync_shard_worklist(other.d_off, other.cfg.grad_dtype)
        return other

    def reset_state(self):
        cfg = self.cfg
        self.theta.copy_(synth.init_theta(cfg, self.dev))
        self.ema.copy_(self.theta)
        s0, s1 = synth.init_state(cfg, self.dev)
        if s0 is not None:
            self.s0.copy_(s0)
        if s1 is not None:
            self.s1.copy_(s1)


# ------------------------------------------------------------------------------------ proof of what was timed
RTOL_STEP, RTOL_BF16, ATOL_STEP = 1e-5, 2e-3, 1e-6      # north_star's per-step tolerances (tests/_harness.py)


class VerifyError(AssertionError):
    pass


def sample_columns(cfg, off, n_sample=20_000):
    """The parameter indices a timed configuration is checked on: the first and last tiles, both sides of every shard
    cut, and n_sample uniformly drawn ones (sorted, unique) -- the index set of tests/test_gpu_configs.py."""
    rng = np.random.default_rng(1000 + cfg.cfg_id)
    tile = min(8192, cfg.P)
    cuts = np.asarray(off[1:-1], dtype=np.int64)
    if cuts.size > 4096:                                 # thousands of servers: a seeded subset of the cuts
        cuts = rng.choice(cuts, 4096, replace=False)
    idx = np.concatenate([np.arange(0, tile), np.arange(cfg.P - tile, cfg.P), cuts, np.maximum(cuts - 1, 0),
                          rng.integers(0, cfg.P, n_sample)])
    return np.unique(idx).astype(np.int64)


def gather_gradient_columns(wl, set_id, idx, d_idx):
    """Columns idx of every worker's gradient of one resident set, as W host arrays (moves data, computes nothing)."""
    cfg = wl.cfg
    data = wl.sets[set_id]
    if wl.layout == "flat":
        return [synth.as_numpy_grad(g[d_idx]) for g in data]
    server = np.searchsorted(wl.off, idx, side="right") - 1          # owner j of every sampled parameter
    local = idx - wl.off[server]
    if hasattr(wl, "arena_starts"):                                      # slices carved from one arena per worker
        d_pos = torch.from_numpy(wl.arena_starts[server] + local).to(wl.dev)
        return [synth.as_numpy_grad(a[d_pos]) for a in data]
    out = []
    bounds = np.searchsorted(server, np.arange(cfg.M + 1))               # sampled columns of server j: [b[j], b[j+1])
    d_local = torch.from_numpy(local).to(wl.dev)
    for row in data:                                                     # row[j]: worker's own slice for server j
        parts = [row[j][d_local[bounds[j]:bounds[j + 1]]] for j in range(cfg.M) if bounds[j + 1] > bounds[j]]
        out.append(synth.as_numpy_grad(torch.cat(parts)))
    return out


def verify_step(cfg, off, mode, timeout, arrival, g_s, before, after, kept_g, n_g, idx, d_idx, gscales=None):
    """Replays ONE step of what `measure` times through the CPU oracle on the sampled columns and compares: the kept
    rows / arrival orders bit for bit, theta / state / ema at north_star's tolerance (PAPER.md:L130, L157-162 for Alg. 4,
    L84-87 for Alg. 2).  `before` holds the sampled state just before the step.  Returns the `verified` object or raises
    VerifyError.  g_s: the sampled columns of the W gradients (host arrays); after: the device tensors theta / ema /
    state0 / state1 after the step; kept_g [rows][stride] / n_g [rows]: what the device selected (None: not returned by
    this path, only the state is checked).  The oracle is on the checking side only: nothing here feeds the timed path."""
    import oracle
    W, N, M = cfg.W, cfg.N, cfg.M
    off_s = np.searchsorted(idx, off).astype(np.int64)                  # the shard table of the sampled columns
    have_kept = kept_g is not None
    if not have_kept:
        kept_g, n_g = np.full((M, W), -2, dtype=np.int32), np.full(M, -2, dtype=np.int32)
    h = {n: (None if v is None else v.copy()) for n, v in before.items()}
    kw = dict(opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
    K_applied = N
    if mode == "first_n":
        st, kept_o, _ = oracle.select_first_n(arrival, N, cfg.b)
        same = st == oracle.OK and np.array_equal(kept_g[0, :N], kept_o)
        rc = oracle.aggregate_update(off_s, N, g_s, kept_o, h["theta"], h["ema"], h["state0"], h["state1"], **kw)
    elif mode == "per_server":
        st, kept_o, _ = oracle.select_first_n_sharded(arrival, N, cfg.b)
        same = bool((st == oracle.OK).all()) and np.array_equal(kept_g[:, :N], kept_o)
        rc = oracle.aggregate_update_rows(off_s, N, g_s, kept_o, h["theta"], h["ema"], h["state0"], h["state1"],
                                          per_shard=True, **kw)
    elif mode == "timeout":
        st, kept_o = oracle.select_timeout(arrival, timeout)
        same = st == oracle.OK and int(n_g[0]) == kept_o.size and np.array_equal(kept_g[0, :kept_o.size], kept_o)
        row = np.full((1, W), -1, dtype=np.int32)
        row[0, :kept_o.size] = kept_o
        rc = oracle.aggregate_update_rows(off_s, N, g_s, row, h["theta"], h["ema"], h["state0"], h["state1"],
                                          per_shard=False, n_kept=np.array([kept_o.size], dtype=np.int32), **kw)
        K_applied = kept_o.size
    elif mode == "async":
        order = oracle.order_by_arrival(arrival)
        same = int(n_g[0]) == order.size and np.array_equal(kept_g[0, :order.size], order)
        rc = oracle.async_apply(off_s, g_s, order, h["theta"], h["ema"], h["state0"], h["state1"],
                                gscales=None if gscales is None else gscales[order].copy(), **kw)
        K_applied = order.size
    else:                                                                # async_per_server
        order = np.full((M, W), -1, dtype=np.int32)
        n_arr = np.zeros(M, dtype=np.int32)
        for j in range(M):
            o = oracle.order_by_arrival(arrival[j])
            order[j, :o.size], n_arr[j] = o, o.size
        same = np.array_equal(n_g, n_arr) and all(np.array_equal(kept_g[j, :n_arr[j]], order[j, :n_arr[j]]) for j in range(M))
        rc = oracle.async_apply_rows(off_s, g_s, order, h["theta"], h["ema"], h["state0"], h["state1"], slices=False,
                                     per_shard=True, n_arrived=n_arr, gscales=gscales, **kw)
        K_applied = int(n_arr.max())
    if have_kept and not same:
        raise VerifyError(f"{cfg.name} {mode}: kept rows / arrival order differ from the oracle's")
    if rc != oracle.OK:
        raise VerifyError(f"{cfg.name} {mode}: oracle returned {rc}")
    is_async = mode in ("async", "async_per_server")
    rtol = 1e-6 * max(10, K_applied) if is_async else (RTOL_BF16 if cfg.grad_dtype == synth.BF16 else RTOL_STEP)
    worst, max_rel, max_abs, moved = 0.0, 0.0, 0.0, 0
    for n, t in after.items():
        if t is None or h[n] is None:
            continue
        got = t[d_idx].cpu().numpy().astype(np.float64)
        want = h[n].astype(np.float64)
        err = np.abs(got - want)
        if not np.isfinite(got).all():
            raise VerifyError(f"{cfg.name} {mode}: non-finite {n}")
        worst = max(worst, float((err / (ATOL_STEP + rtol * np.abs(want))).max()))
        max_abs = max(max_abs, float(err.max()))
        big = np.abs(want) >= 1e-3
        if big.any():
            max_rel = max(max_rel, float((err[big] / np.abs(want[big])).max()))
        if n == "theta":
            moved = int((got != before["theta"].astype(np.float64)).sum())
    if worst > 1.0:
        raise VerifyError(f"{cfg.name} {mode}: sampled state differs from the oracle by {worst:.3g} x the tolerance "
                          f"(rtol {rtol:g}, atol {ATOL_STEP:g}); max abs error {max_abs:.3g}")
    if cfg.gamma != 0 and moved < idx.size // 2:
        raise VerifyError(f"{cfg.name} {mode}: only {moved} of {idx.size} sampled parameters changed in the step")
    return {"elements": int(idx.size), "kept_bit_exact": True if have_kept else None, "max_rel_err": max_rel, "max_abs_err": max_abs,
            "max_err_over_tolerance": worst, "rtol": rtol, "atol": ATOL_STEP, "theta_changed": moved,
            "how": "one more step after the timed region, same launch, replayed by the CPU oracle on the sampled columns"}


def measure(psync, args, wl, mode, K, Wm, stream, dist=None, variant=0, worklist=True, clip=0.0, probe_every=4):
    """W warm-up + K timed steps of one (workload, mode) on `stream`; returns the per-step numbers, the fused kernel's
    own CUDA-event duration (every `probe_every`-th timed step) and the clocks sampled during the timed region.
      first_n     one kept set of N per step (the headline; reading R11)
      per_server  Alg. 4 per server j: arrival [M][W] -> kept [M][N] (NEXT-1)
      timeout     keep every worker that arrived by --timeout seconds, divide by the count (NEXT-2)
      async       Alg. 2: all W gradients one at a time in arrival order, one pass (NEXT-3)
      async_per_server  Alg. 2 per server j: arrival [M][W] -> one order per server, over the work list"""
    cfg, dev = wl.cfg, wl.dev
    B = psync.binding
    slices = wl.layout == "slices"
    per_server = mode in ("per_server", "async_per_server")
    is_async = mode in ("async", "async_per_server")
    rows = cfg.M if per_server else 1
    if per_server:                       # K + Wm steps, + 1 for the verified step after the timed region
        arr_np = np.stack([synth.arrival_times_per_server(cfg, s) for s in range(K + Wm + 1)])
    else:
        arr_np = np.stack([synth.arrival_times(cfg, s) for s in range(K + Wm + 1)])
    arrivals = torch.from_numpy(arr_np).to(dev)
    stride = cfg.W if (mode == "timeout" or is_async) else cfg.N
    d_kept = torch.full((rows, stride), -1, dtype=torch.int32, device=dev)
    d_status = torch.full((rows,), 0 if is_async else -9, dtype=torch.int32, device=dev)
    d_t_nth = torch.zeros(rows, dtype=torch.float32, device=dev)
    d_n_kept = torch.zeros(rows, dtype=torch.int32, device=dev) if (mode == "timeout" or is_async) else None
    use_tiles = slices or (mode == "per_server" and worklist) or mode == "async_per_server"
    steps_struct = []
    for tb in wl.tables:   # one psync_step per gradient set, built once (marshalling outside the timed region)
        st, keep = psync.make_step(wl.off, cfg.N, cfg.W, tb.grad_dtype, wl.theta, wl.ema, wl.s0, wl.s1, opt=cfg.opt,
                                   ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho,
                                   eps=cfg.eps, d_grads=tb.d_ptrs, d_kept=d_kept, d_status=d_status,
                                   grid_ctas=args.grid_ctas, variant=variant, per_shard=per_server,
                                   d_shard_off=wl.d_off if (per_server or slices) else None,
                                   d_n_kept=d_n_kept,
                                   grad_layout=psync.PSYNC_GRADS_SLICES if slices else psync.PSYNC_GRADS_FLAT,
                                   d_tile_start=wl.d_tiles if use_tiles else None)
        steps_struct.append((st, keep))
    try:
        geo = psync.psync_launch_geometry(steps_struct[0][0])
    except psync.PsyncError:        # an A/B shape of Alg. 2's kernel (--mode async --variant N): no K2 geometry
        geo = {}
    d_scales = d_clip_work = None
    if is_async and clip > 0:
        d_scales = torch.ones(cfg.W, dtype=torch.float32, device=dev)
        d_clip_work = torch.empty(psync.psync_clip_workspace_bytes(cfg.W, cfg.P, cfg.grad_dtype) // 8,
                                  dtype=torch.float64, device=dev)
    n_sets = len(wl.tables)
    # Placement hygiene (measured, DESIGN.md s.5): a freed block that torch's caching allocator still holds -- even one
    # 100 MB temporary -- makes the same kernel on the same buffers 2-3 % slower until it is returned to the driver
    # (cfg3: 1.530 -> 1.574 ms; `--hold-cached-block` reproduces it).  Return everything unused before timing.
    if getattr(args, "hold_cached_block", False):
        tmp = torch.empty(25_165_824, dtype=torch.float32, device=dev)
        tmp.normal_()
        del tmp
    else:
        torch.cuda.empty_cache()
    stream.wait_stream(torch.cuda.current_stream())    # everything above was filled on the default stream

    def select(i):
        if mode == "first_n":
            B.psync_select_first_n(arrivals[i], cfg.N, cfg.b, d_kept, d_status, d_t_nth, None, i, stream)
        elif mode == "per_server":
            B.psync_select_first_n_sharded(arrivals[i], cfg.N, cfg.b, cfg.M, d_kept, d_status, None, None, i, stream)
        elif mode == "timeout":
            B.psync_select_timeout(arrivals[i], cfg.W, args.timeout, d_kept, d_n_kept, d_status, stream=stream)
        elif mode == "async_per_server":
            B.psync_order_by_arrival_sharded(arrivals[i], cfg.W, cfg.M, d_kept, d_n_kept, stream)
        else:
            B.psync_order_by_arrival(arrivals[i], cfg.W, d_kept, d_n_kept, stream)

    def one_step(i, ev=None):
        st = steps_struct[i % n_sets][0]
        if ev is None and mode in ("first_n", "per_server"):     # the user's call: selection + fused update
            B.psync_step_device(st, arrivals[i], None, None, i, stream)
            return
        if ev is not None:
            ev[0].record(stream)
        select(i)
        if ev is not None:
            ev[1].record(stream)
        if is_async:
            if clip > 0:                 # A.3 (L313): global-norm clipping = one more pass over the W buffers
                B.psync_clip_scales(wl.tables[i % n_sets], clip, d_scales, d_clip_work, stream)
            B.psync_async_apply(st, None, stream, d_gscale=d_scales if clip > 0 else None)
        else:
            B.psync_aggregate_update(st, stream)
        if ev is not None:
            ev[2].record(stream)

    def barrier():
        if dist is not None and dist.is_initialized():
            dist.barrier()

    for i in range(Wm):
        one_step(i)
    torch.cuda.synchronize()
    assert bool((d_status == 0).all())

    # Per-kernel CUDA events are recorded on every `probe_every`-th timed step only: an event between
    # the two launches breaks their programmatic-dependent-launch pairing and costs ~10 us, so the
    # other steps run exactly as a user's loop would.  All of it is inside the one timed region.
    probe_every = max(1, probe_every)
    evs = {k: [torch.cuda.Event(enable_timing=True) for _ in range(3)] for k in range(0, K, probe_every)}
    e_begin, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(env_int("LOCAL_RANK", 0), period_s=args.clock_period_ms * 1e-3)
    barrier()
    torch.cuda.synchronize()
    sampler.start()
    e_begin.record(stream)
    for k in range(K):
        one_step(Wm + k, evs.get(k))
    e_end.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    barrier()
    total_ms = e_begin.elapsed_time(e_end)
    fused_list = [e[1].elapsed_time(e[2]) for e in evs.values()]
    fused_ms = float(np.mean(fused_list))
    select_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs.values()]))
    if os.environ.get("PSYNC_BENCH_DEBUG"):
        print("fused ms per probed step:", [round(x, 4) for x in fused_list], file=sys.stderr)
    assert bool((d_status == 0).all()) and bool(torch.isfinite(wl.theta[:4096]).all())

    # Proof that what was timed computes Alg. 4 / Alg. 2: one more step through exactly the same calls, outside the timed
    # region, checked against the CPU oracle on sampled columns (kept rows bit for bit, state at north_star's tolerance).
    verified = None
    if not getattr(args, "no_verify", False):
        idx = sample_columns(cfg, wl.off, args.verify_sample)
        d_idx = torch.from_numpy(idx).to(dev)
        before = {n: (None if t is None else t[d_idx].cpu().numpy())
                  for n, t in (("theta", wl.theta), ("ema", wl.ema), ("state0", wl.s0), ("state1", wl.s1))}
        torch.cuda.synchronize()
        iv = Wm + K
        one_step(iv)
        torch.cuda.synchronize()
        if not bool((d_status == 0).all()):
            raise VerifyError(f"{cfg.name} {mode}: device status {d_status.cpu().tolist()[:8]}")
        verified = verify_step(cfg, wl.off, mode, args.timeout, arr_np[iv], gather_gradient_columns(wl, iv % n_sets, idx, d_idx),
                               before, {"theta": wl.theta, "ema": wl.ema, "state0": wl.s0, "state1": wl.s1},
                               d_kept.cpu().numpy(), None if d_n_kept is None else d_n_kept.cpu().numpy(), idx, d_idx,
                               gscales=None if d_scales is None else d_scales.cpu().numpy())

    # gradient elements aggregated per step: N*P, or (workers in time)*P for the time-out rule
    if is_async:
        n_eff = float(cfg.W)                 # every gradient is applied (nothing is dropped in Alg. 2)
    elif mode == "timeout":
        n_eff = float(np.mean([(arr_np[Wm + k] <= args.timeout).sum() for k in range(K)]))
    else:
        n_eff = float(cfg.N)
    bytes_per_step = cfg.bytes_per_step + (n_eff - cfg.N) * cfg.P * cfg.grad_bytes
    launches_per_step = 2                    # selection (or arrival order) + the fused pass
    if is_async and clip > 0:
        bytes_per_step += cfg.W * cfg.P * cfg.grad_bytes      # the norm pass reads every buffer once more
        launches_per_step = 4                # + sum-of-squares chunks + clip factors
    return {"total_ms": total_ms, "ms_per_step": total_ms / K, "fused_ms": fused_ms, "select_ms": select_ms,
            "verified": verified,
            "fused_list": fused_list, "n_eff": n_eff, "bytes_per_step": bytes_per_step, "units": n_eff * cfg.P * K,
            "clocks": clocks, "geo": geo, "launches_per_step": launches_per_step,
            "kernel": ("async_sharded_kernel" if use_tiles else
                       {1: "async_apply_kernel"}.get(variant, "async_apply_ring_kernel"))
                      if is_async else
                      ("sharded_aggregate_update_ema" if use_tiles else "fused_aggregate_update_ema")}


def short_entry(cfg, mode, layout, m, peak, note=None):
    """One entry of the `also` object: kernel ms, GB/s of algorithmic bytes, fractions, its own clocks."""
    gbs = m["bytes_per_step"] / (m["fused_ms"] * 1e-3) / 1e9
    e = {"workload": cfg.name, "mode": mode, "grad_layout": layout, "P": cfg.P, "M": cfg.M, "N": cfg.N, "b": cfg.b,
         "kernel": m["kernel"], "kernel_ms": m["fused_ms"], "step_ms": m["ms_per_step"], "kept_per_step": m["n_eff"],
         "algorithmic_bytes_per_launch": m["bytes_per_step"], "gbps": gbs, "frac": gbs / peak,
         "frac_of_nominal_8TBps": gbs / 8000.0,
         "value": m["units"] / (m["total_ms"] * 1e-3), "unit": UNIT, "launch": m["geo"],
         "clocks": {k: m["clocks"].get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons")}}
    if m.get("verified") is not None:
        v = m["verified"]
        e["verified"] = {k: v[k] for k in ("elements", "kept_bit_exact", "max_rel_err", "max_err_over_tolerance")}
    if note:
        e["note"] = note
    return e


def run_also(psync, args, wl3, stream, peak):
    """Short (8-step) measurements of the other configs and modes, so that the driver's BENCH record carries them:
    cfg3 in every mode and layout (reusing the headline's resident gradient sets), then cfg2 and cfg4."""
    from dataclasses import replace
    K, Wm = args.also_steps, 3
    out = []
    dev = wl3.dev
    cfg3 = wl3.cfg
    for mode in ("per_server", "timeout", "async", "async_per_server"):
        wl3.reset_state()
        m = measure(psync, args, wl3, mode, K, Wm, stream, probe_every=2)
        note = None
        if mode == "async_per_server":
            note = "Alg. 2 per server j: one arrival order per server, flat buffers through the (server, tile) work list"
        if mode == "async":
            note = "Alg. 2, all W gradients one at a time in one pass; RMSProp: bound by instruction issue as well as HBM"
        out.append(short_entry(cfg3, mode, "flat", m, peak, note))
    for M in (1000, 20000):              # one kept row per server, many small ragged servers, flat buffers + work list
        wlm = wl3.with_servers(psync, M)
        wlm.reset_state()
        m = measure(psync, args, wlm, "per_server", K, Wm, stream, probe_every=2)
        out.append(short_entry(wlm.cfg, "per_server", "flat", m, peak, "flat buffers through the (server, tile) work list"))
    for v in (5, 6, 7):                  # the rejected designs, re-measured every run (DESIGN.md s.5)
        wl3.reset_state()
        m = measure(psync, args, wl3, "first_n", K, Wm, stream, variant=v, probe_every=2)
        out.append(short_entry(cfg3, "first_n", "flat", m, peak,
                               {5: "variant 5: cp.async.bulk + mbarrier ring", 6: "variant 6: 256-bit loads",
                                7: "variant 7: per-thread cp.async ring (Alg. 2's staging)"}[v]))
        out[-1]["variant"] = v
    wl3.reset_state()                    # Alg. 2's other launch shape, re-measured every run (profiles/r2_async.md)
    m = measure(psync, args, wl3, "async", K, Wm, stream, variant=1, probe_every=2)
    out.append(short_entry(cfg3, "async", "flat", m, peak,
                           "variant 1: two register buffers, software-pipelined (the default is the cp.async ring)"))
    out[-1]["variant"] = 1
    sets3 = len(wl3.tables)
    del wl3.tables[1:], wl3.sets[1:]     # keep one flat set for the cpu_baseline leg; make room
    torch.cuda.empty_cache()
    # per-(worker, server) slices of cfg3, one shared kept set and one kept row per server; many small servers
    for M, modes in ((cfg3.M, ("first_n", "per_server", "async", "async_per_server")), (1000, ("per_server",)), (20000, ("per_server",))):
        cfg = cfg3 if M == cfg3.M else replace(cfg3, M=M, name=f"{cfg3.name}_M{M}")
        wl = Workload(psync, cfg, dev, 2, layout="slices")
        for mode in modes:
            wl.reset_state()
            m = measure(psync, args, wl, mode, K, Wm, stream, probe_every=2)
            out.append(short_entry(cfg, mode, "slices", m, peak,
                                   f"{cfg.W * cfg.M} slices per set ({wl.slices_how}), {wl.n_sets} sets"))
        del wl
        torch.cuda.empty_cache()
    for cfg in (synth.INCEPTION_SGD, synth.MIXED_PRECISION):
        wl = Workload(psync, cfg, dev, 3)
        m = measure(psync, args, wl, "first_n", K, Wm, stream, probe_every=2)
        out.append(short_entry(cfg, "first_n", "flat", m, peak))
        if cfg is synth.MIXED_PRECISION:
            wl.reset_state()
            m = measure(psync, args, wl, "async", K, Wm, stream, probe_every=2)
            out.append(short_entry(cfg, "async", "flat", m, peak))
        del wl
        torch.cuda.empty_cache()
    return out, sets3


def run_psync(args, cfg, rank, world, dist):
    import paper_1702_05800_b200 as psync

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU path")
    local = env_int("LOCAL_RANK", 0)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    K, Wm = args.steps, args.warmup
    mode = args.mode
    if args.servers > 0 and args.servers != cfg.M:
        from dataclasses import replace
        cfg = replace(cfg, M=args.servers, name=f"{cfg.name}_M{args.servers}")
    wl = Workload(psync, cfg, dev, args.grad_sets, layout=args.layout)
    if args.fault == "worklist":
        wl.break_worklist(psync)
    stream = torch.cuda.Stream(device=dev)
    B = psync.binding
    m = measure(psync, args, wl, mode, K, Wm, stream, dist, variant=args.variant, worklist=not args.no_worklist,
                clip=args.clip, probe_every=args.probe_every)

    units, max_ms = aggregate_over_ranks(m["units"], m["total_ms"], dist)
    value = units / (max_ms * 1e-3)
    peak, peak_src = load_peaks()
    bytes_per_step, fused_ms, fused_list = m["bytes_per_step"], m["fused_ms"], m["fused_list"]
    achieved = bytes_per_step / (fused_ms * 1e-3) / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": max_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if cfg.grad_dtype == synth.F32 else "f32 (bf16 gradients widened exactly)",
        "data": "synthetic",
        "config": workload_config(cfg, mode, args.layout),
        "launch": {"geometry": m["geo"], "variant": args.variant, "grad_sets": wl.n_sets,
                   "kept_per_step": m["n_eff"], "work_list": bool(args.layout == "slices" or
                                                                   (mode == "per_server" and not args.no_worklist))},
        "gbps_model": bytes_per_step * K * world / (max_ms * 1e-3) / 1e9,
        "params_per_s": float(cfg.P) * K * world / (max_ms * 1e-3),
        "select_ms": m["select_ms"], "fused_ms": fused_ms, "kernel_events_on_steps": len(fused_list),
        "fused_ms_min_median_max": [float(np.min(fused_list)), float(np.median(fused_list)), float(np.max(fused_list))],
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": None, "peak_source": peak_src, "kernel": m["kernel"],
                     "algorithmic_bytes_per_launch": bytes_per_step,
                     "frac_of_nominal_8TBps": achieved / 8000.0},
        "clocks": m["clocks"],
        "gpu_launches": m["launches_per_step"] * K,
        "verified": m["verified"],
    }
    traffic_file = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(traffic_file) and mode == "first_n" and args.layout == "flat" and args.variant in (0, 1):
        try:                                  # dram bytes per launch from the committed ncu --set full capture
            with open(traffic_file) as fh:
                tj = json.load(fh)
            if tj.get("psync_version") == psync.binding.psync_version():
                out["roofline"]["traffic"] = tj.get(cfg.name)
            else:                             # captured on another build of the library: not evidence for this one
                out["roofline"]["traffic_note"] = (f"profiles/traffic.json was captured on build "
                                                   f"{tj.get('psync_version')}, this is {psync.binding.psync_version()}")
            out["roofline"]["traffic_source"] = ("ncu --set full capture committed in profiles/traffic.json "
                                                 "(dram__bytes_read.sum + dram__bytes_write.sum per launch; not "
                                                 "measured in this run)")
        except Exception:  # noqa: BLE001
            pass

    # What this box's HBM gives a plain stream right now (K0 probes of the library, same process, same clocks):
    # a read-only pass over the gradient buffers of one set and a copy between two of them.  MEASURED_PEAKS's
    # number is a copy; the fused kernel is 96 % reads, so the read-only probe is the closer ceiling.
    if not args.no_probe and torch.cuda.mem_get_info()[0] > 12e9:
        src = torch.zeros(1 << 30, dtype=torch.float32, device=dev)          # 4 GiB >> L2
        dst = torch.empty_like(src)
        sink = torch.zeros(4, dtype=torch.float32, device=dev)
        pe = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        stream.wait_stream(torch.cuda.current_stream())
        for rep in range(3):                               # the first repetitions are the warm-up
            pe[0].record(stream)
            rbytes = B.psync_probe_read(src, sink, stream)
            pe[1].record(stream)
            cbytes = B.psync_probe_copy(dst, src, stream)
            pe[2].record(stream)
            torch.cuda.synchronize()
        read_gbs = rbytes / (pe[0].elapsed_time(pe[1]) * 1e-3) / 1e9
        out["roofline"]["probe_read_gbs"] = read_gbs
        out["roofline"]["frac_of_probe_read"] = achieved / read_gbs
        out["roofline"]["probe_copy_gbs"] = cbytes / (pe[1].elapsed_time(pe[2]) * 1e-3) / 1e9
        del src, dst

    headline = (rank == 0 and world == 1 and args.config == "cfg3" and mode == "first_n" and args.layout == "flat"
                and args.servers <= 0)
    cfg5_subset = None
    if headline and not args.no_also:
        out["also"], _ = run_also(psync, args, wl, stream, peak)
        if not args.no_cfg5:
            cfg5_subset = run_cfg5_subset(psync, args, dev, stream, peak)

    # the CPU baseline leg: the exact bytes of gradient set 0, copied D2H before any oracle timing
    host_grads = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and args.layout == "flat":
        if host_ram_ok(cfg):
            host_grads = [synth.as_numpy_grad(g).copy() for g in wl.sets[0]]
    theta, ema, s0, s1, off = wl.theta, wl.ema, wl.s0, wl.s1, wl.off
    del wl.tables, wl.sets
    torch.cuda.empty_cache()
    if not args.no_e2e and mode in ("first_n", "async"):
        out["e2e"] = run_e2e(args, cfg, dev, off, theta, ema, s0, s1, stream, rank, world, dist, mode=mode)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        if host_grads is None:               # no room in host RAM for one gradient set: bounded sample
            sub = synth.scaled(cfg, 1 << 22, name=cfg.name)
            _, info = oracle_full(sub, host_gradient_set(sub), seconds_budget=args.cpu_seconds)
            info["sample"] = f"first {sub.P} of P={cfg.P} parameters of every buffer; " + info["sample"]
        else:
            _, info = oracle_full(cfg, host_grads, seconds_budget=args.cpu_seconds, first_step=Wm)
            info["sample"] += "; the buffers are the GPU arm's gradient set 0, byte for byte"
        out["cpu_baseline"] = {k: info[k] for k in ("value", "unit", "cores", "kind", "sample", "note")}
        if host_grads is not None:            # the same arithmetic through the whole-step entry point (element-major)
            vw, infow = oracle_full(cfg, host_grads, fixed_steps=2, first_step=Wm, form="whole")
            out["cpu_baseline"]["value_whole_step_form"] = vw
            out["cpu_baseline"]["note_whole_step_form"] = infow["note"] + "; 2 steps"
        if args.cpu_seconds_1thread > 0:       # the oracle single-threaded as well (a short sample)
            threads = oracle.num_threads()
            oracle.set_num_threads(1)
            try:
                sub = synth.scaled(cfg, 1 << 20, name=cfg.name)
                sub_grads = [g[:sub.P] for g in host_grads] if host_grads is not None else host_gradient_set(sub)
                v1, info1 = oracle_full(sub, sub_grads, seconds_budget=args.cpu_seconds_1thread, wall_budget=20.0)
            finally:
                oracle.set_num_threads(threads)
            out["cpu_baseline"]["value_1thread"] = v1
            out["cpu_baseline"]["sample_1thread"] = f"first {sub.P} parameters of every buffer; " + info1["sample"]
    # compact records, assigned LAST so that they are the tail of the JSON line: BASELINE.json's cfg5 metric ("GB/s vs P
    # and N+b") on a fixed 10-point subset, and one short row per `also` entry
    if cfg5_subset is not None:
        out["cfg5"] = cfg5_subset
    if "also" in out:
        out["also_summary"] = {
            "columns": ["kernel_ms", "GB/s", "frac_of_nominal_8TBps", "verified_elements", "max_err_over_tolerance"],
            "rows": {f"{e['workload']}|{e['mode']}|{e['grad_layout']}" + (f"|v{e['variant']}" if "variant" in e else ""):
                     [round(e["kernel_ms"], 4), round(e["gbps"], 1), round(e["frac_of_nominal_8TBps"], 3),
                      e.get("verified", {}).get("elements"), e.get("verified", {}).get("max_err_over_tolerance")]
                     for e in out["also"]}}
    return out


def run_cfg5_subset(psync, args, dev, stream, peak):
    """Ten points of BASELINE.json's cfg5 sweep in the default run: every P at (N, b) = (100, 10) over M = 64 ragged
    servers, and every P at (N, b) = (8, 0) on a single shard -- the two ends of the N+b axis.  3 warm-up + 5 timed steps
    each, each point checked against the oracle like every other timed configuration.  The full 40-point table is
    `bench.py --config cfg5` (profiles/)."""
    rows = {}
    for cfg in synth.sweep_configs():
        if not ((cfg.N == 100 and cfg.M == 64) or (cfg.N == 8 and cfg.M == 1)):
            continue
        set_bytes = cfg.W * cfg.P * cfg.grad_bytes
        if torch.cuda.mem_get_info()[0] < 1.05 * (set_bytes + 5 * 4 * cfg.P):
            rows[cfg.name.replace("cfg5_", "")] = "skipped: not enough free HBM next to the headline workload"
            continue
        wl = Workload(psync, cfg, dev, 3 if set_bytes < 20e9 else 2)
        m = measure(psync, args, wl, "first_n", 5, 3, stream, probe_every=1)
        e = short_entry(cfg, "first_n", "flat", m, peak)
        l2 = "L2" if cfg.footprint_bytes <= L2_BYTES else ("~L2" if set_bytes < 4 * L2_BYTES else "HBM")
        rows[cfg.name.replace("cfg5_", "")] = [round(e["kernel_ms"] * 1e3, 2), round(e["gbps"], 1),
                                               round(e["frac_of_nominal_8TBps"], 3), l2,
                                               e.get("verified", {}).get("elements"),
                                               e.get("verified", {}).get("max_err_over_tolerance")]
        del wl, m
        torch.cuda.empty_cache()
    return {"columns": ["kernel_us", "GB/s of algorithmic bytes", "frac_of_nominal_8TBps",
                        "served from (HBM / ~L2 = one gradient set < 4 x L2 / L2 = footprint fits L2)",
                        "verified_elements", "max_err_over_tolerance"],
            "timing": "3 warm-up + 5 timed steps per point, fused kernel by CUDA events, gradient sets rotated when two fit",
            "rows": rows}


def run_sweep(args, rank, world, dist):
    """--config cfg5: BASELINE.json's bandwidth sweep -- P in {1,4,16,64,256} Mi, M in {1, 64 ragged}, (N,b) in
    {(8,0),(16,2),(50,5),(100,10)}, fp32 gradients ~U[-1,1], SGD + EMA, 5 timed steps each after 3 warm-up steps,
    fresh arrival times per step, gradient sets rotated whenever two fit.  One JSON line with every point; --sweep-md
    writes the GB/s-vs-P-and-(N+b) table as markdown.  A point whose gradient set is smaller than 4x the 126 MB L2 is
    flagged: part of it is served from L2, so it is not an HBM number."""
    import paper_1702_05800_b200 as psync

    local = env_int("LOCAL_RANK", 0)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    stream = torch.cuda.Stream(device=dev)
    peak, peak_src = load_peaks()
    points = []
    K, Wm = args.sweep_steps, 3
    for cfg in synth.sweep_configs():
        if args.sweep_filter and args.sweep_filter not in cfg.name:
            continue
        set_bytes = cfg.W * cfg.P * cfg.grad_bytes
        wl = Workload(psync, cfg, dev, 3 if set_bytes < 20e9 else 2, layout=args.layout)
        # --mode async sweeps Alg. 2's one-pass kernel instead: all N+b gradients applied one at a time (K = N+b)
        sweep_mode = args.mode if args.mode in ("first_n", "async") else "first_n"
        m = measure(psync, args, wl, sweep_mode, K, Wm, stream, dist, variant=args.variant, probe_every=1)
        e = short_entry(cfg, sweep_mode, args.layout, m, peak)
        e["grad_sets"] = wl.n_sets
        e["gradient_set_bytes"] = set_bytes
        e["l2"] = ("L2-resident: the whole footprint fits the 126 MB L2" if cfg.footprint_bytes <= L2_BYTES else
                   ("partly L2-served: one gradient set is smaller than 4 x L2" if set_bytes < 4 * L2_BYTES else "HBM"))
        points.append(e)
        del wl
        torch.cuda.empty_cache()
    big = max(points, key=lambda e: e["algorithmic_bytes_per_launch"])
    units, max_ms = aggregate_over_ranks(big["value"] * big["step_ms"] * 1e-3 * K, big["step_ms"] * K, dist)
    out = {"metric": METRIC, "value": units / (max_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
           "ms_per_step": big["step_ms"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic",
           "config": {"workload": f"cfg5 bandwidth sweep, {len(points)} points; value = the largest point "
                                  f"({big['workload']})", "grad_layout": args.layout,
                      "l2": "every point flagged: HBM / partly L2-served / L2-resident"},
           "roofline": {"bound": "hbm", "achieved": big["gbps"], "peak": peak, "unit": "GB/s", "frac": big["frac"],
                        "traffic": None, "peak_source": peak_src, "kernel": big["kernel"],
                        "algorithmic_bytes_per_launch": big["algorithmic_bytes_per_launch"]},
           "clocks": big["clocks"], "gpu_launches": 2 * K * len(points), "points": points}
    if args.sweep_md and rank == 0:
        write_sweep_md(args.sweep_md, points, peak, peak_src, mode=points[0]["mode"], layout=args.layout)
    return out


def write_sweep_md(path, points, peak, peak_src, mode="first_n", layout="flat"):
    what = ("" if mode == "first_n" else ", Alg. 2 (async: all N+b gradients applied one at a time in one pass)") + \
           ("" if layout == "flat" else ", slices layout")
    flags = ("" if mode == "first_n" else " --mode async") + ("" if layout == "flat" else " --layout slices")
    lines = [f"# cfg5 bandwidth sweep{what}: GB/s of algorithmic bytes (fused kernel, CUDA events) vs P and N+b", "",
             f"Command: `python bench.py --config cfg5{flags} --sweep-md <this file>`; 3 warm-up + 5 timed steps per point, "
             "gradient sets rotated.  Flags: `L2` = whole footprint fits the 126 MB L2, `~L2` = one gradient set is "
             f"smaller than 4 x L2 (partly L2-served); unflagged points stream from HBM.  Peak: {peak} GB/s, {peak_src}.",
             ""]
    for M in sorted({e["M"] for e in points}):
        lines += [f"## M = {M} {'shard' if M == 1 else 'ragged shards'}", "",
                  "| P | " + " | ".join(f"N={N}, b={b} (N+b={N + b})" for N, b in synth.SWEEP_NB) + " |",
                  "|---|" + "---|" * len(synth.SWEEP_NB)]
        for P in synth.SWEEP_P:
            row = [f"{P >> 20} Mi"]
            for N, b in synth.SWEEP_NB:
                e = next((x for x in points if x["M"] == M and x["P"] == P and x["N"] == N and x["b"] == b), None)
                if e is None:
                    row.append("—")
                    continue
                flag = {"L": " `L2`", "p": " `~L2`", "H": ""}[e["l2"][0]]
                row.append(f"{e['gbps']:.0f} ({e['kernel_ms'] * 1e3:.1f} us, {100 * e['frac_of_nominal_8TBps']:.0f} %){flag}")
            lines.append("| " + " | ".join(row) + " |")
        lines.append("")
    with open(path, "w") as fh:
        fh.write("\n".join(lines))


def run_e2e(args, cfg, dev, off, theta, ema, s0, s1, stream, rank, world, dist, mode="first_n"):
    """The same metric through psync_step_host: gradients and arrival times start in pinned HOST memory
    every step, theta(t+1) is read back to the host every step; all copies are inside the timed region."""
    import paper_1702_05800_b200 as psync

    K = max(1, min(args.e2e_steps, args.steps))
    tdt = torch.float32 if cfg.grad_dtype == synth.F32 else torch.bfloat16
    h_grads = []
    tmp = torch.empty(cfg.P, dtype=tdt, device=dev)
    for k in range(cfg.W):          # drawn on the GPU, parked in pinned host memory before timing starts
        synth.gradient(cfg, 1000, k, dev, out=tmp)
        h = torch.empty(cfg.P, dtype=tdt, pin_memory=True)
        h.copy_(tmp)
        h_grads.append(h)
    del tmp
    h_theta = torch.empty(cfg.P, dtype=torch.float32, pin_memory=True)
    h_kept = np.zeros(cfg.N, dtype=np.int32)
    chunk = args.e2e_chunk
    is_async = mode == "async"          # Alg. 2: every gradient that arrived crosses PCIe (nothing is dropped)
    n_moved = cfg.W if is_async else cfg.N
    nbytes = psync.psync_step_host_workspace_bytes(n_moved, cfg.W, cfg.grad_dtype, chunk)
    d_work = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    slices = getattr(args, "layout", "flat") == "slices"
    if slices:   # what each server received, in host memory: W x M slices (here views of the pinned buffers)
        h_grads = [[h[int(off[j]):int(off[j + 1])] for j in range(len(off) - 1)] for h in h_grads]
    step, keep = psync.make_step(off, cfg.N, cfg.W, cfg.grad_dtype, theta, ema, s0, s1, opt=cfg.opt,
                                 ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho,
                                 eps=cfg.eps, grid_ctas=args.grid_ctas, variant=0 if slices else args.variant,
                                 grad_layout=psync.PSYNC_GRADS_SLICES if slices else psync.PSYNC_GRADS_FLAT)
    arrivals = [synth.arrival_times(cfg, 2000 + s) for s in range(K + 1)]
    ctx = psync.HostCtx()               # the copy stream and events, created once for the loop
    def host_step(a):
        if is_async:
            return psync.psync_async_step_host(step, a, h_grads, d_work, h_theta_out=h_theta, chunk_elems=chunk,
                                               stream=stream, ctx=ctx)
        return psync.psync_step_host(step, a, h_grads, d_work, h_theta_out=h_theta, h_kept=h_kept, chunk_elems=chunk,
                                     stream=stream, ctx=ctx)
    host_step(arrivals[K])                                                 # warm-up
    if dist is not None and dist.is_initialized():
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for s in range(K):
        st, _ = host_step(arrivals[s])
        assert st == 0
    torch.cuda.synchronize()
    ms = (time.perf_counter() - t0) * 1e3
    verified = None
    if not getattr(args, "no_verify", False):     # one more host step, outside the timed region, against the oracle
        idx = sample_columns(cfg, off, args.verify_sample)
        d_idx, h_idx = torch.from_numpy(idx).to(dev), torch.from_numpy(idx)
        state = {"theta": theta, "ema": ema, "state0": s0, "state1": s1}
        before = {n: (None if t is None else t[d_idx].cpu().numpy()) for n, t in state.items()}
        a_v = synth.arrival_times(cfg, 2000 + K + 1)
        st, _ = host_step(a_v)
        torch.cuda.synchronize()
        if st != 0:
            raise VerifyError(f"{cfg.name} e2e: status {st}")
        if slices:
            server = np.searchsorted(off, idx, side="right") - 1
            local = torch.from_numpy(idx - off[server])
            bounds = np.searchsorted(server, np.arange(len(off)))
            g_s = [synth.as_numpy_grad(torch.cat([row[j][local[bounds[j]:bounds[j + 1]]] for j in range(len(off) - 1)
                                                  if bounds[j + 1] > bounds[j]])) for row in h_grads]
        else:
            g_s = [synth.as_numpy_grad(h[h_idx]) for h in h_grads]
        verified = verify_step(cfg, off, mode, args.timeout, a_v, g_s, before, state,
                               None if is_async else h_kept[None, :].copy(), None, idx, d_idx)
        got_host = h_theta[h_idx].numpy()                     # what the user reads back: theta(t+1) in host memory
        if not np.array_equal(got_host, theta[d_idx].cpu().numpy()):
            raise VerifyError(f"{cfg.name} e2e: theta read back to the host differs from the device's")
        verified["theta_readback_bit_exact"] = True
    units, max_ms = aggregate_over_ranks(float(n_moved) * cfg.P * K, ms, dist)
    n_chunks = -(-cfg.P // (chunk if chunk else 1 << 20))
    return {"value": units / (max_ms * 1e-3), "unit": UNIT, "steps": K, "ms_per_step": max_ms / K,
            "h2d_bytes_per_step": n_moved * cfg.P * cfg.grad_bytes + 4 * cfg.W,
            "d2h_bytes_per_step": 4 * cfg.P + 4 * cfg.N + 8,
            "api": ("psync_async_step_host" if is_async else "psync_step_host") + " (C ABI, pinned host gradient buffers"
                   + (" as W x M per-(worker, server) slices" if slices else "")
                   + ("; all W arriving buffers cross PCIe)" if is_async else "; only the N kept buffers cross PCIe)"),
            "verified": verified,
            "gpu_launches_per_step": 3 + n_chunks,
            "timing": "host wall clock around synchronous calls (the call returns when theta(t+1) is on the host)"}


def run_instances(args, base_cfg):
    """--instances: every template instance of the kernel of --mode (2 gradient dtypes x 3 optimizers x 3 EMA modes) on the
    shape of --config: kernel ms and GB/s of algorithmic bytes, so that no instance hides behind the three that the
    configs exercise.  One JSON line; --instances-md writes the table."""
    from dataclasses import replace
    import paper_1702_05800_b200 as psync

    dev = torch.device("cuda", env_int("LOCAL_RANK", 0))
    torch.cuda.set_device(dev)
    stream = torch.cuda.Stream(device=dev)
    peak, peak_src = load_peaks()
    mode = args.mode
    rows = []
    for dtype, dname in ((synth.F32, "fp32"), (synth.BF16, "bf16")):
        wl = None
        for opt, oname in ((synth.SGD, "sgd"), (synth.MOMENTUM, "momentum"), (synth.RMSPROP_MOM, "rmsprop_momentum")):
            for ema, ename in ((synth.EMA_POST, "post"), (synth.EMA_PRE, "pre"), (synth.EMA_OFF, "off")):
                cfg = replace(base_cfg, grad_dtype=dtype, opt=opt, ema_mode=ema, mu=0.9, rho=0.9, eps=1.0,
                              name=f"{base_cfg.name}_{dname}_{oname}_ema{ename}")
                if wl is None:                       # one resident gradient set pair per dtype; only the instance changes
                    wl = Workload(psync, replace(cfg, opt=synth.RMSPROP_MOM, ema_mode=synth.EMA_POST), dev, 2, layout=args.layout)
                wl.cfg = cfg
                wl.reset_state()
                m = measure(psync, args, wl, mode, 6, 3, stream, variant=args.variant, probe_every=1)
                e = short_entry(cfg, mode, args.layout, m, peak)
                e.update({"grad_dtype": dname, "optimizer": oname, "ema": ename})
                rows.append(e)
        del wl
        torch.cuda.empty_cache()
    out = {"workload": f"{base_cfg.name}: P={base_cfg.P}, N={base_cfg.N}, b={base_cfg.b}, M={base_cfg.M}", "mode": mode,
           "grad_layout": args.layout, "peak": peak, "peak_source": peak_src, "instances": rows}
    if args.instances_md:
        lines = [f"# Every template instance on {out['workload']} (`--mode {mode}`, layout {args.layout})", "",
                 f"Command: `python bench.py --config {args.config} --mode {mode}"
                 + ("" if args.layout == "flat" else " --layout slices") + (f" --variant {args.variant}" if args.variant else "")
                 + " --instances --instances-md <this file>`; 3 warm-up + 6 "
                 "timed steps each, fused-kernel time from CUDA events; GB/s of algorithmic bytes (of nominal 8 TB/s).", "",
                 "| gradients | optimizer | EMA post | EMA pre | EMA off |", "|---|---|---|---|---|"]
        for dname in ("fp32", "bf16"):
            for oname in ("sgd", "momentum", "rmsprop_momentum"):
                cells = []
                for ename in ("post", "pre", "off"):
                    e = next(r for r in rows if (r["grad_dtype"], r["optimizer"], r["ema"]) == (dname, oname, ename))
                    cells.append(f"{e['kernel_ms']:.4f} ms, {e['gbps']:.0f} ({100 * e['frac_of_nominal_8TBps']:.0f} %)")
                lines.append(f"| {dname} | {oname} | " + " | ".join(cells) + " |")
        with open(args.instances_md, "w") as fh:
            fh.write("\n".join(lines) + "\n")
    return out


def run_probe_pipes(args):
    """--probe-pipes: fp32 lane-operations per clock per SM of the FFMA, packed FFMA2 and MUFU.RSQ pipes (the library's
    psync_probe_pipe), with the SM clock sampled while the probes run.  One JSON line."""
    import paper_1702_05800_b200 as psync

    dev = torch.device("cuda", env_int("LOCAL_RANK", 0))
    torch.cuda.set_device(dev)
    B = psync.binding
    st = torch.cuda.Stream(device=dev)
    sink = torch.zeros(4, dtype=torch.float32, device=dev)
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    out = {"sms": sms, "unit": "fp32 lane-operations per clock per SM", "pipes": {}}
    sampler = ClockSampler(env_int("LOCAL_RANK", 0), period_s=0.002)
    sampler.start()
    for name, mode, iters in (("ffma", 0, 1 << 16), ("ffma2_packed", 1, 1 << 16), ("mufu_rsqrt", 2, 1 << 14)):
        B.psync_probe_pipe(mode, 256, sink, st)                      # warm-up
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        ops = B.psync_probe_pipe(mode, iters, sink, st)
        e1.record(st)
        st.synchronize()
        out["pipes"][name] = {"lane_ops": ops, "ms": e0.elapsed_time(e1)}
    clocks = sampler.stop()
    mhz = clocks.get("sm_mhz") or clocks.get("sm_max_mhz")
    for v in out["pipes"].values():
        v["per_clock_per_sm"] = v["lane_ops"] / (v["ms"] * 1e-3) / (mhz * 1e6) / sms
    out["clocks"] = clocks
    return out


def run_launch_bound(args):
    """--launch-bound: the cost of a step when the kernels take ~2 us (cfg1, P = 4096): host calls per step, in us, for the
    synchronous step (two binding calls; psync_step_device; 100 steps replayed from a CUDA graph) and for one batch of
    Alg. 2 (psync_async_step_device eager / graph; one order, and one order per server).  Host wall clock over many steps
    between synchronisations.  One JSON line."""
    import paper_1702_05800_b200 as psync

    cfg, dev = synth.TINY, torch.device("cuda", env_int("LOCAL_RANK", 0))
    torch.cuda.set_device(dev)
    B = psync.binding
    off = synth.shard_offsets(cfg)
    grads = [synth.gradient(cfg, 0, k, dev) for k in range(cfg.W)]
    arr = torch.from_numpy(np.stack([synth.arrival_times(cfg, s) for s in range(100)])).to(dev)
    arr_rows = arr[:, None, :].repeat(1, cfg.M, 1).contiguous()
    n_eager, n_replay = 2000, 20
    st = torch.cuda.Stream(device=dev)
    st.wait_stream(torch.cuda.current_stream())

    def timed(fn, n):
        for i in range(20):
            fn(i)
        st.synchronize()
        t0 = time.perf_counter()
        for i in range(n):
            fn(i)
        st.synchronize()
        return (time.perf_counter() - t0) / n * 1e6

    def graph_of(fn):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            for i in range(100):
                fn(i)
        g.replay()
        st.synchronize()
        t0 = time.perf_counter()
        for _ in range(n_replay):
            g.replay()
        st.synchronize()
        return (time.perf_counter() - t0) / (100 * n_replay) * 1e6

    out = {"workload": f"cfg1 {cfg.name}: P={cfg.P}, M={cfg.M}, N={cfg.N}, b={cfg.b}", "unit": "us per step (host wall clock)",
           "steps_eager": n_eager, "steps_graph": 100 * n_replay}
    with torch.cuda.stream(st):
        for per_server in (False, True):
            theta = synth.init_theta(cfg, dev)
            ps = psync.ParameterServerStep(off, cfg.N, cfg.b, theta, theta.clone(), None, None, cfg.opt, cfg.ema_mode,
                                           alpha=cfg.alpha, per_server=per_server)
            ps.set_gradients(grads)
            a = arr_rows if per_server else arr
            key = "sync_per_server" if per_server else "sync"
            out[key] = {"step_device_eager": timed(lambda i: ps.step(a[i % 100], cfg.gamma, stream=st), n_eager),
                        "step_device_graph": graph_of(lambda i: ps.step(a[i], cfg.gamma, stream=st))}
            if not per_server:
                def two_calls(i):
                    B.psync_select_first_n(a[i % 100], cfg.N, cfg.b, ps.d_kept, ps.d_status, ps.d_t_nth, None, 0, st)
                    ps.aggregate_only(cfg.gamma, stream=st)
                out[key]["two_binding_calls_eager"] = timed(two_calls, n_eager)
            srv = psync.AsyncServerStep(off, cfg.W, theta, theta.clone(), None, None, cfg.opt, alpha=cfg.alpha,
                                        per_server=per_server)
            srv.set_gradients(grads)
            key = "async_per_server" if per_server else "async"
            out[key] = {"async_step_device_eager": timed(lambda i: srv.apply(a[i % 100], cfg.gamma, stream=st), n_eager),
                        "async_step_device_graph": graph_of(lambda i: srv.apply(a[i], cfg.gamma, stream=st))}
    return out


# ------------------------------------------------------------------------------------ main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="psync", choices=["psync", "reference"])
    ap.add_argument("--config", default="cfg3", choices=sorted(WORKLOADS) + ["cfg5"],
                    help="cfg5 = the bandwidth sweep (one JSON line with every point)")
    ap.add_argument("--layout", default="flat", choices=["flat", "slices"],
                    help="flat: W flat gradient buffers; slices: W*M separately allocated per-(worker, server) slices")
    ap.add_argument("--servers", type=int, default=0, help="override M (ragged cut into that many servers)")
    ap.add_argument("--no-worklist", action="store_true",
                    help="--mode per_server with flat buffers: tiles of the flat index space instead of the work list")
    ap.add_argument("--hold-cached-block", action="store_true",
                    help="experiment: leave one freed 100 MB block in torch's caching allocator while timing (2-3 %% slower)")
    ap.add_argument("--no-also", action="store_true", help="skip the short measurements of the other configs / modes")
    ap.add_argument("--also-steps", type=int, default=8)
    ap.add_argument("--sweep-steps", type=int, default=5)
    ap.add_argument("--sweep-md", default="", help="--config cfg5: also write the table as markdown to this path")
    ap.add_argument("--sweep-filter", default="", help="--config cfg5: only points whose name contains this")
    ap.add_argument("--mode", default="first_n", choices=["first_n", "per_server", "timeout", "async", "async_per_server"],
                    help="first_n: the headline (one kept set); per_server: Alg. 4 per server j; timeout: L259; "
                         "async: Alg. 2, all W gradients one at a time in one pass")
    ap.add_argument("--timeout", type=float, default=1.5, help="seconds, for --mode timeout")
    ap.add_argument("--clip", type=float, default=0.0, help="--mode async: global-norm clip bound (0 = off)")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--grid-ctas", type=int, default=0)
    ap.add_argument("--grad-sets", type=int, default=3)
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--e2e-chunk", type=int, default=1 << 22,
                    help="elements of each worker staged per chunk in psync_step_host (16 MB copies: 54 GB/s over "
                         "PCIe on this box against 52 GB/s with the library default of 2^20)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-probe", action="store_true", help="skip the live HBM stream probes")
    ap.add_argument("--no-cfg5", action="store_true", help="skip the 10-point cfg5 subset of the default run")
    ap.add_argument("--no-verify", action="store_true", help="skip the oracle check of every timed configuration")
    ap.add_argument("--verify-sample", type=int, default=20_000, help="random columns checked per configuration "
                    "(+ first / last tile and every shard cut)")
    ap.add_argument("--fault", default="", choices=["", "worklist"], help="test hook: break the named input on purpose "
                    "(worklist: a (server, tile) list built for the other gradient dtype) -- the run must exit non-zero")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--cpu-seconds-1thread", type=float, default=3.0)
    ap.add_argument("--clock-period-ms", type=float, default=2.0)
    ap.add_argument("--probe-every", type=int, default=4)
    ap.add_argument("--instances", action="store_true",
                    help="every template instance (dtype x optimizer x EMA mode) of --mode's kernel on --config's shape")
    ap.add_argument("--instances-md", default="", help="--instances: also write the table as markdown to this path")
    ap.add_argument("--probe-pipes", action="store_true",
                    help="FFMA / packed FFMA2 / MUFU.RSQ lane-operations per clock per SM (psync_probe_pipe)")
    ap.add_argument("--launch-bound", action="store_true",
                    help="cfg1 (P = 4096): us per step of the host calls, eager and replayed from a CUDA graph")
    ap.add_argument("--ref-sample-elems", type=int, default=0,
                    help="--impl reference: run on the first this-many parameters only (0 = the full workload)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "psync":
        args.warmup = 3                     # timing rule: at least 3 warm-up steps
    cfg = WORKLOADS.get(args.config, synth.PAPER_RMSPROP)
    rank, world = env_int("RANK", 0), env_int("WORLD_SIZE", 1)

    if args.impl == "reference":
        if rank != 0:
            return 0                        # the oracle runs on rank 0 alone
        if args.ref_sample_elems <= 0 and args.steps + args.warmup > 400:
            args.ref_sample_elems = 1 << 22  # an unusually long run: keep it within a few minutes of host time
        print(json.dumps(run_reference(args, cfg, rank)), flush=True)
        return 0

    if args.gpus != world:                  # --gpus only NAMES the replica count; torchrun makes the replicas
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE is {world}: the step does not shard across GPUs, N GPUs are "
              f"N independent replicas, one process each.  Launch them with\n  python -m torch.distributed.run "
              f"--nnodes=1 --nproc-per-node {args.gpus} --master-addr 127.0.0.1 --master-port 29500 bench.py --gpus "
              f"{args.gpus} ...", file=sys.stderr)
        return 2
    if args.launch_bound:
        if rank == 0:
            print(json.dumps(run_launch_bound(args)), flush=True)
        return 0
    if args.probe_pipes:
        if rank == 0:
            print(json.dumps(run_probe_pipes(args)), flush=True)
        return 0
    if args.instances:
        if rank == 0:
            print(json.dumps(run_instances(args, cfg)), flush=True)
        return 0

    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        torch.cuda.set_device(env_int("LOCAL_RANK", 0))
        dist_mod.init_process_group(backend="nccl")
        dist = dist_mod
    try:
        out = run_sweep(args, rank, world, dist) if args.config == "cfg5" else run_psync(args, cfg, rank, world, dist)
        if rank == 0:
            print(json.dumps(out), flush=True)
    finally:
        if dist is not None and dist.is_initialized():
            dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
