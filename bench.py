#!/usr/bin/env python
"""bench.py -- whole-job throughput of the parameter-server step (Alg. 4) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg3] [--impl psync|reference]

A "step" is one pass of the whole hot path -- psync_select_first_n then the fused
psync_aggregate_update (sum of the N kept gradients, optimizer update, EMA) -- over one batch of
synthetic input (fresh arrival times every step, gradient buffers rotated over several resident
sets far larger than L2).  Prints ONE JSON line (rank 0).  Metric: aggregated gradient elements
per second = N * P * steps / time; GB/s uses north_star's bytes model
N*P*sizeof(grad) + P*8*(1 + n_state + 1).

Multi-GPU (--gpus N under torchrun): the step does not shard across GPUs (north_star: no
collectives) -> N independent replicas, weak scaling; value = units of all ranks / max-over-ranks
time.  `--impl reference` times the CPU oracle (oracle/) on the host cores on a bounded sample.
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
def oracle_sample(cfg, seconds_budget=12.0, sample_elems=1 << 22, max_steps=2000, warmup=0, fixed_steps=None,
                  wall_budget=60.0):
    """Times the oracle AS IT STANDS on the host cores on a bounded sample of the workload: the first
    `sample_elems` parameters of every buffer (same N, b, M-way ragged cut, optimizer, distributions).
    The W gradient buffers of the sample are drawn once (not timed); every step has fresh arrival
    times, hence a fresh kept set, and continues from the previous step's theta / state / ema.
    Runs `fixed_steps` steps, else until `seconds_budget` seconds of oracle time (or `wall_budget`
    seconds of wall clock).  Returns (grad-elements/s, info)."""
    import oracle  # the one place bench.py executes oracle/ (cpu_baseline / --impl reference)

    Ps = int(min(sample_elems, cfg.P))
    sub = synth.scaled(cfg, Ps, name=cfg.name + "_sample")
    off = synth.shard_offsets(sub)
    theta = synth.init_theta(sub).numpy().copy()
    s0, s1 = synth.init_state(sub)
    s0 = None if s0 is None else s0.numpy().copy()
    s1 = None if s1 is None else s1.numpy().copy()
    ema = theta.copy()
    t_begin = time.perf_counter()
    grads = [synth.as_numpy_grad(synth.gradient(sub, 0, k)) for k in range(sub.W)]   # not timed
    times = []
    total_steps = (fixed_steps + warmup) if fixed_steps is not None else max_steps
    for s in range(total_steps):
        arrival = synth.arrival_times(sub, s)
        t0 = time.perf_counter()
        st, kept, _ = oracle.select_first_n(arrival, sub.N, sub.b)
        rc = oracle.aggregate_update(off, sub.N, grads, kept, theta, ema, s0, s1, opt=sub.opt, ema_mode=sub.ema_mode,
                                     gamma_t=sub.gamma, alpha=sub.alpha, mu=sub.mu, rho=sub.rho, eps=sub.eps)
        t1 = time.perf_counter()
        assert st == 0 and rc == 0
        if s >= warmup:
            times.append(t1 - t0)
        if fixed_steps is None and times and (sum(times) > seconds_budget or t1 - t_begin > wall_budget):
            break
    sec = float(np.sum(times))
    value = sub.N * Ps * len(times) / sec
    info = {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"first {Ps} of P={cfg.P} parameters of every buffer, N={cfg.N} b={cfg.b}, "
                      f"{len(times)} steps, {sec:.2f} s of oracle time (select + aggregate/update/EMA; "
                      f"input generation excluded)",
            "ms_per_step_sample": 1e3 * sec / len(times),
            "gbps": sub.bytes_per_step * len(times) / sec / 1e9}
    return value, info


def run_reference(args, cfg, rank):
    """--impl reference: the oracle on the host cores, K steps of a bounded sample, same metric."""
    if rank != 0:
        return None
    value, info = oracle_sample(cfg, sample_elems=args.ref_sample_elems, warmup=args.warmup, fixed_steps=args.steps)
    return {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": info["ms_per_step_sample"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64 arithmetic on f32 storage", "data": "synthetic",
            "config": workload_config(cfg, extra={"sample": info["sample"]}),
            "cpu_baseline": {k: info[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def workload_config(cfg, extra=None):
    c = {"workload": f"{cfg.name}: P={cfg.P} fp32 params in M={cfg.M} ragged shards, N={cfg.N}, b={cfg.b}, "
                     f"{'bf16' if cfg.grad_dtype == synth.BF16 else 'fp32'} gradients, {OPT_NAME[cfg.opt]}, EMA",
         "P": cfg.P, "M": cfg.M, "N": cfg.N, "b": cfg.b, "optimizer": OPT_NAME[cfg.opt],
         "grad_dtype": "bf16" if cfg.grad_dtype == synth.BF16 else "fp32", "gamma": cfg.gamma, "alpha": cfg.alpha,
         "bytes_per_step_model": cfg.bytes_per_step, "parallelism": "replicas only (no sharding across GPUs)"}
    if extra:
        c.update(extra)
    return c


# ------------------------------------------------------------------------------------ the CUDA arm
def run_psync(args, cfg, rank, world, dist):
    import paper_1702_05800_b200 as psync

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU path")
    local = env_int("LOCAL_RANK", 0)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    K, Wm = args.steps, args.warmup
    off = synth.shard_offsets(cfg)
    # resident gradient sets, rotated step by step: every step streams buffers it did not just touch
    set_bytes = cfg.W * cfg.P * cfg.grad_bytes
    free, _ = torch.cuda.mem_get_info()
    n_sets = int(max(1, min(args.grad_sets, (0.7 * free) // max(set_bytes, 1))))
    tdt = torch.float32 if cfg.grad_dtype == synth.F32 else torch.bfloat16
    tables = []
    for r in range(n_sets):
        bufs = [torch.empty(cfg.P, dtype=tdt, device=dev) for _ in range(cfg.W)]
        for k in range(cfg.W):
            synth.gradient(cfg, r, k, dev, out=bufs[k])
        tables.append(psync.make_grad_table(bufs))
    theta = synth.init_theta(cfg, dev)
    s0, s1 = synth.init_state(cfg, dev)
    ema = theta.clone()
    ps = psync.ParameterServerStep(off, cfg.N, cfg.b, theta, ema, s0, s1, cfg.opt, cfg.ema_mode, alpha=cfg.alpha,
                                   mu=cfg.mu, rho=cfg.rho, eps=cfg.eps, grid_ctas=args.grid_ctas, variant=args.variant)

    # --mode first_n (default, the headline): one kept set of N per step (reading R11).
    # --mode per_server: Alg. 4 per server j, arrival [M][W] -> kept [M][N] (NEXT-1).
    # --mode timeout: keep every worker that arrived by --timeout seconds, divide by the count (NEXT-2).
    mode = args.mode
    rows = cfg.M if mode == "per_server" else 1
    if mode == "per_server":
        arr_np = np.stack([synth.arrival_times_per_server(cfg, s) for s in range(K + Wm)])
    else:
        arr_np = np.stack([synth.arrival_times(cfg, s) for s in range(K + Wm)])
    arrivals = torch.from_numpy(arr_np).to(dev)
    # --mode async: Alg. 2 -- all W gradients applied one at a time in arrival order, one pass (NEXT-3).
    stride = cfg.W if mode in ("timeout", "async") else cfg.N
    d_kept = torch.full((rows, stride), -1, dtype=torch.int32, device=dev) if mode != "first_n" else ps.d_kept
    d_status = torch.full((rows,), 0 if mode == "async" else -9, dtype=torch.int32,
                          device=dev) if mode != "first_n" else ps.d_status
    d_n_kept = torch.zeros(rows, dtype=torch.int32, device=dev) if mode in ("timeout", "async") else None
    d_off = torch.from_numpy(off).to(dev) if mode == "per_server" else None
    steps_struct = []
    for tb in tables:   # one psync_step per gradient set, built once (marshalling outside the timed region)
        st, keep = psync.make_step(off, cfg.N, cfg.W, tb.grad_dtype, theta, ema, s0, s1, opt=cfg.opt,
                                   ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho,
                                   eps=cfg.eps, d_grads=tb.d_ptrs, d_kept=d_kept, d_status=d_status,
                                   grid_ctas=args.grid_ctas, variant=args.variant, per_shard=(mode == "per_server"),
                                   d_shard_off=d_off, d_n_kept=d_n_kept)
        steps_struct.append((st, keep))
    geo = psync.psync_launch_geometry(steps_struct[0][0])
    d_scales = d_clip_work = None
    if mode == "async" and args.clip > 0:
        d_scales = torch.ones(cfg.W, dtype=torch.float32, device=dev)
        d_clip_work = torch.empty(psync.psync_clip_workspace_bytes(cfg.W, cfg.P, cfg.grad_dtype) // 8,
                                  dtype=torch.float64, device=dev)

    stream = torch.cuda.Stream(device=dev)
    stream.wait_stream(torch.cuda.current_stream())    # tables, kept[] and status were filled on the default stream
    B = psync.binding

    def select(i):
        if mode == "first_n":
            B.psync_select_first_n(arrivals[i], cfg.N, cfg.b, ps.d_kept, ps.d_status, ps.d_t_nth, None, i, stream)
        elif mode == "per_server":
            B.psync_select_first_n_sharded(arrivals[i], cfg.N, cfg.b, cfg.M, d_kept, d_status, None, None, i, stream)
        elif mode == "timeout":
            B.psync_select_timeout(arrivals[i], cfg.W, args.timeout, d_kept, d_n_kept, d_status, stream=stream)
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
        if mode == "async":
            if args.clip > 0:            # A.3 (L313): global-norm clipping = one more pass over the W buffers
                B.psync_clip_scales(tables[i % n_sets], args.clip, d_scales, d_clip_work, stream)
            B.psync_async_apply(st, None, stream, d_gscale=d_scales if args.clip > 0 else None)
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
    probe_every = max(1, args.probe_every)
    evs = {k: [torch.cuda.Event(enable_timing=True) for _ in range(3)] for k in range(0, K, probe_every)}
    e_begin, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local, period_s=args.clock_period_ms * 1e-3)
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
    assert bool((d_status == 0).all()) and bool(torch.isfinite(theta[:4096]).all())

    # gradient elements aggregated per step: N*P, or (workers in time)*P for the time-out rule
    if mode == "async":
        n_eff = float(cfg.W)                 # every gradient is applied (nothing is dropped in Alg. 2)
    elif mode == "timeout":
        n_eff = float(np.mean([(arr_np[Wm + k] <= args.timeout).sum() for k in range(K)]))
    else:
        n_eff = float(cfg.N)
    bytes_per_step = cfg.bytes_per_step + (n_eff - cfg.N) * cfg.P * cfg.grad_bytes
    if mode == "async" and args.clip > 0:
        bytes_per_step += cfg.W * cfg.P * cfg.grad_bytes      # the norm pass reads every buffer once more
    units_local = n_eff * cfg.P * K
    units, max_ms = aggregate_over_ranks(units_local, total_ms, dist)
    value = units / (max_ms * 1e-3)
    peak, peak_src = load_peaks()
    achieved = bytes_per_step / (fused_ms * 1e-3) / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": max_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if cfg.grad_dtype == synth.F32 else "f32 (bf16 gradients widened exactly)",
        "data": "synthetic",
        "config": workload_config(cfg, extra={
            "l2": f"no flush: each step streams {cfg.bytes_per_step / 1e9:.2f} GB (>> 126 MB L2) and gradient "
                  f"buffers rotate over {n_sets} resident sets",
            "grad_sets": n_sets, "launch": geo, "variant": args.variant, "mode": mode,
            "kept_per_step": n_eff}),
        "gbps_model": bytes_per_step * K * world / (max_ms * 1e-3) / 1e9,
        "params_per_s": float(cfg.P) * K * world / (max_ms * 1e-3),
        "select_ms": select_ms, "fused_ms": fused_ms, "kernel_events_on_steps": len(fused_list),
        "fused_ms_min_median_max": [float(np.min(fused_list)), float(np.median(fused_list)), float(np.max(fused_list))],
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": None, "peak_source": peak_src, "kernel": "async_apply_kernel" if mode == "async" else "fused_aggregate_update_ema",
                     "algorithmic_bytes_per_launch": bytes_per_step,
                     "frac_of_nominal_8TBps": achieved / 8000.0},
        "clocks": clocks,
        "gpu_launches": 2 * K,
    }
    traffic_file = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(traffic_file) and mode == "first_n":   # dram bytes per launch from the committed ncu --set full capture
        try:
            with open(traffic_file) as fh:
                out["roofline"]["traffic"] = json.load(fh).get(cfg.name)
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

    # free the resident gradient sets before the host-buffer (e2e) leg
    del tables, steps_struct
    torch.cuda.empty_cache()
    if not args.no_e2e and mode == "first_n":
        out["e2e"] = run_e2e(args, cfg, dev, off, theta, ema, s0, s1, stream, rank, world, dist)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        _, info = oracle_sample(cfg, seconds_budget=args.cpu_seconds, sample_elems=1 << 22)
        out["cpu_baseline"] = {k: info[k] for k in ("value", "unit", "cores", "kind", "sample")}
        if args.cpu_seconds_1thread > 0:       # the oracle single-threaded as well (a short sample)
            import oracle
            threads = oracle.num_threads()
            oracle.set_num_threads(1)
            try:
                v1, info1 = oracle_sample(cfg, seconds_budget=args.cpu_seconds_1thread, sample_elems=1 << 20,
                                          wall_budget=20.0)
            finally:
                oracle.set_num_threads(threads)
            out["cpu_baseline"]["value_1thread"] = v1
            out["cpu_baseline"]["sample_1thread"] = info1["sample"]
    return out


def run_e2e(args, cfg, dev, off, theta, ema, s0, s1, stream, rank, world, dist):
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
    nbytes = psync.psync_step_host_workspace_bytes(cfg.N, cfg.W, cfg.grad_dtype, chunk)
    d_work = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    step, keep = psync.make_step(off, cfg.N, cfg.W, cfg.grad_dtype, theta, ema, s0, s1, opt=cfg.opt,
                                 ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho,
                                 eps=cfg.eps, grid_ctas=args.grid_ctas, variant=args.variant)
    arrivals = [synth.arrival_times(cfg, 2000 + s) for s in range(K + 1)]
    psync.psync_step_host(step, arrivals[K], h_grads, d_work, h_theta_out=h_theta, h_kept=h_kept, chunk_elems=chunk,
                          stream=stream)                                   # warm-up
    if dist is not None and dist.is_initialized():
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for s in range(K):
        st, _ = psync.psync_step_host(step, arrivals[s], h_grads, d_work, h_theta_out=h_theta, h_kept=h_kept,
                                      chunk_elems=chunk, stream=stream)
        assert st == 0
    torch.cuda.synchronize()
    ms = (time.perf_counter() - t0) * 1e3
    units, max_ms = aggregate_over_ranks(float(cfg.N) * cfg.P * K, ms, dist)
    n_chunks = -(-cfg.P // (chunk if chunk else 1 << 20))
    return {"value": units / (max_ms * 1e-3), "unit": UNIT, "steps": K, "ms_per_step": max_ms / K,
            "h2d_bytes_per_step": cfg.N * cfg.P * cfg.grad_bytes + 4 * cfg.W,
            "d2h_bytes_per_step": 4 * cfg.P + 4 * cfg.N + 8,
            "api": "psync_step_host (C ABI, pinned host gradient buffers; only the N kept buffers cross PCIe)",
            "gpu_launches_per_step": 3 + n_chunks,
            "timing": "host wall clock around synchronous calls (the call returns when theta(t+1) is on the host)"}


# ------------------------------------------------------------------------------------ main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="psync", choices=["psync", "reference"])
    ap.add_argument("--config", default="cfg3", choices=sorted(WORKLOADS))
    ap.add_argument("--mode", default="first_n", choices=["first_n", "per_server", "timeout", "async"],
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
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--cpu-seconds-1thread", type=float, default=3.0)
    ap.add_argument("--clock-period-ms", type=float, default=2.0)
    ap.add_argument("--probe-every", type=int, default=4)
    ap.add_argument("--ref-sample-elems", type=int, default=0)
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "psync":
        args.warmup = 3                     # timing rule: at least 3 warm-up steps
    cfg = WORKLOADS[args.config]
    rank, world = env_int("RANK", 0), env_int("WORLD_SIZE", 1)

    if args.impl == "reference":
        if rank != 0:
            return 0                        # the oracle runs on rank 0 alone
        if args.ref_sample_elems <= 0:      # bounded sample: K steps stay within a few minutes of host time
            elems = int((1 << 22) * min(1.0, 60.0 / max(1, args.steps + args.warmup)))
            args.ref_sample_elems = max(1 << 14, (elems >> 14) << 14)
        print(json.dumps(run_reference(args, cfg, rank)), flush=True)
        return 0

    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        torch.cuda.set_device(env_int("LOCAL_RANK", 0))
        dist_mod.init_process_group(backend="nccl")
        dist = dist_mod
    try:
        out = run_psync(args, cfg, rank, world, dist)
        if rank == 0:
            print(json.dumps(out), flush=True)
    finally:
        if dist is not None and dist.is_initialized():
            dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
