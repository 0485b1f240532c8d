"""cfg5 of BASELINE.json: the bandwidth sweep.  `python -m paper_1702_05800_b200.sweep [--out FILE.md]`

P in {1,4,16,64,256} Mi fp32 parameters, single shard and M=64 ragged shards, (N,b) in
{(8,0),(16,2),(50,5),(100,10)}, fp32 gradients ~U[-1,1], SGD gamma=0.01 + EMA alpha=0.999, 5 timed
steps each (after 3 warm-up steps), fresh arrival times per step.  Reports GB/s (north_star bytes
model) against P and N+b.  Points whose whole working set fits the 126 MB L2 are flagged: they are
not HBM numbers.  Cases above 170 GB of HBM are skipped (none is).
"""
from __future__ import annotations

import argparse
import json
import sys

import numpy as np
import torch

from . import binding as B
from . import synth
from .server import ParameterServerStep

L2_BYTES = 126 * 10**6


def run_point(cfg: synth.Config, dev, steps: int, warmup: int = 3) -> dict:
    off = synth.shard_offsets(cfg)
    bufs = [torch.empty(cfg.P, dtype=torch.float32, device=dev) for _ in range(cfg.W)]
    for k in range(cfg.W):
        synth.gradient(cfg, 0, k, dev, out=bufs[k])
    theta = synth.init_theta(cfg, dev)
    ema = theta.clone()
    ps = ParameterServerStep(off, cfg.N, cfg.b, theta, ema, None, None, cfg.opt, cfg.ema_mode, alpha=cfg.alpha)
    ps.set_gradients(bufs)
    arrivals = torch.from_numpy(np.stack([synth.arrival_times(cfg, s) for s in range(steps + warmup)])).to(dev)
    stream = torch.cuda.current_stream()
    for s in range(warmup):
        ps.step(arrivals[s], cfg.gamma, stream=stream)
    torch.cuda.synchronize()
    # pass 1: the steps as a user runs them (selection + fused launch back to back), one event pair
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for s in range(steps):
        ps.step(arrivals[warmup + s], cfg.gamma, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    assert int(ps.d_status.item()) == 0
    step_ms = e0.elapsed_time(e1) / steps
    # pass 2: the fused kernel alone between events
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(steps)]
    for s in range(steps):
        B.psync_select_first_n(arrivals[warmup + s], cfg.N, cfg.b, ps.d_kept, ps.d_status, ps.d_t_nth, None, 0, stream)
        evs[s][0].record(stream)
        ps.aggregate_only(cfg.gamma, stream)
        evs[s][1].record(stream)
    torch.cuda.synchronize()
    fused_ms = float(np.median([e[0].elapsed_time(e[1]) for e in evs]))
    return {"name": cfg.name, "P": cfg.P, "M": cfg.M, "N": cfg.N, "b": cfg.b, "W": cfg.W,
            "bytes_per_step": cfg.bytes_per_step, "footprint": cfg.footprint_bytes, "step_ms": step_ms,
            "fused_ms": fused_ms, "gbps_step": cfg.bytes_per_step / step_ms / 1e6,
            "gbps_fused": cfg.bytes_per_step / fused_ms / 1e6,
            "grad_elems_per_s": cfg.N * cfg.P / (step_ms * 1e-3),
            "l2_resident": cfg.footprint_bytes <= L2_BYTES}


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=None)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--max-bytes", type=float, default=synth.HBM_LIMIT_BYTES)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise RuntimeError("the sweep needs a CUDA device")
    dev = torch.device("cuda", 0)
    rows = []
    for cfg in synth.sweep_configs():
        free, _ = torch.cuda.mem_get_info()
        if cfg.footprint_bytes > args.max_bytes or cfg.footprint_bytes + cfg.P * 8 > 0.97 * free:
            rows.append({"name": cfg.name, "skipped": f"footprint {cfg.footprint_bytes / 1e9:.1f} GB"})
            continue
        rows.append(run_point(cfg, dev, args.steps))
        torch.cuda.empty_cache()
        print(json.dumps(rows[-1]), file=sys.stderr, flush=True)
    lines = ["| P | M | N | b | N+b | bytes/step | step ms | fused ms | GB/s (step) | GB/s (fused kernel) | note |",
             "|---:|---:|---:|---:|---:|---:|---:|---:|---:|---:|---|"]
    for r in rows:
        if "skipped" in r:
            lines.append(f"| {r['name']} | | | | | | | | | | skipped: {r['skipped']} |")
            continue
        note = "L2-resident (not an HBM number)" if r["l2_resident"] else ""
        lines.append(f"| {r['P'] >> 20} Mi | {r['M']} | {r['N']} | {r['b']} | {r['W']} | {r['bytes_per_step'] / 1e9:.3f} GB | "
                     f"{r['step_ms']:.4f} | {r['fused_ms']:.4f} | {r['gbps_step']:.0f} | {r['gbps_fused']:.0f} | {note} |")
    text = "\n".join(lines) + "\n"
    if args.out:
        with open(args.out, "w") as fh:
            fh.write(text)
    print(text)
    return 0


if __name__ == "__main__":
    sys.exit(main())
