"""CPU-only tests of bench.py's host logic: the N>1 aggregation (world_size 2, gloo), the reference
arm's JSON contract and rank gating, and the bytes model of the configs."""
import json
import os
import socket
import subprocess
import sys

import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    units, ms = bench.aggregate_over_ranks(100.0 * (rank + 1), 10.0 + 5.0 * rank, dist)
    dist.barrier()
    q.put((rank, units, ms))
    dist.destroy_process_group()


def test_aggregate_over_ranks_world2_gloo():
    """Replicas: units add up over ranks, time is the max over ranks."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got == [(0, 300.0, 15.0), (1, 300.0, 15.0)]


def test_aggregate_single_process_is_identity():
    import bench
    assert bench.aggregate_over_ranks(7.0, 3.0, None) == (7.0, 3.0)


def test_reference_arm_json_and_rank_gating():
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2", "--warmup", "1",
           "--ref-sample-elems", "16384", "--gpus", "2"]
    env = dict(os.environ, RANK="0", WORLD_SIZE="2")
    out = subprocess.run(cmd, capture_output=True, text=True, env=env, check=True, timeout=300).stdout.strip()
    line = json.loads(out.splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "grad-elements/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0,
                           "d2h_bytes_per_step": 0}
    assert line["steps"] == 2 and line["higher_is_better"] is True and line["n_gpus"] == 2
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""     # other ranks exit 0 without work


def test_bytes_model_matches_survey_table():
    from paper_1702_05800_b200 import synth
    assert synth.TINY.bytes_per_element == 32
    assert synth.INCEPTION_SGD.bytes_per_element == 216
    assert synth.PAPER_RMSPROP.bytes_per_element == 432
    assert synth.MIXED_PRECISION.bytes_per_element == 224
    assert synth.PAPER_RMSPROP.bytes_per_step == 10_871_635_968
    sweep = synth.sweep_configs()
    assert len(sweep) == 5 * 2 * 4 and max(c.footprint_bytes for c in sweep) < synth.HBM_LIMIT_BYTES
    for cfg in list(synth.CONFIGS.values()) + sweep[:4]:
        off = synth.shard_offsets(cfg)
        assert off[0] == 0 and off[-1] == cfg.P and len(off) == cfg.M + 1


def test_gpus_flag_without_torchrun_exits_instead_of_measuring_one_gpu():
    """`--gpus N` names the replica count, torchrun makes the replicas: a bare `python bench.py --gpus 8` must not print a
    one-GPU number labelled n_gpus = 1."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "8", "--steps", "2"], capture_output=True,
                       text=True, env=env, timeout=300)
    assert r.returncode == 2 and r.stdout.strip() == "" and "torch.distributed.run" in r.stderr
