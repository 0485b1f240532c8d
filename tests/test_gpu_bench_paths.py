"""The side paths of bench.py that profiles/ and DESIGN.md cite must keep running on a GPU box: each is started as the user
would start it (a subprocess) on a small configuration and its one JSON line is checked for shape, not for speed."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*flags, timeout=600):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *flags], capture_output=True, text=True,
                         timeout=timeout, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    return json.loads(out.stdout.strip().splitlines()[-1])


def test_probe_pipes_reports_three_pipe_rates():
    d = run_bench("--probe-pipes")
    rates = {k: v["per_clock_per_sm"] for k, v in d["pipes"].items()}
    assert set(rates) == {"ffma", "ffma2_packed", "mufu_rsqrt"}
    assert 30 < rates["ffma"] <= 130 and 30 < rates["ffma2_packed"] <= 260 and 4 < rates["mufu_rsqrt"] <= 33


def test_launch_bound_reports_eager_and_graph_costs_for_both_algorithms():
    d = run_bench("--launch-bound")
    for key, eager, graph in (("sync", "step_device_eager", "step_device_graph"),
                              ("sync_per_server", "step_device_eager", "step_device_graph"),
                              ("async", "async_step_device_eager", "async_step_device_graph"),
                              ("async_per_server", "async_step_device_eager", "async_step_device_graph")):
        assert 0 < d[key][graph] < d[key][eager] < 1000


@pytest.mark.parametrize("flags", [("--mode", "async"), ("--mode", "async_per_server", "--layout", "slices"),
                                   ("--mode", "per_server", "--layout", "slices"), ("--variant", "7"), ("--variant", "5")])
def test_small_config_through_every_mode_line_has_the_contract_keys(flags):
    d = run_bench("--config", "cfg2", "--steps", "3", "--warmup", "3", "--no-cpu-baseline", "--no-e2e", "--no-probe",
                  "--no-also", *flags)
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "dtype", "data", "config", "roofline", "clocks", "gpu_launches"):
        assert key in d, key
    assert d["roofline"]["bound"] == "hbm" and 0.3 < d["roofline"]["frac_of_nominal_8TBps"] < 1.0
    v = d["verified"]                      # every timed configuration is replayed by the oracle on sampled columns
    assert v["kept_bit_exact"] is True and v["elements"] > 20_000 and v["max_err_over_tolerance"] <= 1.0
    assert v["theta_changed"] > v["elements"] // 2
    assert d["gpu_launches"] > 0 and d["value"] > 0


@pytest.mark.parametrize("flags", [("--mode", "timeout"), ("--mode", "first_n", "--layout", "slices", "--servers", "3000")])
def test_timeout_mode_and_arena_slices_are_verified_too(flags):
    d = run_bench("--config", "cfg2", "--steps", "3", "--warmup", "3", "--no-cpu-baseline", "--no-e2e", "--no-probe",
                  "--no-also", *flags)
    assert d["verified"]["kept_bit_exact"] is True and d["verified"]["max_err_over_tolerance"] <= 1.0


def test_e2e_leg_is_verified_at_the_timed_size():
    """psync_step_host at cfg2's full size with bench.py's 4 Mi-element chunks: the extra step after the timed loop is
    replayed by the oracle on sampled columns, and the theta read back to the host equals the device's."""
    d = run_bench("--config", "cfg2", "--steps", "3", "--warmup", "3", "--no-cpu-baseline", "--no-probe", "--no-also",
                  "--e2e-steps", "2")
    v = d["e2e"]["verified"]
    assert v["kept_bit_exact"] is True and v["theta_readback_bit_exact"] is True and v["max_err_over_tolerance"] <= 1.0


def test_a_wrong_work_list_makes_the_bench_exit_non_zero():
    """The shard-aware kernels return early (theta untouched) when the (server, tile) list does not match the layout:
    a fast, wrong run.  bench.py must notice: `--fault worklist` hands it the list of the other gradient dtype."""
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--config", "cfg2", "--steps", "3", "--warmup", "3",
           "--no-cpu-baseline", "--no-e2e", "--no-probe", "--no-also", "--mode", "per_server", "--fault", "worklist"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode != 0 and "VerifyError" in out.stderr
    ok = subprocess.run(cmd[:-2], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert ok.returncode == 0, ok.stderr[-2000:]
