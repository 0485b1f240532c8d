"""GPU parity on the BASELINE.json configs: cfg1 in full; cfg2-4 at a reduced P the oracle finishes
in seconds (several tiles + ragged tail, same N/b/M/optimizer/hyper-parameters) element by element;
and at FULL size, in the launch configuration bench.py times, on sampled outputs the oracle
computes one by one.  Also the host-buffer entry point psync_step_host."""
from dataclasses import replace

import numpy as np
import pytest
import torch

import oracle
import paper_1702_05800_b200 as psync
from paper_1702_05800_b200 import synth

from _harness import ATOL_STEP, RTOL_BF16, RTOL_FREE_100, RTOL_STEP, Pair, assert_close, to_np

pytestmark = pytest.mark.gpu
DEV = "cuda"


def test_cfg1_tiny_all_10_steps_lockstep_and_free_run():
    Pair(synth.TINY).run(synth.TINY.steps, lockstep=True)
    Pair(synth.TINY).run(synth.TINY.steps, lockstep=False, rtol=RTOL_FREE_100)


@pytest.mark.parametrize("cfg", [synth.INCEPTION_SGD, synth.PAPER_RMSPROP, synth.MIXED_PRECISION],
                         ids=lambda c: c.name)
def test_cfg2_3_4_reduced_P_lockstep(cfg):
    small = synth.scaled(cfg, 786_432 + 13)      # 768 Ki + ragged tail: hundreds of tiles, M ragged shards
    rtol = RTOL_BF16 if cfg.grad_dtype == synth.BF16 else RTOL_STEP
    Pair(small).run(3, lockstep=True, rtol=rtol, atol=ATOL_STEP)
    if cfg.grad_dtype == synth.BF16:              # widening is exact, so the tight bound holds too
        Pair(small).run(1, lockstep=True, rtol=RTOL_STEP, atol=ATOL_STEP)


@pytest.mark.parametrize("cfg", [synth.INCEPTION_SGD, synth.PAPER_RMSPROP, synth.MIXED_PRECISION],
                         ids=lambda c: c.name)
def test_free_run_100_steps(cfg):
    """north_star: 1e-4 relative after 100 steps of free running (2e-3 with bf16 gradients)."""
    small = synth.scaled(cfg, 16_384 + 5)
    rtol = RTOL_BF16 if cfg.grad_dtype == synth.BF16 else RTOL_FREE_100
    Pair(small).run(100, lockstep=False, rtol=rtol, atol=ATOL_STEP, check_every=25)


def test_cfg5_sweep_points_reduced():
    for cfg in synth.sweep_configs():
        if cfg.P != synth.SWEEP_P[0]:
            continue
        Pair(synth.scaled(cfg, 262_144 + 3)).run(2, lockstep=True)


# ------------------------------------------------------------------ full size, bench launch config
def _full_size_sampled(cfg, steps=2, n_sample=40_000):
    """Run the real config on the GPU; check sampled elements against the oracle run on the gathered
    columns (gathering by index moves data, it computes nothing)."""
    free, _ = torch.cuda.mem_get_info()
    if cfg.footprint_bytes * 1.15 > free:
        pytest.skip("not enough free HBM for the full-size config")
    pair = Pair(cfg)          # default variant / grid = what bench.py launches
    rng = np.random.default_rng(cfg.cfg_id)
    tile = 8192
    idx = np.unique(np.concatenate([
        np.arange(0, 2 * tile), np.arange(cfg.P - 2 * tile, cfg.P),           # first and last tiles
        pair.shard_off[1:-1], np.maximum(pair.shard_off[1:-1] - 1, 0),                        # every shard cut
        rng.integers(0, cfg.P, n_sample)])).astype(np.int64)
    d_idx = torch.from_numpy(idx).to(DEV)
    off_s = np.array([0, idx.size], dtype=np.int64)
    host = {n: (None if getattr(pair.ps, n) is None else to_np(getattr(pair.ps, n)[d_idx]))
            for n in ("theta", "ema", "state0", "state1")}
    grads = [torch.empty(cfg.P, dtype=torch.float32 if cfg.grad_dtype == synth.F32 else torch.bfloat16, device=DEV)
             for _ in range(cfg.W)]
    for s in range(steps):
        for k in range(cfg.W):
            synth.gradient(cfg, s, k, DEV, out=grads[k])
        arrival = synth.arrival_times(cfg, s)
        st, kept, tn = pair.gpu_step(grads, arrival)
        st_o, kept_o, tn_o = oracle.select_first_n(arrival, cfg.N, cfg.b)
        assert st == st_o == 0 and np.array_equal(kept, kept_o) and tn == tn_o
        g_s = [synth.as_numpy_grad(g[d_idx]) for g in grads]
        rc = oracle.aggregate_update(off_s, cfg.N, g_s, kept_o, host["theta"], host["ema"], host["state0"],
                                     host["state1"], opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma,
                                     alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
        assert rc == oracle.OK
        rtol = RTOL_BF16 if cfg.grad_dtype == synth.BF16 else RTOL_STEP
        for n in ("theta", "ema", "state0", "state1"):
            if host[n] is not None:
                got = to_np(getattr(pair.ps, n)[d_idx])
                assert_close(got, host[n], rtol, ATOL_STEP, f"{cfg.name} step {s} {n} (sampled)")
                host[n] = got                                               # lock-step
        # property that holds at any size: nothing outside tolerance can hide as NaN/Inf
        assert bool(torch.isfinite(pair.ps.theta).all())
    geo = pair.ps.geometry(cfg.gamma)
    assert geo["grid"] == -(-cfg.P // geo["tile_elems"])          # one tile per CTA, the bench's launch


def _full_size_every_element(cfg, steps=2):
    """The real config in bench.py's launch configuration, ALL P elements of theta / state / ema compared after every
    step (lock-step) with the oracle's streamed form: oracle.accumulate over the kept workers' buffers in ascending
    order (one buffer D2H at a time), then oracle.apply_sum -- bit-identical to the whole-step oracle (pinned in
    tests/test_oracle_update.py::test_shard_layout_invariance_and_streamed_form)."""
    free, _ = torch.cuda.mem_get_info()
    if cfg.footprint_bytes * 1.15 > free:
        pytest.skip("not enough free HBM for the full-size config")
    pair = Pair(cfg)
    grads = [torch.empty(cfg.P, dtype=torch.float32 if cfg.grad_dtype == synth.F32 else torch.bfloat16, device=DEV)
             for _ in range(cfg.W)]
    S = np.zeros(cfg.P, np.float64)
    rtol = RTOL_BF16 if cfg.grad_dtype == synth.BF16 else RTOL_STEP
    for s in range(steps):
        h = pair.host                                                # lock-step: re-synchronised after every step
        for k in range(cfg.W):
            synth.gradient(cfg, s, k, DEV, out=grads[k])
        arrival = synth.arrival_times(cfg, s)
        st, kept, tn = pair.gpu_step(grads, arrival)
        st_o, kept_o, tn_o = oracle.select_first_n(arrival, cfg.N, cfg.b)
        assert st == st_o == 0 and np.array_equal(kept, kept_o) and tn == tn_o
        S[:] = 0.0
        for k in kept_o:
            assert oracle.accumulate(S, synth.as_numpy_grad(grads[k])) == oracle.OK
        assert oracle.apply_sum(pair.shard_off, cfg.N, S, h["theta"], h["ema"], h["state0"], h["state1"], opt=cfg.opt,
                                ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho,
                                eps=cfg.eps) == oracle.OK
        pair.compare(rtol, ATOL_STEP, f"{cfg.name} full size, every element, step {s}")
        pair.sync_host_from_gpu()


def test_full_size_cfg3_paper_rmsprop_every_element():
    _full_size_every_element(synth.PAPER_RMSPROP)


def test_full_size_cfg2_inception_sgd_every_element():
    _full_size_every_element(synth.INCEPTION_SGD)


def test_full_size_cfg4_mixed_precision_every_element():
    _full_size_every_element(synth.MIXED_PRECISION, steps=1)


def test_full_size_cfg3_paper_rmsprop_sampled():
    _full_size_sampled(synth.PAPER_RMSPROP)


def test_full_size_cfg2_inception_sgd_sampled():
    _full_size_sampled(synth.INCEPTION_SGD)


def test_full_size_cfg4_mixed_precision_sampled():
    _full_size_sampled(synth.MIXED_PRECISION, steps=1)


# ------------------------------------------------------------------ host-buffer entry point
@pytest.mark.parametrize("cfg,chunk", [(synth.scaled(synth.PAPER_RMSPROP, 300_000 + 7), 65_536),
                                       (synth.scaled(synth.MIXED_PRECISION, 200_000 + 3), 0),
                                       (synth.TINY, 1024)], ids=["rmsprop_chunked", "bf16_default_chunk", "tiny"])
def test_step_host_matches_oracle(cfg, chunk):
    pair = Pair(cfg)
    nbytes = psync.psync_step_host_workspace_bytes(cfg.N, cfg.W, cfg.grad_dtype, chunk)
    assert nbytes > 0
    d_work = torch.empty(nbytes, dtype=torch.uint8, device=DEV)
    h_theta = torch.empty(cfg.P, dtype=torch.float32).pin_memory()
    h_kept = np.full(cfg.N, -1, dtype=np.int32)
    for s in range(2):
        h_grads = [synth.gradient(cfg, s, k, "cpu").pin_memory() for k in range(cfg.W)]
        arrival = synth.arrival_times(cfg, s)
        step, keep = psync.make_step(pair.shard_off, cfg.N, cfg.W, cfg.grad_dtype, pair.ps.theta, pair.ps.ema,
                                     pair.ps.state0, pair.ps.state1, opt=cfg.opt, ema_mode=cfg.ema_mode,
                                     gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
        st, t_nth = psync.psync_step_host(step, arrival, h_grads, d_work, h_theta_out=h_theta, h_kept=h_kept,
                                          chunk_elems=chunk)
        st_o, kept_o, tn_o = pair.oracle_step(h_grads, arrival)
        assert st == st_o == 0 and np.array_equal(h_kept, kept_o) and t_nth == tn_o
        rtol = RTOL_BF16 if cfg.grad_dtype == synth.BF16 else RTOL_STEP
        pair.compare(rtol, ATOL_STEP, f"host step {s}")
        assert np.array_equal(h_theta.numpy(), to_np(pair.ps.theta))       # theta(t+1) came back to the host
        pair.sync_host_from_gpu()


def test_step_host_too_few_and_bad_workspace():
    cfg = synth.scaled(synth.TINY, 2048)
    pair = Pair(cfg)
    before = to_np(pair.ps.theta)
    nbytes = psync.psync_step_host_workspace_bytes(cfg.N, cfg.W, cfg.grad_dtype, 0)
    d_work = torch.empty(nbytes, dtype=torch.uint8, device=DEV)
    h_grads = [synth.gradient(cfg, 0, k, "cpu") for k in range(cfg.W)]       # pageable memory is allowed
    step, keep = psync.make_step(pair.shard_off, cfg.N, cfg.W, cfg.grad_dtype, pair.ps.theta, pair.ps.ema,
                                 opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha)
    arrival = np.array([0.1, np.nan, np.inf, 0.2, 0.3], dtype=np.float32)
    st, _ = psync.psync_step_host(step, arrival, h_grads, d_work)
    assert st == psync.PSYNC_ETOOFEW and np.array_equal(before, to_np(pair.ps.theta))
    st, _ = psync.psync_step_host(step, synth.arrival_times(cfg, 0), h_grads, d_work[: nbytes // 2], check=False)
    assert st == psync.PSYNC_EINVAL
    assert psync.psync_step_host_workspace_bytes(cfg.N, cfg.W, cfg.grad_dtype, 100) == 0   # not a multiple of 64
    st, _ = psync.psync_step_host(step, synth.arrival_times(cfg, 0), h_grads, d_work)
    assert st == psync.PSYNC_OK
    pair.oracle_step(h_grads, synth.arrival_times(cfg, 0))
    pair.compare(RTOL_STEP, ATOL_STEP, "host pageable")


# ------------------------------------------------------------------ back-to-back launches (PDL ordering)
@pytest.mark.parametrize("P", [4096, 300_000 + 5, 6_000_000 + 3])
def test_back_to_back_steps_without_host_sync(P):
    """Both kernels use programmatic dependent launch: the next step's selection may become resident
    while this step's fused kernel drains.  Enqueue many steps with NO synchronisation in between
    (shared kept[]/status buffers, fresh arrival times, rotating gradient sets) and compare the final
    state with the oracle's free run: any early overwrite of kept[] or early read of theta would show."""
    cfg = replace(synth.scaled(synth.PAPER_RMSPROP, P), N=12, b=4, M=5, name=f"b2b_{P}")
    T, n_sets = 24, 3
    pair = Pair(cfg)
    sets = [[synth.gradient(cfg, r, k, DEV) for k in range(cfg.W)] for r in range(n_sets)]
    tables = [psync.make_grad_table(s) for s in sets]
    arrivals_h = [synth.arrival_times(cfg, s) for s in range(T)]
    arrivals = torch.from_numpy(np.stack(arrivals_h)).to(DEV)
    ps = pair.ps
    steps = [psync.make_step(pair.shard_off, cfg.N, cfg.W, tb.grad_dtype, ps.theta, ps.ema, ps.state0, ps.state1,
                             opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu,
                             rho=cfg.rho, eps=cfg.eps, d_grads=tb.d_ptrs, d_kept=ps.d_kept, d_status=ps.d_status)
             for tb in tables]
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    for s in range(T):
        psync.psync_select_first_n(arrivals[s], cfg.N, cfg.b, ps.d_kept, ps.d_status, ps.d_t_nth, None, 0, stream)
        psync.psync_aggregate_update(steps[s % n_sets][0], stream)
    stream.synchronize()
    for s in range(T):
        st, _, _ = pair.oracle_step(sets[s % n_sets], arrivals_h[s])
        assert st == 0
    pair.compare(RTOL_FREE_100, ATOL_STEP, "back-to-back free run")
    st, kept, tn = oracle.select_first_n(arrivals_h[T - 1], cfg.N, cfg.b)
    assert np.array_equal(ps.d_kept.cpu().numpy(), kept) and float(ps.d_t_nth.item()) == tn


# ------------------------------------------------------------------ one-call step and CUDA graph capture
def test_step_device_equals_the_two_calls_bitwise():
    cfg = synth.scaled(synth.PAPER_RMSPROP, 150_001)
    arrival = synth.arrival_times(cfg, 0)
    out = []
    for one_call in (True, False):
        pair = Pair(cfg)
        grads = pair.gradients(0)
        pair.ps.set_gradients(grads)
        d_arr = torch.from_numpy(arrival).to(DEV)
        if one_call:
            pair.ps.step(d_arr, cfg.gamma)
        else:
            psync.psync_select_first_n(d_arr, cfg.N, cfg.b, pair.ps.d_kept, pair.ps.d_status, pair.ps.d_t_nth)
            pair.ps.aggregate_only(cfg.gamma)
        torch.cuda.synchronize()
        out.append([to_np(getattr(pair.ps, n)) for n in ("theta", "ema", "state0", "state1", "d_kept", "d_t_nth")])
    for a, b_ in zip(*out):
        assert np.array_equal(a, b_)


@pytest.mark.parametrize("cfg", [synth.TINY, synth.scaled(synth.PAPER_RMSPROP, 40_003)])
def test_cuda_graph_capture_and_replay_matches_oracle(cfg):
    """The step is capturable (no synchronising call inside): capture 3 steps reading a fixed arrival buffer,
    replay twice with fresh arrival times, compare with the oracle after every replay."""
    pair = Pair(cfg)
    grads = pair.gradients(0)
    pair.ps.set_gradients(grads)
    steps_per_graph = 3
    d_arr = torch.zeros(steps_per_graph, cfg.W, dtype=torch.float32, device=DEV)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        d_arr.copy_(torch.from_numpy(np.stack([synth.arrival_times(cfg, 100 + i) for i in range(steps_per_graph)])))
        snapshot = {n: (None if getattr(pair.ps, n) is None else getattr(pair.ps, n).clone())
                    for n in ("theta", "ema", "state0", "state1")}
        pair.ps.step(d_arr[0], cfg.gamma, stream=side)                     # warm-up outside capture
        side.synchronize()
        for n, v in snapshot.items():                                      # undo the warm-up step
            if v is not None:
                getattr(pair.ps, n).copy_(v)
        with torch.cuda.graph(graph, stream=side):
            for i in range(steps_per_graph):
                pair.ps.step(d_arr[i], cfg.gamma, stream=side)
    torch.cuda.synchronize()
    s = 0
    for replay in range(2):
        arr = np.stack([synth.arrival_times(cfg, s + i) for i in range(steps_per_graph)])
        d_arr.copy_(torch.from_numpy(arr))
        graph.replay()
        torch.cuda.synchronize()
        for i in range(steps_per_graph):
            st, kept, _ = pair.oracle_step(grads, arr[i])
            assert st == 0
        assert np.array_equal(pair.ps.d_kept.cpu().numpy(), kept)
        pair.compare(RTOL_STEP * steps_per_graph, ATOL_STEP, f"graph replay {replay}")
        pair.sync_host_from_gpu()
        s += steps_per_graph


# ------------------------------------------------------------------ stale gradients across steps (Alg. 4 l.5-6)
def test_stale_gradients_of_dropped_workers_carry_into_the_next_step_and_are_dropped():
    """NEXT-2: the b workers dropped at step t-1 deliver that old gradient, tagged t-1, EARLY in step t (before
    anyone else).  Alg. 4 l.5-6 drops it by its tag; the server then keeps the first N of the
    remaining workers.  The stale buffers hold NaN, so any use of them would poison theta."""
    cfg = replace(synth.scaled(synth.PAPER_RMSPROP, 60_001), N=20, b=6, M=5, name="stale_carry")
    pair = Pair(cfg)
    stale = np.array([], dtype=np.int64)
    for t in range(5):
        grads = pair.gradients(t)
        arrival = synth.arrival_times(cfg, t)
        tags = np.full(cfg.W, t, dtype=np.int32)
        if stale.size:
            tags[stale] = t - 1
            arrival[stale] = np.float32(1e-3) * (1 + np.arange(stale.size, dtype=np.float32))   # first to arrive
            for k in stale:
                grads[k].fill_(float("nan"))
        st_g, kept_g, tn_g = pair.gpu_step(grads, arrival, tags=tags, t=t)
        st_o, kept_o, tn_o = pair.oracle_step(grads, arrival, tags=tags, t=t)
        assert st_g == st_o == 0 and np.array_equal(kept_g, kept_o) and tn_g == tn_o
        assert not set(kept_g.tolist()) & set(stale.tolist())
        assert tn_g > 0.1                                        # the server waited for fresh gradients
        pair.compare(RTOL_STEP, ATOL_STEP, f"stale carry step {t}")
        pair.sync_host_from_gpu()
        assert bool(torch.isfinite(pair.ps.theta).all())
        stale = np.setdiff1d(np.arange(cfg.W), kept_g)[:cfg.b]   # this step's dropped workers are next step's stale
    # more stale workers than backups: the server can never collect N fresh gradients
    tags = np.full(cfg.W, 9, dtype=np.int32)
    tags[:cfg.b + 1] = 8
    before = to_np(pair.ps.theta)
    st_g, _, _ = pair.gpu_step(pair.gradients(9), synth.arrival_times(cfg, 9), tags=tags, t=9)
    assert st_g == psync.PSYNC_ETOOFEW and np.array_equal(before, to_np(pair.ps.theta))


# ------------------------------------------------------------------ re-entrancy and 64-bit indexing
def test_two_servers_on_two_streams_are_independent():
    """The library keeps no state: two servers stepping concurrently on two streams give, bit for bit, what each
    gives alone."""
    cfg = synth.scaled(synth.PAPER_RMSPROP, 2_000_003)
    results = []
    for concurrent in (False, True):
        pairs = [Pair(cfg), Pair(replace(cfg, cfg_id=33))]
        grads = [p.gradients(0) for p in pairs]
        for p, g in zip(pairs, grads):
            p.ps.set_gradients(g)
        streams = [torch.cuda.Stream(), torch.cuda.Stream()] if concurrent else [torch.cuda.current_stream()] * 2
        torch.cuda.synchronize()
        for s in range(6):
            for p, st in zip(pairs, streams):
                d_arr = torch.from_numpy(synth.arrival_times(p.cfg, s)).to(DEV)
                st.wait_stream(torch.cuda.current_stream())
                p.ps.step(d_arr, cfg.gamma, stream=st)
                d_arr.record_stream(st)
        torch.cuda.synchronize()
        results.append([[to_np(getattr(p.ps, n)) for n in ("theta", "ema", "state0", "state1", "d_kept")]
                        for p in pairs])
    for alone, together in zip(results[0], results[1]):
        for a, b_ in zip(alone, together):
            assert np.array_equal(a, b_)


def test_more_than_2_to_31_parameters_sampled():
    """P = 2^31 + 2^20 + 5: element indices and byte offsets need 64 bits (the last tile starts beyond 8 GiB).
    SGD + EMA, N=2, b=1; sampled elements (first and last tiles, around 2^31, random) against the oracle."""
    P = (1 << 31) + (1 << 20) + 5
    cfg = replace(synth.INCEPTION_SGD, P=P, M=3, N=2, b=1, name="huge_P")
    free, _ = torch.cuda.mem_get_info()
    if cfg.footprint_bytes * 1.3 > free:
        pytest.skip("not enough free HBM for 2^31 parameters")
    pair = Pair(cfg)
    rng = np.random.default_rng(2)
    idx = np.unique(np.concatenate([np.arange(0, 2048), np.arange(P - 2048, P),
                                    np.arange((1 << 31) - 1500, (1 << 31) + 1500),
                                    pair.shard_off[1:-1], rng.integers(0, P, 20_000)])).astype(np.int64)
    d_idx = torch.from_numpy(idx).to(DEV)
    off_s = np.array([0, idx.size], dtype=np.int64)
    host = {n: to_np(getattr(pair.ps, n)[d_idx]) for n in ("theta", "ema")}
    grads = [torch.empty(P, dtype=torch.float32, device=DEV) for _ in range(cfg.W)]
    for k in range(cfg.W):
        synth.gradient(cfg, 0, k, DEV, out=grads[k])
    arrival = synth.arrival_times(cfg, 0)
    st, kept, _ = pair.gpu_step(grads, arrival)
    st_o, kept_o, _ = oracle.select_first_n(arrival, cfg.N, cfg.b)
    assert st == st_o == 0 and np.array_equal(kept, kept_o)
    rc = oracle.aggregate_update(off_s, cfg.N, [synth.as_numpy_grad(g[d_idx]) for g in grads], kept_o, host["theta"],
                                 host["ema"], opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha)
    assert rc == oracle.OK
    for n in ("theta", "ema"):
        assert_close(to_np(getattr(pair.ps, n)[d_idx]), host[n], RTOL_STEP, ATOL_STEP, f"huge P {n} (sampled)")
    geo = pair.ps.geometry(cfg.gamma)
    assert geo["grid"] == -(-P // geo["tile_elems"]) and geo["grid"] > (1 << 21)


def test_full_size_largest_sweep_point_sampled():
    """cfg5's largest point at full size: P = 256 Mi, N = 100, b = 10, M = 64 ragged (120.3 GB resident)."""
    cfg = [c for c in synth.sweep_configs() if c.P == synth.SWEEP_P[-1] and c.M == 64 and c.N == 100][0]
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if cfg.footprint_bytes * 1.1 > free:
        pytest.skip("not enough free HBM for the 120 GB sweep point")
    _full_size_sampled(cfg, steps=1, n_sample=20_000)
    torch.cuda.empty_cache()


def test_plain_c_client_of_the_abi(tmp_path):
    """A C program (gcc, no Python, no torch) includes include/psync.h, links libpsync.so and runs one hand-checkable
    step: the boundary really is a C ABI with plain pointers."""
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    exe = tmp_path / "abi_smoke"
    pkg = os.path.join(root, "paper_1702_05800_b200")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-O1", os.path.join(root, "tests", "c", "abi_smoke.c"),
                    "-I", os.path.join(root, "include"), "-I", os.path.join(cuda, "include"), "-L", pkg, "-lpsync",
                    "-L", os.path.join(cuda, "lib64"), "-lcudart", "-lm", f"-Wl,-rpath,{pkg}",
                    f"-Wl,-rpath,{os.path.join(cuda, 'lib64')}", "-o", str(exe)], check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True)
    assert out.returncode == 0, out.stderr
    assert "abi_smoke ok" in out.stdout
