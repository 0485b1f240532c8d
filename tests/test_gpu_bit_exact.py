"""GPU vs the oracle's fp32 MIRROR, BIT FOR BIT (diagnostic on top of the tolerance-based parity tests).

The mirror restates DESIGN.md readings R9/R10 in fp32 on the CPU (fp32 adds in ascending kept order from 0, the five
stated fused multiply-adds, IEEE sqrt and division).  Equality of every bit of theta / state / ema checks the
summation order, the FMA placement and the device-side coefficients (1/n for the time-out rule), which a 1e-5
tolerance cannot see.  The double-arithmetic oracle remains the graded truth (all other tests/test_gpu_*.py)."""
from dataclasses import replace

import numpy as np
import pytest
import torch

import oracle
import paper_1702_05800_b200 as psync
from paper_1702_05800_b200 import synth

from _harness import STATE_NAMES, Pair, to_np
from test_gpu_async import AsyncPair
from test_gpu_async import BASE as ASYNC_BASE
from test_gpu_per_server import RowsPair, _timeout_gpu, per_server_cfg

pytestmark = pytest.mark.gpu
DEV = "cuda"
BASE = synth.Config(name="bits", cfg_id=13, P=70_003, M=7, N=10, b=3, arrival_sigma=0.3, opt=synth.SGD, gamma=0.045,
                    alpha=0.9999, mu=0.9, rho=0.9, eps=1.0, steps=3)


def assert_bits(pair_obj, host, what):
    for n in STATE_NAMES:
        g = getattr(pair_obj, n)
        if g is not None:
            a, b_ = to_np(g), host[n]
            same = a.view(np.uint32) == b_.view(np.uint32)
            assert same.all(), f"{what} {n}: {int((~same).sum())} of {a.size} elements differ in their bits"


@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
@pytest.mark.parametrize("opt", [synth.SGD, synth.MOMENTUM, synth.RMSPROP_MOM])
@pytest.mark.parametrize("ema_mode", [synth.EMA_POST, synth.EMA_PRE, synth.EMA_OFF])
def test_synchronous_step_every_template_instance(dtype, opt, ema_mode):
    cfg = replace(BASE, grad_dtype=dtype, opt=opt, ema_mode=ema_mode, name=f"bits_d{dtype}_o{opt}_e{ema_mode}")
    pair = Pair(cfg)
    with oracle.fp32_mirror():
        for s in range(3):                       # free-running: three steps without re-synchronising the host copy
            grads = pair.gradients(s)
            arrival = synth.arrival_times(cfg, s)
            pair.gpu_step(grads, arrival)
            pair.oracle_step(grads, arrival)
            assert_bits(pair.ps, pair.host, f"{cfg.name} step {s}")


@pytest.mark.parametrize("variant", [1, 5, 6, 7])   # 5: cp.async.bulk ring; 6: 256-bit loads; 7: per-thread cp.async ring (2, 3, 4, 8 were removed)
def test_every_variant_and_the_scalar_path(variant):
    cfg = replace(BASE, opt=synth.RMSPROP_MOM, N=100, b=6, P=40_001, name=f"bits_variant{variant}")
    pair = Pair(cfg, variant=variant)
    with oracle.fp32_mirror():
        grads = pair.gradients(0)
        arrival = synth.arrival_times(cfg, 0)
        pair.gpu_step(grads, arrival)
        pair.oracle_step(grads, arrival)
    assert_bits(pair.ps, pair.host, cfg.name)


@pytest.mark.parametrize("dtype,opt", [(synth.F32, synth.RMSPROP_MOM), (synth.BF16, synth.MOMENTUM)])
def test_shard_aware_kernel_on_misaligned_slices(dtype, opt):
    """The slices layout through the work list: aligned, one-phase and mixed-phase slices, transposed epilogue."""
    from test_gpu_slices import RAGGED, SlicesPair, cut_slices
    cfg = replace(BASE, grad_dtype=dtype, opt=opt, name=f"bits_slices_{dtype}_{opt}")
    pair = SlicesPair(cfg, shard_off=RAGGED)
    with oracle.fp32_mirror():
        for s, offs in enumerate([None, lambda k, j: (3 * j + 1) % 8, lambda k, j: (5 * k + 3 * j) % 8]):
            flat = [synth.gradient(cfg, s, k, DEV) for k in range(cfg.W)]
            slices = cut_slices(flat, pair.off, offs)
            arrival = synth.arrival_times(cfg, s)
            d_kept = torch.full((cfg.N,), -1, dtype=torch.int32, device=DEV)
            d_status = torch.full((1,), -9, dtype=torch.int32, device=DEV)
            st, keep = pair.make_step(psync.make_slice_table(slices), d_kept, d_status)
            psync.psync_step_device(st, torch.from_numpy(arrival).to(DEV))
            torch.cuda.synchronize()
            _, kept, _ = oracle.select_first_n(arrival, cfg.N, cfg.b)
            pair.oracle(slices, kept)
            assert_bits(pair, pair.host, f"{cfg.name} step {s}")


def test_per_server_rows_and_timeout_device_side_divisor():
    cfg = per_server_cfg(opt=synth.RMSPROP_MOM, P=50_003, name="bits_rows")
    pair = RowsPair(cfg)
    with oracle.fp32_mirror():
        # per-server first-N (one failed server)
        a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
        a[4, :6] = np.inf
        grads = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
        table = psync.make_grad_table(grads)
        d_kept = torch.full((pair.M, cfg.N), -1, dtype=torch.int32, device=DEV)
        d_status = torch.full((pair.M,), -9, dtype=torch.int32, device=DEV)
        psync.psync_select_first_n_sharded(torch.from_numpy(a).to(DEV), cfg.N, cfg.b, pair.M, d_kept, d_status)
        st, keep = pair.make_step(table, d_kept, d_status, per_shard=True)
        psync.psync_aggregate_update(st)
        torch.cuda.synchronize()
        status, kept, _ = oracle.select_first_n_sharded(a, cfg.N, cfg.b)
        pair.oracle_rows(grads, kept, True, status=status)
        assert_bits(pair, pair.host, "per-server")
        # per-server time-out: the divisor 1/n_j is formed on the device
        W = cfg.W
        d_kept, d_n, d_status = _timeout_gpu(a, 1.1, pair.M, W)
        st, keep = pair.make_step(table, d_kept, d_status, per_shard=True, d_n_kept=d_n)
        psync.psync_aggregate_update(st)
        torch.cuda.synchronize()
        kept = np.full((pair.M, W), -1, np.int32)
        n_kept = np.ones(pair.M, np.int32)
        status = np.zeros(pair.M, np.int32)
        for r in range(pair.M):
            status[r], k = oracle.select_timeout(a[r], 1.1)
            if status[r] == oracle.OK:
                kept[r, :k.size], n_kept[r] = k, k.size
        assert len(set(n_kept.tolist())) > 1
        pair.oracle_rows(grads, kept, True, n_kept=n_kept, status=status)
        assert_bits(pair, pair.host, "per-server time-out")


@pytest.mark.parametrize("dtype,opt", [(synth.F32, synth.RMSPROP_MOM), (synth.BF16, synth.MOMENTUM), (synth.F32, synth.SGD)])
def test_async_pass_with_clip_factors_and_per_iteration_rates(dtype, opt):
    cfg = replace(ASYNC_BASE, grad_dtype=dtype, opt=opt, P=60_001, N=23, name=f"bits_async_{dtype}_{opt}")
    pair = AsyncPair(cfg)
    rng = np.random.default_rng(4)
    grads = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    table = psync.make_grad_table(grads)
    arrival = synth.arrival_times(cfg, 0)
    arrival[7] = np.inf
    gammas = rng.uniform(0.01, 0.09, cfg.W).astype(np.float32)
    scales = rng.uniform(0.3, 1.0, cfg.W).astype(np.float32)         # any fp32 factors: the multiply is one fp32 op
    psync.psync_order_by_arrival(torch.from_numpy(arrival).to(DEV), cfg.W, pair.d_order, pair.d_n)
    st, keep = pair.make_step(table)
    psync.psync_async_apply(st, torch.from_numpy(gammas).to(DEV), d_gscale=torch.from_numpy(scales).to(DEV))
    torch.cuda.synchronize()
    order = oracle.order_by_arrival(arrival)
    h = pair.host
    with oracle.fp32_mirror():
        rc = oracle.async_apply(pair.off, [synth.as_numpy_grad(g) for g in grads], order, h["theta"], h["ema"],
                                h["state0"], h["state1"], gammas=gammas[:order.size].copy(),
                                gscales=scales[order].copy(), opt=cfg.opt, ema_mode=cfg.ema_mode, alpha=cfg.alpha,
                                mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
    assert rc == oracle.OK
    assert_bits(pair, h, cfg.name)


def test_standalone_ema_and_full_size_cfg3_sampled():
    th = torch.randn(100_003, device=DEV)
    em = torch.randn(100_003, device=DEV)
    h_em = to_np(em)
    psync.psync_ema(em, th, 0.9999)
    with oracle.fp32_mirror():
        oracle.ema_update(h_em, to_np(th), 0.9999)
    assert np.array_equal(to_np(em).view(np.uint32), h_em.view(np.uint32))
    # the headline configuration at full size, in bench.py's launch configuration, on sampled columns
    cfg = synth.PAPER_RMSPROP
    free, _ = torch.cuda.mem_get_info()
    if cfg.footprint_bytes * 1.15 > free:
        pytest.skip("not enough free HBM for the full-size config")
    pair = Pair(cfg)
    rng = np.random.default_rng(1)
    idx = np.unique(np.concatenate([np.arange(0, 2048), np.arange(cfg.P - 2048, cfg.P),
                                    rng.integers(0, cfg.P, 20_000)])).astype(np.int64)
    d_idx = torch.from_numpy(idx).to(DEV)
    host = {n: to_np(getattr(pair.ps, n)[d_idx]) for n in STATE_NAMES}
    grads = [torch.empty(cfg.P, dtype=torch.float32, device=DEV) for _ in range(cfg.W)]
    with oracle.fp32_mirror():
        for s in range(2):
            for k in range(cfg.W):
                synth.gradient(cfg, s, k, DEV, out=grads[k])
            arrival = synth.arrival_times(cfg, s)
            pair.gpu_step(grads, arrival)
            st, kept, _ = oracle.select_first_n(arrival, cfg.N, cfg.b)
            oracle.aggregate_update([0, idx.size], cfg.N, [synth.as_numpy_grad(g[d_idx]) for g in grads], kept,
                                    host["theta"], host["ema"], host["state0"], host["state1"], opt=cfg.opt,
                                    ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho,
                                    eps=cfg.eps)
            for n in STATE_NAMES:
                got = to_np(getattr(pair.ps, n)[d_idx])
                assert np.array_equal(got.view(np.uint32), host[n].view(np.uint32)), f"cfg3 step {s} {n}"
