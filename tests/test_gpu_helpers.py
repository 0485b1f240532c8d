"""GPU parity for the NEXT-4 helpers through the C ABI: learning-rate schedule, global-norm
clip factors and the clipped asynchronous update, against the CPU oracle."""
from dataclasses import replace

import numpy as np
import pytest
import torch

import oracle
import paper_1702_05800_b200 as psync
from paper_1702_05800_b200 import synth

from _harness import ATOL_STEP, STATE_NAMES, assert_close, to_np
from test_gpu_async import BASE, AsyncPair, rtol_async

pytestmark = pytest.mark.gpu
DEV = "cuda"


def ulp_diff(a, b):
    ia = np.asarray(a, np.float32).view(np.int32).astype(np.int64)
    ib = np.asarray(b, np.float32).view(np.int32).astype(np.int64)
    return np.abs(ia - ib)


@pytest.mark.parametrize("gamma0,beta,t0,K,s", [(4.5, 0.94, 0, 200, 100 / (2 * 40037.0)), (0.045, 0.94, 10**6, 1024, 1 / 80074.0),
                                                (0.1, 0.5, 3, 2, 1.0), (2.25, 0.94, 12345, 1, 50 / 80074.0), (1.0, 1.0, 0, 33, 9.0)])
def test_lr_schedule_matches_oracle(gamma0, beta, t0, K, s):
    d = torch.full((K + 2,), -1.0, dtype=torch.float32, device=DEV)
    psync.psync_lr_schedule(gamma0, beta, t0, K, s, d)
    want = oracle.lr_schedule(gamma0, beta, t0, K, s)
    got = d.cpu().numpy()
    assert ulp_diff(got[:K], want).max() <= 1          # double pow on both sides, one rounding to fp32
    assert (got[K:] == -1.0).all()
    assert psync.psync_lr_schedule(gamma0, beta, t0, 0, s, d) == psync.PSYNC_OK
    L = psync.binding.lib()
    assert L.psync_lr_schedule(0.1, 0.0, 0, 1, 1.0, d.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_lr_schedule(0.1, 0.5, -1, 1, 1.0, d.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_lr_schedule(0.1, 0.5, 0, 1, 1.0, None, None) == psync.PSYNC_EINVAL


def test_lr_schedule_counted_advances_by_the_largest_count_and_restarts():
    """psync_lr_schedule_counted: *d_t <- t_set or *d_t + max_r d_n_add[r], then the same bits as psync_lr_schedule."""
    gamma0, beta, s, K = 0.045, 0.94, 1.0 / 11.0, 37
    d_t = torch.tensor([100], dtype=torch.int64, device=DEV)
    d_n = torch.tensor([5, 31, 0, 17], dtype=torch.int32, device=DEV)
    d = torch.zeros(K, dtype=torch.float32, device=DEV)
    psync.psync_lr_schedule_counted(gamma0, beta, d_t, K, s, d, d_n_add=d_n)
    assert int(d_t.item()) == 131 and np.array_equal(d.cpu().numpy(), oracle.lr_schedule(gamma0, beta, 131, K, s))
    psync.psync_lr_schedule_counted(gamma0, beta, d_t, K, s, d, d_n_add=d_n[:1])
    assert int(d_t.item()) == 136 and np.array_equal(d.cpu().numpy(), oracle.lr_schedule(gamma0, beta, 136, K, s))
    psync.psync_lr_schedule_counted(gamma0, beta, d_t, K, s, d)                         # no counts: the counter stays
    assert int(d_t.item()) == 136
    psync.psync_lr_schedule_counted(gamma0, beta, d_t, K, s, d, d_n_add=d_n, t_set=7)   # restart: counts ignored
    assert int(d_t.item()) == 7 and np.array_equal(d.cpu().numpy(), oracle.lr_schedule(gamma0, beta, 7, K, s))
    big = torch.arange(5000, dtype=torch.int32, device=DEV) % 1000                      # more rows than threads
    psync.psync_lr_schedule_counted(gamma0, beta, d_t, 1, s, d, d_n_add=big)
    assert int(d_t.item()) == 7 + 999
    ref = torch.zeros(K, dtype=torch.float32, device=DEV)
    psync.psync_lr_schedule(gamma0, beta, 7 + 999, 1, s, ref)
    assert d[0].item() == ref[0].item()
    L = psync.binding.lib()
    assert L.psync_lr_schedule_counted(0.1, 0.5, None, -1, None, 0, 1, 1.0, d.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_lr_schedule_counted(0.1, 0.5, d_t.data_ptr(), -1, None, 0, 1025, 1.0, d.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_lr_schedule_counted(0.1, 0.0, d_t.data_ptr(), -1, None, 0, 1, 1.0, d.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_lr_schedule_counted(0.1, 0.5, d_t.data_ptr(), -1, d_n.data_ptr(), 0, 1, 1.0, d.data_ptr(), None) == psync.PSYNC_EINVAL


def _clip_gpu(grads, clip):
    table = psync.make_grad_table(grads)
    nbytes = psync.psync_clip_workspace_bytes(table.W, grads[0].numel(), table.grad_dtype)
    assert nbytes >= 8 * table.W
    d_work = torch.empty(nbytes // 8, dtype=torch.float64, device=DEV)
    d_scales = torch.full((table.W,), -1.0, dtype=torch.float32, device=DEV)
    psync.psync_clip_scales(table, clip, d_scales, d_work)
    torch.cuda.synchronize()
    return d_scales


@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
@pytest.mark.parametrize("P", [1, 7, 8, 9, 1000, 32_768, 32_769, 300_001])
def test_clip_scales_match_oracle(dtype, P):
    rng = np.random.default_rng(P + dtype)
    W = 6
    grads = []
    for k in range(W):
        g = torch.randn(P, device=DEV) * float(10.0 ** rng.integers(-4, 1))
        grads.append(g.to(torch.bfloat16) if dtype == synth.BF16 else g)
    clip = 0.05
    got = _clip_gpu(grads, clip).cpu().numpy()
    want = oracle.clip_scales([synth.as_numpy_grad(g) for g in grads], clip)
    assert np.abs(got - want).max() <= 1e-6 * np.abs(want).max() + 1e-12
    assert ((want == 1.0) == (got == 1.0)).all() or np.abs(got - want).max() < 2e-7


def test_clip_scales_3_4_5_and_determinism_and_unaligned():
    g = [torch.tensor([3.0, 4.0], device=DEV), torch.zeros(2, device=DEV), torch.tensor([-6.0, 8.0], device=DEV)]
    assert _clip_gpu(g, 2.5).cpu().tolist() == [0.5, 1.0, 0.25]
    big = [torch.randn(1_000_003, device=DEV) for _ in range(3)]
    a, b = _clip_gpu(big, 1.0).cpu().numpy(), _clip_gpu(big, 1.0).cpu().numpy()
    assert np.array_equal(a, b)                                              # no atomics: run-to-run identical
    buf = torch.randn(50_010, device=DEV)
    shifted = [buf[1:50_001], buf[2:50_002], buf[3:50_003]]                   # 4-, 8-, 12-byte offsets
    got = _clip_gpu([s for s in shifted], 1.0).cpu().numpy()
    want = oracle.clip_scales([s.cpu().numpy().copy() for s in shifted], 1.0)
    assert np.abs(got - want).max() <= 1e-6


def test_clip_invalid_arguments():
    L = psync.binding.lib()
    assert L.psync_clip_scales(None, 1, 4, 0, 1.0, None, None, 0, None) == psync.PSYNC_EINVAL
    assert L.psync_clip_scales(8, 0, 4, 0, 1.0, 8, 8, 64, None) == psync.PSYNC_EINVAL
    assert L.psync_clip_scales(8, 1, 4, 0, 0.0, 8, 8, 64, None) == psync.PSYNC_EINVAL
    assert L.psync_clip_scales(8, 1, 4, 2, 1.0, 8, 8, 64, None) == psync.PSYNC_EINVAL
    assert L.psync_clip_scales(8, 1, 4, 0, 1.0, 8, 8, 4, None) == psync.PSYNC_EINVAL      # workspace too small
    assert psync.psync_clip_workspace_bytes(0, 4, 0) == 0


@pytest.mark.parametrize("dtype,opt", [(synth.F32, synth.RMSPROP_MOM), (synth.BF16, synth.MOMENTUM), (synth.F32, synth.SGD)])
def test_async_with_clipping_and_schedule_matches_oracle(dtype, opt):
    """The paper's Async-Opt recipe end to end (A.3): arrival order, global-norm clipping of every gradient, a
    decaying learning rate per iteration, RMSProp / momentum / SGD, EMA."""
    cfg = replace(BASE, grad_dtype=dtype, opt=opt, P=90_001, grad_dist=("normal", 1e-2), name=f"async_clip_{dtype}_{opt}")
    pair = AsyncPair(cfg)
    clip = 2.0                                          # ||G|| ~ 1e-2 * sqrt(90001) = 3: every gradient is clipped
    for s in range(2):
        grads = [synth.gradient(cfg, s, k, DEV) for k in range(cfg.W)]
        if s == 1:
            grads[5] = grads[5] * 0.1                   # one gradient inside the bound: factor exactly 1
        table = psync.make_grad_table(grads)
        arrival = synth.arrival_times(cfg, s)
        psync.psync_order_by_arrival(torch.from_numpy(arrival).to(DEV), cfg.W, pair.d_order, pair.d_n)
        d_work = torch.empty(psync.psync_clip_workspace_bytes(cfg.W, cfg.P, table.grad_dtype) // 8, dtype=torch.float64,
                             device=DEV)
        d_scales = torch.empty(cfg.W, dtype=torch.float32, device=DEV)
        psync.psync_clip_scales(table, clip, d_scales, d_work)
        d_gamma = torch.empty(cfg.W, dtype=torch.float32, device=DEV)
        psync.psync_lr_schedule(0.045, 0.94, 1000 * s, cfg.W, 0.01, d_gamma)
        st, keep = pair.make_step(table)
        psync.psync_async_apply(st, d_gamma, d_gscale=d_scales)
        torch.cuda.synchronize()
        # oracle, fed the GPU's clip factors and rates (each checked against its own oracle first): lock-step
        order = oracle.order_by_arrival(arrival)
        np_grads = [synth.as_numpy_grad(g) for g in grads]
        sc_o = oracle.clip_scales(np_grads, clip)
        sc_g = d_scales.cpu().numpy()
        assert np.abs(sc_g - sc_o).max() <= 1e-6 and (s == 0 or sc_g[5] == 1.0) and (np.delete(sc_g, 5) < 1.0).all()
        gm_o = oracle.lr_schedule(0.045, 0.94, 1000 * s, cfg.W, 0.01)
        gm_g = d_gamma.cpu().numpy()
        assert ulp_diff(gm_g, gm_o).max() <= 1
        h = pair.host
        rc = oracle.async_apply(pair.off, np_grads, order, h["theta"], h["ema"], h["state0"], h["state1"],
                                gammas=gm_g[:order.size].copy(), gscales=sc_g[order].copy(), opt=cfg.opt,
                                ema_mode=cfg.ema_mode, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
        assert rc == oracle.OK
        for n in STATE_NAMES:
            g = getattr(pair, n)
            if g is not None:
                assert_close(to_np(g), h[n], rtol_async(order.size), ATOL_STEP, f"{cfg.name} step {s} {n}")
                h[n] = to_np(g)


def test_unit_scale_is_bit_identical_to_no_scale():
    cfg = replace(BASE, P=50_003, opt=synth.RMSPROP_MOM, name="async_unit_scale")
    arrival = synth.arrival_times(cfg, 0)
    grads = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    table = psync.make_grad_table(grads)
    out = []
    for scaled in (False, True):
        pair = AsyncPair(cfg)
        psync.psync_order_by_arrival(torch.from_numpy(arrival).to(DEV), cfg.W, pair.d_order, pair.d_n)
        st, keep = pair.make_step(table)
        psync.psync_async_apply(st, d_gscale=torch.ones(cfg.W, device=DEV) if scaled else None)
        torch.cuda.synchronize()
        out.append({n: to_np(getattr(pair, n)) for n in STATE_NAMES})
    for n in STATE_NAMES:
        assert np.array_equal(out[0][n], out[1][n])


# ------------------------------------------------------------------ straggler statistics (section 3.1)
def _stats_gpu(a, iters=None):
    T, W = a.shape
    d_sorted = torch.full((T, W), -1.0, dtype=torch.float32, device=DEV)
    d_count = torch.full((W,), -1, dtype=torch.int32, device=DEV)
    d_mean = torch.zeros(W, dtype=torch.float64, device=DEV)
    d_median = torch.zeros(W, dtype=torch.float64, device=DEV)
    d_iters = None if iters is None else torch.from_numpy(iters).to(DEV)
    d_est = None if iters is None else torch.zeros(W, dtype=torch.float64, device=DEV)
    psync.psync_kth_arrival_stats(torch.from_numpy(a).to(DEV), d_sorted, d_count, d_mean, d_median, d_iters, d_est)
    torch.cuda.synchronize()
    out = dict(sorted=d_sorted.cpu().numpy(), count=d_count.cpu().numpy(), mean=d_mean.cpu().numpy(),
               median=d_median.cpu().numpy())
    if iters is not None:
        out["est_time"] = d_est.cpu().numpy()
    return out


@pytest.mark.parametrize("T,W", [(1, 1), (3, 3), (7, 33), (50, 106), (1000, 106), (257, 1024), (4001, 12)])
def test_kth_arrival_stats_match_oracle(T, W):
    rng = np.random.default_rng(T * 1000 + W)
    a = rng.lognormal(0, 0.25, (T, W)).astype(np.float32)
    a[rng.random((T, W)) < 0.02] *= 5
    ties = rng.random((T, W)) < 0.1
    a[ties] = rng.choice(np.array([1.0, 1.5, 0.0, -0.0, -1.0], np.float32), size=int(ties.sum()))
    a[rng.random((T, W)) < 0.05] = np.inf
    a[rng.random((T, W)) < 0.02] = np.nan
    if W > 2:
        a[:, -1] = np.inf                                     # a worker that never reports: last column count 0
    iters = rng.uniform(7e4, 1.4e5, W)
    got, want = _stats_gpu(a, iters), oracle.kth_arrival_stats(a, iters)
    assert np.array_equal(got["sorted"], want["sorted"])                         # bit-exact (0.0 == -0.0)
    assert np.array_equal(got["count"], want["count"])
    assert np.array_equal(got["median"], want["median"], equal_nan=True)         # exact selection
    ok = want["count"] > 0
    assert np.isnan(got["mean"][~ok]).all() and np.isnan(got["est_time"][~ok]).all()
    assert np.allclose(got["mean"][ok], want["mean"][ok], rtol=1e-13, atol=0)    # double sums, different order
    assert np.allclose(got["est_time"][ok], want["est_time"][ok], rtol=1e-13, atol=0)


def test_kth_arrival_stats_paper_shape_and_link_to_selection():
    """cfg3's arrival recipe, N+b = 106, 500 iterations: column N-1 of the sorted matrix is the time the
    synchronous server waits (t_Nth of the selection kernel), and the tail grows as in Fig. 4."""
    cfg = synth.PAPER_RMSPROP
    a = np.stack([synth.arrival_times(cfg, s) for s in range(500)])
    got = _stats_gpu(a)
    assert (np.diff(got["mean"]) >= 0).all() and (got["count"] == 500).all()
    assert got["mean"][-1] - got["mean"][-7] > got["mean"][60] - got["mean"][54]      # the last few are the slow ones
    d_kept = torch.zeros(cfg.N, dtype=torch.int32, device=DEV)
    d_status = torch.zeros(1, dtype=torch.int32, device=DEV)
    d_tn = torch.zeros(1, dtype=torch.float32, device=DEV)
    for t in (0, 17, 499):
        psync.psync_select_first_n(torch.from_numpy(a[t]).to(DEV), cfg.N, cfg.b, d_kept, d_status, d_tn)
        assert float(d_tn.item()) == got["sorted"][t, cfg.N - 1]


def test_kth_arrival_stats_invalid_arguments():
    L = psync.binding.lib()
    assert L.psync_kth_arrival_stats(None, 1, 1, None, None, None, None, None, None, None) == psync.PSYNC_EINVAL
    assert L.psync_kth_arrival_stats(8, 0, 1, 8, 8, 8, 8, None, None, None) == psync.PSYNC_EINVAL
    assert L.psync_kth_arrival_stats(8, 1, 1025, 8, 8, 8, 8, None, None, None) == psync.PSYNC_EINVAL
    assert L.psync_kth_arrival_stats(8, 1, 4, 8, 8, 8, 8, 8, None, None) == psync.PSYNC_EINVAL   # iters without est_time


def test_interp_iterations_and_fig6_estimate_on_the_gpu():
    """Fig. 5 -> Fig. 6: the paper's two printed points interpolated to every N, then mean time to
    collect N gradients x iterations(N) on cfg3's synthetic arrival times; bit-equal to the oracle."""
    W = 106
    d_iters = torch.full((W + 1,), -1.0, dtype=torch.float64, device=DEV)
    for N_pts, iters in (([50, 100], [137.5e3, 76.2e3]), ([50, 70, 80, 90, 100], [137.5e3, 111e3, 98.7e3, 85.1e3, 76.2e3]),
                         ([7], [5.0])):
        psync.psync_interp_iterations(N_pts, iters, W, d_iters)
        got = d_iters.cpu().numpy()
        assert np.array_equal(got[:W], oracle.interp_iterations(N_pts, iters, W)) and got[W] == -1.0
    psync.psync_interp_iterations([50, 100], [137.5e3, 76.2e3], W, d_iters)
    assert abs(float(d_iters[95]) - 81104.0) < 1e-6 and float(d_iters[74]) == 106850.0
    cfg = synth.PAPER_RMSPROP
    a = np.stack([synth.arrival_times(cfg, s) for s in range(300)])
    it = d_iters[:W].clone()
    d_sorted = torch.empty((300, W), dtype=torch.float32, device=DEV)
    d_count = torch.empty(W, dtype=torch.int32, device=DEV)
    d_mean = torch.empty(W, dtype=torch.float64, device=DEV)
    d_median = torch.empty(W, dtype=torch.float64, device=DEV)
    d_est = torch.empty(W, dtype=torch.float64, device=DEV)
    psync.psync_kth_arrival_stats(torch.from_numpy(a).to(DEV), d_sorted, d_count, d_mean, d_median, it, d_est)
    want = oracle.kth_arrival_stats(a, oracle.interp_iterations([50, 100], [137.5e3, 76.2e3], W))
    assert np.allclose(d_est.cpu().numpy(), want["est_time"], rtol=1e-13)
    best = int(np.argmin(d_est.cpu().numpy()[49:100])) + 50
    assert best == int(np.argmin(want["est_time"][49:100])) + 50 and 90 <= best <= 100   # a few backups win, as in Fig. 6
    L = psync.binding.lib()
    n2 = np.array([50, 50], np.int32); i2 = np.array([1.0, 2.0])
    assert L.psync_interp_iterations(n2.ctypes.data, i2.ctypes.data, 2, W, d_iters.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_interp_iterations(n2.ctypes.data, i2.ctypes.data, 0, W, d_iters.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_interp_iterations(None, i2.ctypes.data, 1, W, d_iters.data_ptr(), None) == psync.PSYNC_EINVAL


def test_probe_pipe_counts_its_lane_operations_and_validates():
    """Bench support (psync_probe_pipe): the reported operation count is CTAs x 256 threads x 8 chains x iters (x 2 packed)."""
    sink = torch.zeros(4, dtype=torch.float32, device=DEV)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    B = psync.binding
    assert B.psync_probe_pipe(0, 16, sink) == sms * 8 * 256 * 8 * 16
    assert B.psync_probe_pipe(1, 16, sink) == sms * 8 * 256 * 8 * 16 * 2
    assert B.psync_probe_pipe(2, 16, sink) == sms * 8 * 256 * 8 * 16
    torch.cuda.synchronize()
    L = B.lib()
    assert L.psync_probe_pipe(3, 16, sink.data_ptr(), None, None) == psync.PSYNC_EINVAL
    assert L.psync_probe_pipe(0, 0, sink.data_ptr(), None, None) == psync.PSYNC_EINVAL
    assert L.psync_probe_pipe(0, 16, None, None, None) == psync.PSYNC_EINVAL
