"""GPU parity for Alg. 2 run PER PARAMETER SERVER j (K4s, "Async-SGD Parameter Server j"): one
arrival order per server, the gradients as per-(worker, server) slices or flat buffers, over the (server, tile) work
list -- against oracle.async_apply_rows through the C ABI.  Orders bit-exact; theta / state / ema within Alg. 2's
tolerance (R21: rtol 1e-6 * max(10, K), atol 1e-6); bit-identity with the flat single-order kernel K4 is a
property checked at any size."""
from dataclasses import replace

import numpy as np
import pytest
import torch

import oracle
import paper_1702_05800_b200 as psync
from paper_1702_05800_b200 import synth

from _harness import ATOL_STEP, RTOL_BF16, RTOL_STEP, STATE_NAMES, assert_close, to_np
from test_gpu_slices import RAGGED, cut_slices, np_slices

pytestmark = pytest.mark.gpu
DEV = "cuda"

BASE = synth.Config(name="async_rows", cfg_id=16, P=70_003, M=7, N=13, b=0, arrival_sigma=0.3, opt=synth.SGD,
                    gamma=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0, ema_mode=synth.EMA_PRE, steps=3)


def rtol_async(K):
    return 1e-6 * max(10, K)


class RowsPair:
    """One parameter-server state on the GPU and on the host, stepped by Alg. 2 server by server."""

    def __init__(self, cfg, shard_off=None, state_misalign=0):
        self.cfg = cfg
        self.off = synth.shard_offsets(cfg) if shard_off is None else np.asarray(shard_off, dtype=np.int64)
        self.M = self.off.size - 1

        def place(t):
            if t is None or not state_misalign:
                return t
            buf = torch.empty(t.numel() + 8, dtype=t.dtype, device=DEV)
            view = buf[state_misalign:state_misalign + t.numel()]
            view.copy_(t)
            return view

        self.theta = place(synth.init_theta(cfg, DEV))
        s0, s1 = synth.init_state(cfg, DEV)
        self.state0, self.state1 = place(s0), place(s1)
        self.ema = place(self.theta.clone()) if cfg.ema_mode != synth.EMA_OFF else None
        self.d_off = torch.from_numpy(self.off).to(DEV)
        self.d_tiles = psync.psync_shard_worklist(self.d_off, cfg.grad_dtype)
        self.host = {n: to_np(getattr(self, n)) for n in STATE_NAMES}
        self.d_order = torch.full((self.M, cfg.W), -1, dtype=torch.int32, device=DEV)
        self.d_n = torch.full((self.M,), -7, dtype=torch.int32, device=DEV)

    def make_step(self, table, per_shard=True, slices=True, d_status=None, d_n=True, N=None):
        cfg = self.cfg
        return psync.make_step(self.off, cfg.W if N is None else N, cfg.W, table.grad_dtype, self.theta, self.ema,
                               self.state0, self.state1, opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma,
                               alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps, d_grads=table.d_ptrs,
                               d_kept=self.d_order, d_status=d_status, per_shard=per_shard, d_shard_off=self.d_off,
                               d_n_kept=self.d_n if d_n else None, kept_stride=cfg.W,
                               grad_layout=psync.PSYNC_GRADS_SLICES if slices else psync.PSYNC_GRADS_FLAT,
                               d_tile_start=self.d_tiles)

    def compare_and_sync(self, what, K):
        for n in STATE_NAMES:
            g = getattr(self, n)
            if g is not None:
                assert_close(to_np(g), self.host[n], rtol_async(K), ATOL_STEP, f"{what} {n}")
                self.host[n] = to_np(g)

    def step(self, s, arrival_rows, slices=True, offset_of=None, gammas=None, gscales=None, status=None):
        """arrival_rows fp32 [M][W]: order per server on the device, one K4s pass, the oracle server by server."""
        cfg = self.cfg
        flat = [synth.gradient(cfg, s, k, DEV) for k in range(cfg.W)]
        sl = cut_slices(flat, self.off, offset_of) if slices else None
        table = psync.make_slice_table(sl) if slices else psync.make_grad_table(flat)
        psync.psync_order_by_arrival_sharded(torch.from_numpy(arrival_rows).to(DEV), cfg.W, self.M, self.d_order, self.d_n)
        d_status = None if status is None else torch.from_numpy(status).to(DEV)
        st, keep = self.make_step(table, slices=slices, d_status=d_status)
        d_gamma = None if gammas is None else torch.from_numpy(gammas).to(DEV)
        d_gscale = None if gscales is None else torch.from_numpy(gscales).to(DEV)
        psync.psync_async_apply(st, d_gamma, d_gscale=d_gscale)
        torch.cuda.synchronize()
        order = np.full((self.M, cfg.W), -1, dtype=np.int32)
        n_arr = np.zeros(self.M, dtype=np.int32)
        for j in range(self.M):
            o = oracle.order_by_arrival(arrival_rows[j])
            order[j, :o.size], n_arr[j] = o, o.size
        assert np.array_equal(self.d_n.cpu().numpy(), n_arr)
        got = self.d_order.cpu().numpy()
        for j in range(self.M):                      # entries past the count are not written
            assert np.array_equal(got[j, :n_arr[j]], order[j, :n_arr[j]]), f"server {j}: arrival order differs"
        h = self.host
        safe = np.where(order < 0, 0, order)
        rc = oracle.async_apply_rows(self.off, np_slices(sl) if slices else [synth.as_numpy_grad(g) for g in flat], safe,
                                     h["theta"], h["ema"], h["state0"], h["state1"], slices=slices, per_shard=True,
                                     n_arrived=n_arr, status=status, gammas=gammas, gscales=gscales, opt=cfg.opt,
                                     ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho,
                                     eps=cfg.eps)
        assert rc == oracle.OK
        self.compare_and_sync(f"{cfg.name} step {s}", int(n_arr.max(initial=1)))
        return order, n_arr


# ------------------------------------------------------------------ K1c per server
def test_order_by_arrival_sharded_matches_the_oracle_row_by_row():
    rng = np.random.default_rng(1600)
    M, W = 37, 106
    a = rng.lognormal(0, 0.3, (M, W)).astype(np.float32)
    a[rng.random((M, W)) < 0.2] = 1.0
    a[rng.random((M, W)) < 0.05] = np.inf
    a[rng.random((M, W)) < 0.03] = np.nan
    a[5] = np.nan                                    # nothing reached server 5
    d_order = torch.full((M, W), -1, dtype=torch.int32, device=DEV)
    d_n = torch.full((M,), -7, dtype=torch.int32, device=DEV)
    psync.psync_order_by_arrival_sharded(torch.from_numpy(a).to(DEV), W, M, d_order, d_n)
    got, n = d_order.cpu().numpy(), d_n.cpu().numpy()
    for j in range(M):
        want = oracle.order_by_arrival(a[j])
        assert n[j] == want.size and np.array_equal(got[j, :want.size], want) and (got[j, want.size:] == -1).all()
    assert n[5] == 0
    L = psync.binding.lib()
    assert L.psync_order_by_arrival_sharded(None, 4, 2, None, None, None) == psync.PSYNC_EINVAL
    assert L.psync_order_by_arrival_sharded(8, 4, 0, 8, 8, None) == psync.PSYNC_EINVAL
    assert L.psync_order_by_arrival_sharded(8, 1025, 1, 8, 8, None) == psync.PSYNC_EINVAL


# ------------------------------------------------------------------ every template instance, lock-step
@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
@pytest.mark.parametrize("opt", [synth.SGD, synth.MOMENTUM, synth.RMSPROP_MOM])
@pytest.mark.parametrize("ema_mode", [synth.EMA_PRE, synth.EMA_POST, synth.EMA_OFF])
def test_every_template_instance_lockstep_on_ragged_slices(dtype, opt, ema_mode):
    cfg = replace(BASE, grad_dtype=dtype, opt=opt, ema_mode=ema_mode, name=f"arows_d{dtype}_o{opt}_e{ema_mode}")
    pair = RowsPair(cfg, shard_off=RAGGED)
    rng = np.random.default_rng(11)
    for s in range(3):
        # step 0: allocator-aligned slices (theta's slices are not co-aligned: transposed state); step 1: one odd
        # phase per server (head peel), per-iteration rates, two workers never reach some servers; step 2: phases
        # differ between workers (narrow loads), clip factors per worker
        offs = [None, lambda k, j: (3 * j + 1) % 8, lambda k, j: (5 * k + 3 * j) % 8][s]
        a = synth.arrival_times_per_server(cfg, s, server_sigma=0.3)
        gammas = gscales = None
        if s == 1:
            a[1::2, 2] = np.inf
            a[4:, 9] = np.nan
            gammas = rng.uniform(0.01, 0.09, cfg.W).astype(np.float32)
        if s == 2:
            gscales = rng.uniform(0.25, 1.0, cfg.W).astype(np.float32)
        order, n = pair.step(s, a, offset_of=offs, gammas=gammas, gscales=gscales)
        assert len({tuple(r) for r in order.tolist()}) > 1, "the servers should not all see the same order"


@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
@pytest.mark.parametrize("opt", [synth.MOMENTUM, synth.RMSPROP_MOM])
def test_flat_buffers_with_one_order_row_per_server(dtype, opt):
    cfg = replace(BASE, grad_dtype=dtype, opt=opt, name=f"arows_flat_d{dtype}_o{opt}")
    pair = RowsPair(cfg, shard_off=RAGGED)
    for s in range(2):
        pair.step(s, synth.arrival_times_per_server(cfg, s, server_sigma=0.3), slices=False)


@pytest.mark.parametrize("K", [1, 2, 3, 4, 5, 7, 8, 9, 12, 33])
def test_arrival_counts_cross_the_batch_boundaries(K):
    cfg = replace(BASE, N=K, P=20_011, M=3, opt=synth.RMSPROP_MOM, name=f"arows_K{K}")
    RowsPair(cfg).step(0, synth.arrival_times_per_server(cfg, 0, server_sigma=0.3))


def test_aligned_cuts_take_the_128_bit_state_path_and_misaligned_state_does_not():
    cfg = replace(BASE, P=65_536, M=4, ragged=False, opt=synth.RMSPROP_MOM, name="arows_aligned")
    RowsPair(cfg).step(0, synth.arrival_times_per_server(cfg, 0, server_sigma=0.3))
    RowsPair(cfg, state_misalign=1).step(0, synth.arrival_times_per_server(cfg, 0, server_sigma=0.3))


def test_failed_and_empty_servers_are_left_untouched():
    cfg = replace(BASE, opt=synth.MOMENTUM, name="arows_failed")
    pair = RowsPair(cfg, shard_off=RAGGED)
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    a[3] = np.inf                                                    # nothing reached server 3: K_3 = 0
    status = np.zeros(pair.M, dtype=np.int32)
    status[5] = psync.PSYNC_ETOOFEW                                  # server 5 is marked failed
    before = {n: to_np(getattr(pair, n)) for n in STATE_NAMES}
    order, n = pair.step(0, a, status=status)
    assert n[3] == 0
    for j in (3, 5):
        lo, hi = int(pair.off[j]), int(pair.off[j + 1])
        for nm in STATE_NAMES:
            if before[nm] is not None:
                assert np.array_equal(to_np(getattr(pair, nm))[lo:hi], before[nm][lo:hi]), (j, nm)
    lo, hi = int(pair.off[4]), int(pair.off[5])
    assert not np.array_equal(to_np(pair.theta)[lo:hi], before["theta"][lo:hi])


def test_one_shared_order_on_slices_equals_the_flat_single_order_kernel_bit_for_bit():
    """per_shard = 0 with the slices layout: every server applies row 0.  K4s must give the bits of K4."""
    for dtype, opt in ((synth.F32, synth.RMSPROP_MOM), (synth.BF16, synth.MOMENTUM), (synth.F32, synth.SGD)):
        cfg = replace(BASE, P=200_003, M=9, N=11, grad_dtype=dtype, opt=opt, name="arows_vs_k4")
        a = synth.arrival_times(cfg, 0)
        flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
        rng = np.random.default_rng(5)
        gam = torch.from_numpy(rng.uniform(0.01, 0.09, cfg.W).astype(np.float32)).to(DEV)
        gsc = torch.from_numpy(rng.uniform(0.25, 1.0, cfg.W).astype(np.float32)).to(DEV)
        one = RowsPair(cfg)
        d_order = torch.full((cfg.W,), -1, dtype=torch.int32, device=DEV)
        d_n = torch.full((1,), -7, dtype=torch.int32, device=DEV)
        psync.psync_order_by_arrival(torch.from_numpy(a).to(DEV), cfg.W, d_order, d_n)
        t_flat = psync.make_grad_table(flat)
        st, keep = psync.make_step(one.off, cfg.W, cfg.W, t_flat.grad_dtype, one.theta, one.ema, one.state0, one.state1,
                                   opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu,
                                   rho=cfg.rho, eps=cfg.eps, d_grads=t_flat.d_ptrs, d_kept=d_order, d_n_kept=d_n,
                                   kept_stride=cfg.W)
        psync.psync_async_apply(st, gam, d_gscale=gsc)
        two = RowsPair(cfg)
        sl = cut_slices(flat, two.off, lambda k, j: (k + j) % 4)
        t_sl = psync.make_slice_table(sl)
        two.d_order[0].copy_(d_order)
        two.d_n[:1].copy_(d_n)
        st2, keep2 = two.make_step(t_sl, per_shard=False)
        psync.psync_async_apply(st2, gam, d_gscale=gsc)
        torch.cuda.synchronize()
        for n in STATE_NAMES:
            if getattr(one, n) is not None:
                assert np.array_equal(to_np(getattr(one, n)), to_np(getattr(two, n))), (dtype, opt, n)


@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
@pytest.mark.parametrize("side", ["low", "high"])
def test_second_moment_outside_the_packed_rsqrt_range_is_redone_with_the_checked_routine(dtype, side):
    """RMSProp: on a sparse set of elements ms + eps stays below 2^-63 (ms_0 = eps = 1e-30, gradients ~1e-12) or above
    2^65 (ms_0 = 1e30) for the whole pass: outside the range of the unchecked packed rsqrt, so the warp redoes its units
    from memory with the checked scalar routine.  Both K4s and K4."""
    if side == "low":
        cfg = replace(BASE, grad_dtype=dtype, opt=synth.RMSPROP_MOM, eps=1e-30, gamma=1e-4, grad_dist=("normal", 1e-12),
                      name=f"arows_range_low_d{dtype}")
        ms0 = 1e-30
    else:
        cfg = replace(BASE, grad_dtype=dtype, opt=synth.RMSPROP_MOM, name=f"arows_range_high_d{dtype}")
        ms0 = 1e30
    rng = np.random.default_rng(21)
    tiny = torch.from_numpy(np.unique(rng.integers(0, cfg.P, 400))).to(DEV)
    pair = RowsPair(cfg, shard_off=RAGGED)
    pair.state0[tiny] = ms0
    pair.host["state0"] = to_np(pair.state0)
    pair.step(0, synth.arrival_times_per_server(cfg, 0, server_sigma=0.3))
    assert bool(torch.isfinite(pair.theta).all()) and bool(torch.isfinite(pair.state1).all())
    # the flat single-order kernel on the same data
    one = RowsPair(cfg, shard_off=[0, cfg.P])
    one.state0[tiny] = ms0
    one.host["state0"] = to_np(one.state0)
    a = synth.arrival_times(cfg, 0)
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    table = psync.make_grad_table(flat)
    d_order = torch.full((cfg.W,), -1, dtype=torch.int32, device=DEV)
    d_n = torch.full((1,), -7, dtype=torch.int32, device=DEV)
    psync.psync_order_by_arrival(torch.from_numpy(a).to(DEV), cfg.W, d_order, d_n)
    st, keep = psync.make_step(one.off, cfg.W, cfg.W, table.grad_dtype, one.theta, one.ema, one.state0, one.state1,
                               opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu,
                               rho=cfg.rho, eps=cfg.eps, d_grads=table.d_ptrs, d_kept=d_order, d_n_kept=d_n,
                               kept_stride=cfg.W)
    psync.psync_async_apply(st)
    torch.cuda.synchronize()
    h = one.host
    order = oracle.order_by_arrival(a)
    rc = oracle.async_apply(one.off, [synth.as_numpy_grad(g) for g in flat], order, h["theta"], h["ema"], h["state0"],
                            h["state1"], opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha,
                            mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
    assert rc == oracle.OK
    one.compare_and_sync("K4 range", order.size)


def test_many_tiny_servers_and_the_maximum_worker_count():
    """M = 600 ragged servers of ~50 parameters (every tile mostly empty, most of every server is head / tail peel);
    then W = 1024 arrivals on a small vector (the shared tables are full)."""
    cfg = replace(BASE, P=30_011, M=600, opt=synth.MOMENTUM, name="arows_tiny_servers")
    RowsPair(cfg).step(0, synth.arrival_times_per_server(cfg, 0, server_sigma=0.3))
    cfg = replace(BASE, N=1024, P=3_001, M=3, opt=synth.MOMENTUM, grad_dist=("normal", 1e-4), name="arows_K1024")
    order, n = RowsPair(cfg).step(0, synth.arrival_times_per_server(cfg, 0, server_sigma=0.3))
    assert (n == 1024).all()


def test_abi_validation_and_a_foreign_work_list_touch_nothing():
    cfg = replace(BASE, P=4096, M=2, N=3, ragged=False, name="arows_abi")
    pair = RowsPair(cfg)
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    table = psync.make_slice_table(cut_slices(flat, pair.off))
    pair.d_order[:] = torch.arange(3, dtype=torch.int32, device=DEV)
    pair.d_n.fill_(3)
    before = to_np(pair.theta)
    st, keep = pair.make_step(table)
    st.d_tile_start = None
    assert psync.psync_async_apply(st, check=False) == psync.PSYNC_EINVAL          # slices need the work list
    st, keep = pair.make_step(psync.make_grad_table(flat), slices=False)
    st.d_tile_start = None
    assert psync.psync_async_apply(st, check=False) == psync.PSYNC_EUNSUPPORTED    # rows without a work list
    st, keep = pair.make_step(table)
    st.d_shard_off = None
    assert psync.psync_async_apply(st, check=False) == psync.PSYNC_EINVAL
    # a work list built for the other gradient dtype: detected on the device
    pair.d_tiles = psync.psync_shard_worklist(torch.from_numpy(np.array([0, 2048, 8192], np.int64)).to(DEV), synth.F32)
    st, keep = pair.make_step(table)
    assert psync.psync_async_apply(st) == psync.PSYNC_OK
    # a count nobody wrote
    pair.d_tiles = psync.psync_shard_worklist(pair.d_off, synth.F32)
    pair.d_n.fill_(-7)
    st, keep = pair.make_step(table)
    assert psync.psync_async_apply(st) == psync.PSYNC_OK
    pair.d_n.fill_(4)                                                               # > kept_stride = W = 3
    assert psync.psync_async_apply(st) == psync.PSYNC_OK
    torch.cuda.synchronize()
    assert np.array_equal(to_np(pair.theta), before)
    pair.d_n.fill_(3)
    assert psync.psync_async_apply(st) == psync.PSYNC_OK
    torch.cuda.synchronize()
    assert not np.array_equal(to_np(pair.theta), before)


def test_full_size_cfg3_shape_every_element_on_separately_allocated_slices():
    """cfg3's shape (P = 25,165,824, M = 20 ragged, W = 106, RMSProp + EMA) through Alg. 2 per server: 2,120 separately
    allocated slices (every third one placed 1-3 elements off its allocation), 20 different arrival orders, EVERY
    element against the oracle."""
    cfg = replace(synth.PAPER_RMSPROP, N=106, b=0, ema_mode=synth.EMA_PRE, name="arows_cfg3")
    free, _ = torch.cuda.mem_get_info()
    if cfg.footprint_bytes * 1.25 > free:
        pytest.skip("not enough free HBM")
    pair = RowsPair(cfg)
    sl = []
    for k in range(cfg.W):
        g = synth.gradient(cfg, 0, k, DEV)
        sl.append(cut_slices([g], pair.off, lambda _k, j, k=k: ((k + j) % 4) if (k + j) % 3 == 0 else 0)[0])
        del g
    table = psync.make_slice_table(sl)
    a = synth.arrival_times_per_server(cfg, 0)
    a[7, 13] = np.inf                                                 # worker 13's slice never reaches server 7
    psync.psync_order_by_arrival_sharded(torch.from_numpy(a).to(DEV), cfg.W, pair.M, pair.d_order, pair.d_n)
    st, keep = pair.make_step(table)
    psync.psync_async_apply(st)
    torch.cuda.synchronize()
    order = np.zeros((pair.M, cfg.W), dtype=np.int32)
    n_arr = np.zeros(pair.M, dtype=np.int32)
    for j in range(pair.M):
        o = oracle.order_by_arrival(a[j])
        order[j, :o.size], n_arr[j] = o, o.size
    assert n_arr[7] == 105 and np.array_equal(pair.d_n.cpu().numpy(), n_arr)
    h = pair.host
    rc = oracle.async_apply_rows(pair.off, np_slices(sl), order, h["theta"], h["ema"], h["state0"], h["state1"],
                                 slices=True, per_shard=True, n_arrived=n_arr, opt=cfg.opt, ema_mode=cfg.ema_mode,
                                 gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
    assert rc == oracle.OK
    pair.compare_and_sync("async rows cfg3 (every element)", 106)


# ------------------------------------------------------------------ AsyncServerStep: the calls of one batch, chained
def test_async_server_step_flat_with_clipping_schedule_and_staleness_chained_batches():
    """Order -> clip factors -> learning rates -> K iterations -> staleness, enqueued without a host sync, two batches;
    every piece against its own oracle function."""
    cfg = replace(BASE, P=50_021, M=5, opt=synth.RMSPROP_MOM, grad_dist=("normal", 2e-3), name="aserver_flat")
    off = synth.shard_offsets(cfg)
    theta = synth.init_theta(cfg, DEV)
    s0, s1 = synth.init_state(cfg, DEV)
    ema = theta.clone()
    lr = (0.045, 0.94, 1.0 / 40.0)
    clip = 0.4                                              # ||G|| ~ 2e-3 * sqrt(P) ~ 0.45: some workers are clipped
    srv = psync.AsyncServerStep(off, cfg.W, theta, ema, s0, s1, cfg.opt, cfg.ema_mode, alpha=cfg.alpha, mu=cfg.mu,
                                rho=cfg.rho, eps=cfg.eps, clip=clip, lr=lr, track_staleness=True, lag=2)
    h = {"theta": to_np(theta), "ema": to_np(ema), "state0": to_np(s0), "state1": to_np(s1)}
    read = np.zeros(cfg.W, np.int64)
    t_srv = 0
    for s in range(2):
        grads = [synth.gradient(cfg, s, k, DEV) for k in range(cfg.W)]
        for k in range(0, cfg.W, 2):
            grads[k].mul_(0.5)                              # these workers' norms are within the bound: factor 1
        a = synth.arrival_times(cfg, s)
        if s == 1:
            a[4] = np.inf
        srv.set_gradients(grads)
        srv.apply(torch.from_numpy(a).to(DEV))
        torch.cuda.synchronize()
        order = oracle.order_by_arrival(a)
        K = order.size
        np_g = [synth.as_numpy_grad(g) for g in grads]
        scales = oracle.clip_scales(np_g, clip)
        gammas = oracle.lr_schedule(lr[0], lr[1], s * cfg.W, cfg.W, lr[2])
        assert np.array_equal(srv.d_order.cpu().numpy()[0, :K], order) and int(srv.d_n_arrived.item()) == K
        assert np.array_equal(srv.d_gscale.cpu().numpy(), scales) and (scales < 1).any() and (scales == 1).any()
        assert np.array_equal(srv.d_gamma.cpu().numpy(), gammas)
        rc = oracle.async_apply(off, np_g, order, h["theta"], h["ema"], h["state0"], h["state1"], gammas=gammas[:K].copy(),
                                gscales=scales[order].copy(), opt=cfg.opt, ema_mode=cfg.ema_mode, alpha=cfg.alpha, mu=cfg.mu,
                                rho=cfg.rho, eps=cfg.eps)
        assert rc == oracle.OK
        for n, t in (("theta", theta), ("ema", ema), ("state0", s0), ("state1", s1)):
            assert_close(to_np(t), h[n], rtol_async(K), ATOL_STEP, f"aserver batch {s} {n}")
            h[n] = to_np(t)
        st, stale, read, stats = oracle.staleness(read, order, t_srv, lag=2)
        t_srv += K
        assert st == oracle.OK and int(srv.d_stale_status.item()) == 0 and int(srv.d_t.item()) == t_srv
        assert np.array_equal(srv.d_staleness.cpu().numpy()[0, :K], stale)
        assert np.array_equal(srv.d_read_iter.cpu().numpy()[0], read)
        assert np.array_equal(srv.d_stale_stats.cpu().numpy()[0], stats)


def test_async_server_step_schedule_follows_the_applied_count_over_partial_batches():
    """L84-87: every received gradient is one iteration, so after a batch of K < W arrivals the schedule (L315) advances
    by K, not W.  Three batches, the middle one partial (and the first too), no t0 given: the rates of batch s must be
    gamma_{t + i} with t = the sum of the K of the batches before it -- the device counter, no host synchronisation."""
    cfg = replace(BASE, P=9_001, M=3, opt=synth.SGD, name="aserver_partial")
    off = synth.shard_offsets(cfg)
    theta = synth.init_theta(cfg, DEV)
    ema = theta.clone()
    lr = (0.045, 0.94, 1.0 / 7.0)                           # a steep schedule: an off-by-(W-K) start is far outside 1 ulp
    srv = psync.AsyncServerStep(off, cfg.W, theta, ema, None, None, cfg.opt, cfg.ema_mode, alpha=cfg.alpha, lr=lr)
    h = {"theta": to_np(theta), "ema": to_np(ema)}
    applied = 0
    missing = [(1,), (0, 3, 4), ()]
    for s in range(3):
        grads = [synth.gradient(cfg, s, k, DEV) for k in range(cfg.W)]
        a = synth.arrival_times(cfg, s)
        a[list(missing[s])] = np.inf
        srv.set_gradients(grads)
        srv.apply(torch.from_numpy(a).to(DEV))              # no synchronisation between the calls of a batch
        torch.cuda.synchronize()
        order = oracle.order_by_arrival(a)
        K = order.size
        assert K == cfg.W - len(missing[s])
        gammas = oracle.lr_schedule(lr[0], lr[1], applied, cfg.W, lr[2])
        assert np.array_equal(srv.d_gamma.cpu().numpy(), gammas), f"batch {s}: schedule does not start at t = {applied}"
        assert int(srv.d_t_sched.item()) == applied
        if 0 < applied < s * cfg.W:
            assert not np.array_equal(gammas, oracle.lr_schedule(lr[0], lr[1], s * cfg.W, cfg.W, lr[2]))
        rc = oracle.async_apply(off, [synth.as_numpy_grad(g) for g in grads], order, h["theta"], h["ema"], None, None,
                                gammas=gammas[:K].copy(), opt=cfg.opt, ema_mode=cfg.ema_mode, alpha=cfg.alpha)
        assert rc == oracle.OK
        for n, t in (("theta", theta), ("ema", ema)):
            assert_close(to_np(t), h[n], rtol_async(K), ATOL_STEP, f"aserver partial batch {s} {n}")
            h[n] = to_np(t)
        applied += K
    srv.set_gradients(grads)
    srv.apply(torch.from_numpy(a).to(DEV), t0=5)            # an explicit t0 restarts the count
    torch.cuda.synchronize()
    assert np.array_equal(srv.d_gamma.cpu().numpy(), oracle.lr_schedule(lr[0], lr[1], 5, cfg.W, lr[2]))
    assert int(srv.d_t_sched.item()) == 5


def test_async_server_step_per_server_on_slices_chained_batches():
    cfg = replace(BASE, opt=synth.MOMENTUM, grad_dtype=synth.BF16, name="aserver_rows")
    off = np.asarray(RAGGED, dtype=np.int64)
    theta = synth.init_theta(cfg, DEV)
    s0, _ = synth.init_state(cfg, DEV)
    ema = theta.clone()
    lr = (0.045, 0.94, 1.0 / 40.0)
    srv = psync.AsyncServerStep(off, cfg.W, theta, ema, s0, None, cfg.opt, cfg.ema_mode, alpha=cfg.alpha, mu=cfg.mu,
                                per_server=True, lr=lr)
    h = {"theta": to_np(theta), "ema": to_np(ema), "state0": to_np(s0)}
    M = off.size - 1
    for s in range(2):
        flat = [synth.gradient(cfg, s, k, DEV) for k in range(cfg.W)]
        sl = cut_slices(flat, off, lambda k, j: (k + 2 * j) % 8 if s else 0)
        a = synth.arrival_times_per_server(cfg, s, server_sigma=0.3)
        a[2, 5] = np.nan
        srv.set_gradient_slices(sl)
        srv.apply(torch.from_numpy(a).to(DEV))
        torch.cuda.synchronize()
        order = np.zeros((M, cfg.W), dtype=np.int32)
        n_arr = np.zeros(M, dtype=np.int32)
        for j in range(M):
            o = oracle.order_by_arrival(a[j])
            order[j, :o.size], n_arr[j] = o, o.size
        assert np.array_equal(srv.d_n_arrived.cpu().numpy(), n_arr) and n_arr[2] == cfg.W - 1
        gammas = oracle.lr_schedule(lr[0], lr[1], s * cfg.W, cfg.W, lr[2])
        rc = oracle.async_apply_rows(off, np_slices(sl), order, h["theta"], h["ema"], h["state0"], None, slices=True,
                                     per_shard=True, n_arrived=n_arr, gammas=gammas, opt=cfg.opt, ema_mode=cfg.ema_mode,
                                     alpha=cfg.alpha, mu=cfg.mu)
        assert rc == oracle.OK
        for n, t in (("theta", theta), ("ema", ema), ("state0", s0)):
            assert_close(to_np(t), h[n], rtol_async(cfg.W), ATOL_STEP, f"aserver rows batch {s} {n}")
            h[n] = to_np(t)


# ------------------------------------------------------------------ K5s: clip factors of sliced gradients
@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
def test_clip_scales_slices_match_the_oracle_and_the_flat_kernel(dtype):
    """Norm over ALL of a worker's slices: ragged servers (an empty and a one-element one), slices at odd element offsets,
    several 8192-unit chunks per server and a partial last chunk."""
    cfg = replace(BASE, P=300_007, M=5, N=9, grad_dtype=dtype, grad_dist=("normal", 2e-3), name=f"clips_d{dtype}")
    off = np.array([0, 1, 1, 70_001, 140_000, 300_007], np.int64)
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    for k in range(0, cfg.W, 2):
        flat[k].mul_(0.25)
    sl = cut_slices(flat, off, lambda k, j: (3 * k + j) % 8)
    table = psync.make_slice_table(sl)
    d_off = torch.from_numpy(off).to(DEV)
    clip = 0.6
    nbytes = psync.psync_clip_slices_workspace_bytes(cfg.W, off, table.grad_dtype)
    assert nbytes > 0
    d_work = torch.empty((nbytes + 7) // 8, dtype=torch.float64, device=DEV)
    d_scales = torch.full((cfg.W,), -1.0, device=DEV)
    psync.psync_clip_scales_slices(table, off, d_off, clip, d_scales, d_work)
    torch.cuda.synchronize()
    want = oracle.clip_scales_slices(off, np_slices(sl), clip)
    got = d_scales.cpu().numpy()
    assert (want < 1).any() and (want == 1).any()
    assert np.array_equal(got, want)
    # the flat kernel on the uncut buffers gives the same factors
    ft = psync.make_grad_table(flat)
    d_w2 = torch.empty(psync.psync_clip_workspace_bytes(cfg.W, cfg.P, ft.grad_dtype) // 8, dtype=torch.float64, device=DEV)
    d_s2 = torch.full((cfg.W,), -1.0, device=DEV)
    psync.psync_clip_scales(ft, clip, d_s2, d_w2)
    torch.cuda.synchronize()
    assert np.array_equal(d_s2.cpu().numpy(), got)
    L = psync.binding.lib()
    assert L.psync_clip_scales_slices(None, 3, 2, None, None, 0, 1.0, None, None, 0, None) == psync.PSYNC_EINVAL
    assert psync.psync_clip_scales_slices(table, off, d_off, 0.0, d_scales, d_work, check=False) == psync.PSYNC_EINVAL
    assert psync.psync_clip_scales_slices(table, off, d_off, clip, d_scales, d_work[:2], check=False) == psync.PSYNC_EINVAL


def test_async_server_step_clips_sliced_gradients_per_server():
    cfg = replace(BASE, P=50_021, M=7, opt=synth.SGD, grad_dist=("normal", 2e-3), name="aserver_clip_slices")
    off = np.asarray(synth.shard_offsets(cfg), dtype=np.int64)
    theta = synth.init_theta(cfg, DEV)
    ema = theta.clone()
    clip = 0.4
    srv = psync.AsyncServerStep(off, cfg.W, theta, ema, None, None, cfg.opt, cfg.ema_mode, alpha=cfg.alpha,
                                per_server=True, clip=clip)
    h = {"theta": to_np(theta), "ema": to_np(ema)}
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    for k in range(1, cfg.W, 2):
        flat[k].mul_(0.5)
    sl = cut_slices(flat, off, lambda k, j: (k + j) % 4)
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    srv.set_gradient_slices(sl)
    srv.apply(torch.from_numpy(a).to(DEV), cfg.gamma)
    torch.cuda.synchronize()
    scales = oracle.clip_scales_slices(off, np_slices(sl), clip)
    assert np.array_equal(srv.d_gscale.cpu().numpy(), scales) and (scales < 1).any() and (scales == 1).any()
    order = np.stack([oracle.order_by_arrival(a[j]) for j in range(cfg.M)])
    rc = oracle.async_apply_rows(off, np_slices(sl), order, h["theta"], h["ema"], slices=True, per_shard=True,
                                 gscales=scales, opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha)
    assert rc == oracle.OK
    assert_close(to_np(theta), h["theta"], rtol_async(cfg.W), ATOL_STEP, "aserver clip slices theta")
    assert_close(to_np(ema), h["ema"], rtol_async(cfg.W), ATOL_STEP, "aserver clip slices ema")


def test_every_server_of_a_per_server_pass_has_the_bits_of_the_flat_kernel_run_with_that_servers_order():
    """K4s with M different orders == for every j, K4 (flat, one order) run with server j's order, restricted to
    server j's slice: bit for bit, RMSProp + per-iteration rates + clip factors."""
    cfg = replace(BASE, P=120_007, M=6, N=11, opt=synth.RMSPROP_MOM, name="arows_vs_k4_rows")
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.4)
    a[3, 7] = np.inf
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    rng = np.random.default_rng(5)
    gam = torch.from_numpy(rng.uniform(0.01, 0.09, cfg.W).astype(np.float32)).to(DEV)
    gsc = torch.from_numpy(rng.uniform(0.25, 1.0, cfg.W).astype(np.float32)).to(DEV)
    rows = RowsPair(cfg)
    sl = cut_slices(flat, rows.off, lambda k, j: (k + j) % 4)
    psync.psync_order_by_arrival_sharded(torch.from_numpy(a).to(DEV), cfg.W, rows.M, rows.d_order, rows.d_n)
    st, keep = rows.make_step(psync.make_slice_table(sl))
    psync.psync_async_apply(st, gam, d_gscale=gsc)
    torch.cuda.synchronize()
    t_flat = psync.make_grad_table(flat)
    assert len({tuple(r) for r in rows.d_order.cpu().numpy().tolist()}) == rows.M
    for j in range(rows.M):
        one = RowsPair(cfg)
        st1, keep1 = psync.make_step(one.off, cfg.W, cfg.W, t_flat.grad_dtype, one.theta, one.ema, one.state0, one.state1,
                                     opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu,
                                     rho=cfg.rho, eps=cfg.eps, d_grads=t_flat.d_ptrs, d_kept=rows.d_order[j],
                                     d_n_kept=rows.d_n[j:j + 1], kept_stride=cfg.W)
        psync.psync_async_apply(st1, gam, d_gscale=gsc)
        torch.cuda.synchronize()
        lo, hi = int(rows.off[j]), int(rows.off[j + 1])
        for n in STATE_NAMES:
            assert np.array_equal(to_np(getattr(rows, n))[lo:hi], to_np(getattr(one, n))[lo:hi]), (j, n)


def test_async_server_step_is_capturable_in_a_cuda_graph_and_replays_bit_identically():
    """One batch of Alg. 2 per server on slices with clipping and a schedule -- order, norms (3 launches), rates, the
    one-pass application -- makes no synchronising call: captured once, replayed with new arrival times, the result is
    bit-identical to the same calls made eagerly."""
    cfg = replace(BASE, P=50_021, M=7, opt=synth.MOMENTUM, grad_dist=("normal", 2e-3), name="aserver_graph")
    off = np.asarray(synth.shard_offsets(cfg), dtype=np.int64)
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    sl = cut_slices(flat, off, lambda k, j: (k + j) % 4)

    def server():
        theta = synth.init_theta(cfg, DEV)
        s0, _ = synth.init_state(cfg, DEV)
        srv = psync.AsyncServerStep(off, cfg.W, theta, theta.clone(), s0, None, cfg.opt, cfg.ema_mode, alpha=cfg.alpha,
                                    mu=cfg.mu, per_server=True, clip=0.4, lr=(0.045, 0.94, 1.0 / 40.0))
        srv.set_gradient_slices(sl)
        return srv

    arrs = [torch.from_numpy(synth.arrival_times_per_server(cfg, s, server_sigma=0.3)).to(DEV) for s in range(3)]
    eager = server()
    for s in (1, 2):
        eager.apply(arrs[s], t0=0)
    torch.cuda.synchronize()

    cap = server()
    d_arr = arrs[0].clone()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        snap = {n: getattr(cap, n).clone() for n in ("theta", "ema", "state0")}
        cap.apply(d_arr, t0=0, stream=side)                      # warm-up outside capture (builds work list, workspace)
        side.synchronize()
        for n, v in snap.items():
            getattr(cap, n).copy_(v)
        with torch.cuda.graph(graph, stream=side):
            cap.apply(d_arr, t0=0, stream=side)
    torch.cuda.synchronize()
    for s in (1, 2):
        d_arr.copy_(arrs[s])
        graph.replay()
    torch.cuda.synchronize()
    for n in ("theta", "ema", "state0"):
        assert np.array_equal(to_np(getattr(cap, n)), to_np(getattr(eager, n))), n
    assert not np.array_equal(to_np(cap.theta), to_np(snap["theta"]))


def test_staleness_per_server_chained_batches_match_the_oracle_row_by_row():
    """psync_staleness_sharded: every server keeps its own counter and its own record of when each worker last read from
    it; row j is exactly the single-order bookkeeping (the pinned oracle function) on server j's order.  Three chained
    batches, different counts per server, a fixed lag, one server with a bad batch (a worker listed twice)."""
    rng = np.random.default_rng(77)
    M, W, lag = 5, 40, 3
    d_read = torch.zeros((M, W), dtype=torch.int64, device=DEV)
    d_t = torch.zeros(M, dtype=torch.int64, device=DEV)
    d_order = torch.full((M, W), -1, dtype=torch.int32, device=DEV)
    d_n = torch.zeros(M, dtype=torch.int32, device=DEV)
    d_st = torch.full((M, W), -7, dtype=torch.int64, device=DEV)
    d_stats = torch.full((M, 6), -7.0, dtype=torch.float64, device=DEV)
    d_status = torch.full((M,), -9, dtype=torch.int32, device=DEV)
    read = np.zeros((M, W), np.int64)
    t = np.zeros(M, np.int64)
    for batch in range(3):
        a = rng.lognormal(0, 0.4, (M, W)).astype(np.float32)
        a[rng.random((M, W)) < 0.15] = np.inf
        psync.psync_order_by_arrival_sharded(torch.from_numpy(a).to(DEV), W, M, d_order, d_n)
        if batch == 1:                                    # server 2's order row is corrupted: a worker appears twice
            torch.cuda.synchronize()
            row = d_order[2].clone()
            row[1] = row[0]
            d_order[2].copy_(row)
        psync.psync_staleness_sharded(d_read, d_order, d_t, d_st, d_stats, d_status, d_n_arrived=d_n, lag=lag)
        torch.cuda.synchronize()
        got_order, got_n = d_order.cpu().numpy(), d_n.cpu().numpy()
        for j in range(M):
            order = got_order[j, :got_n[j]].copy()
            rc, stale, nxt, stats = oracle.staleness(read[j].copy(), order, int(t[j]), lag=lag)
            if batch == 1 and j == 2:
                assert rc != oracle.OK and int(d_status[j].item()) == psync.PSYNC_EINVAL
                assert np.array_equal(d_read[j].cpu().numpy(), read[j]) and int(d_t[j].item()) == t[j]
                continue
            assert rc == oracle.OK and int(d_status[j].item()) == 0
            read[j], t[j] = nxt, t[j] + order.size
            assert np.array_equal(d_st[j].cpu().numpy()[:order.size], stale)
            assert np.array_equal(d_read[j].cpu().numpy(), read[j]) and int(d_t[j].item()) == t[j]
            assert np.array_equal(d_stats[j].cpu().numpy(), stats)
    L = psync.binding.lib()
    assert L.psync_staleness_sharded(None, 4, 2, None, None, 0, None, 0, None, None, None, None) == psync.PSYNC_EINVAL
    assert L.psync_staleness_sharded(8, 4, 0, 8, None, 0, 8, 0, 8, 8, 8, None) == psync.PSYNC_EINVAL


def test_fixed_count_without_a_count_array_applies_exactly_N_per_server():
    """d_n_kept = NULL: every server applies the first step->N entries of its order row (here N = 9 of 13 arrivals)."""
    cfg = replace(BASE, opt=synth.MOMENTUM, name="arows_fixedN")
    pair = RowsPair(cfg, shard_off=RAGGED)
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    sl = cut_slices(flat, pair.off)
    psync.psync_order_by_arrival_sharded(torch.from_numpy(a).to(DEV), cfg.W, pair.M, pair.d_order, pair.d_n)
    st, keep = pair.make_step(psync.make_slice_table(sl), d_n=False, N=9)
    psync.psync_async_apply(st)
    torch.cuda.synchronize()
    order = np.stack([oracle.order_by_arrival(a[j]) for j in range(pair.M)])
    h = pair.host
    rc = oracle.async_apply_rows(pair.off, np_slices(sl), order, h["theta"], h["ema"], h["state0"], h["state1"], slices=True,
                                 per_shard=True, n_arrived=np.full(pair.M, 9, np.int32), opt=cfg.opt, ema_mode=cfg.ema_mode,
                                 gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
    assert rc == oracle.OK
    pair.compare_and_sync("fixed N per server", 9)


def test_async_step_device_is_the_two_calls_in_one_and_validates_its_outputs():
    cfg = replace(BASE, opt=synth.RMSPROP_MOM, name="arows_onecall")
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    a[2, 4] = np.inf
    d_a = torch.from_numpy(a).to(DEV)
    two, one = RowsPair(cfg, shard_off=RAGGED), RowsPair(cfg, shard_off=RAGGED)
    sl = cut_slices(flat, two.off, lambda k, j: (k + j) % 4)
    table = psync.make_slice_table(sl)
    psync.psync_order_by_arrival_sharded(d_a, cfg.W, two.M, two.d_order, two.d_n)
    st2, keep2 = two.make_step(table)
    psync.psync_async_apply(st2)
    st1, keep1 = one.make_step(table, N=1)               # N is ignored by the one-call form
    psync.psync_async_step_device(st1, d_a)
    torch.cuda.synchronize()
    assert np.array_equal(one.d_n.cpu().numpy(), two.d_n.cpu().numpy()) and int(one.d_n[2].item()) == cfg.W - 1
    for n in STATE_NAMES:
        assert np.array_equal(to_np(getattr(one, n)), to_np(getattr(two, n))), n
    before = to_np(one.theta)
    st1.d_n_kept = None
    assert psync.psync_async_step_device(st1, d_a, check=False) == psync.PSYNC_EINVAL
    st1, keep1 = one.make_step(table)
    st1.kept_stride = cfg.W - 1
    assert psync.psync_async_step_device(st1, d_a, check=False) == psync.PSYNC_EINVAL
    torch.cuda.synchronize()
    assert np.array_equal(to_np(one.theta), before)
    # flat buffers, one order: d_arrival [W]
    f1, f2 = RowsPair(cfg), RowsPair(cfg)
    ft = psync.make_grad_table(flat)
    d_o = torch.full((cfg.W,), -1, dtype=torch.int32, device=DEV)
    d_n = torch.zeros(1, dtype=torch.int32, device=DEV)

    def flat_step(pair):
        return psync.make_step(pair.off, cfg.W, cfg.W, ft.grad_dtype, pair.theta, pair.ema, pair.state0, pair.state1,
                               opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho,
                               eps=cfg.eps, d_grads=ft.d_ptrs, d_kept=d_o, d_n_kept=d_n, kept_stride=cfg.W)
    sa, ka = flat_step(f1)
    psync.psync_order_by_arrival(d_a[0], cfg.W, d_o, d_n)
    psync.psync_async_apply(sa)
    sb, kb = flat_step(f2)
    psync.psync_async_step_device(sb, d_a[0])
    torch.cuda.synchronize()
    for n in STATE_NAMES:
        assert np.array_equal(to_np(getattr(f1, n)), to_np(getattr(f2, n))), n


# ------------------------------------------------------------------ guard bands (compute-sanitizer is closed on this pool)
@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
@pytest.mark.parametrize("kernel", ["K2s", "K4s"])
def test_guard_bands_around_every_slice_and_around_theta_state_ema(kernel, dtype):
    """Every (worker, server) slice sits inside its own allocation whose guard bands hold NaN (a USED out-of-bounds read
    would poison the result and fail parity); theta / state / ema sit inside allocations whose bands hold a sentinel (an
    out-of-bounds write would change it).  Ragged servers incl. an empty and a one-element one, odd element offsets (head
    peel, mixed phases), both shard-aware kernels."""
    cfg = replace(BASE, grad_dtype=dtype, opt=synth.RMSPROP_MOM, name=f"guard_{kernel}_d{dtype}")
    off = np.asarray(RAGGED, dtype=np.int64)
    M, P, PAD, SENT = off.size - 1, int(off[-1]), 64, 12345.0
    tdt = torch.float32 if dtype == synth.F32 else torch.bfloat16

    def banded_state(t):
        raw = torch.full((P + 2 * PAD,), SENT, dtype=torch.float32, device=DEV)
        raw[PAD:PAD + P].copy_(t)
        return raw, raw[PAD:PAD + P]

    th_raw, theta = banded_state(synth.init_theta(cfg, DEV))
    s0i, s1i = synth.init_state(cfg, DEV)
    s0_raw, s0 = banded_state(s0i)
    s1_raw, s1 = banded_state(s1i)
    em_raw, ema = banded_state(theta.clone())
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    raws, sl = [], []
    for k, g in enumerate(flat):
        row = []
        for j in range(M):
            lo, hi = int(off[j]), int(off[j + 1])
            o = PAD + (3 * k + 5 * j) % 8
            raw = torch.full((hi - lo + o + PAD,), float("nan"), dtype=tdt, device=DEV)
            raw[o:o + hi - lo].copy_(g[lo:hi])
            raws.append((raw, o, hi - lo))
            row.append(raw[o:o + hi - lo])
        sl.append(row)
    table = psync.make_slice_table(sl)
    d_off = torch.from_numpy(off).to(DEV)
    d_tiles = psync.psync_shard_worklist(d_off, cfg.grad_dtype)
    host = {"theta": to_np(theta), "ema": to_np(ema), "state0": to_np(s0), "state1": to_np(s1)}
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    common = dict(opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
    if kernel == "K2s":
        N, b = 10, 3
        d_kept = torch.full((M, N), -1, dtype=torch.int32, device=DEV)
        d_status = torch.full((M,), -9, dtype=torch.int32, device=DEV)
        st, keep = psync.make_step(off, N, cfg.W, table.grad_dtype, theta, ema, s0, s1, d_grads=table.d_ptrs, d_kept=d_kept,
                                   d_status=d_status, per_shard=True, d_shard_off=d_off,
                                   grad_layout=psync.PSYNC_GRADS_SLICES, d_tile_start=d_tiles, **common)
        psync.psync_step_device(st, torch.from_numpy(a).to(DEV))
        torch.cuda.synchronize()
        status, kept, _ = oracle.select_first_n_sharded(a, N, b)
        assert np.array_equal(d_kept.cpu().numpy(), kept)
        rc = oracle.aggregate_update_slices(off, N, np_slices(sl), kept, host["theta"], host["ema"], host["state0"],
                                            host["state1"], per_shard=True, status=status, **common)
        rtol = RTOL_BF16 if dtype == synth.BF16 else RTOL_STEP
    else:
        d_order = torch.full((M, cfg.W), -1, dtype=torch.int32, device=DEV)
        d_n = torch.zeros(M, dtype=torch.int32, device=DEV)
        st, keep = psync.make_step(off, cfg.W, cfg.W, table.grad_dtype, theta, ema, s0, s1, d_grads=table.d_ptrs,
                                   d_kept=d_order, d_n_kept=d_n, kept_stride=cfg.W, per_shard=True, d_shard_off=d_off,
                                   grad_layout=psync.PSYNC_GRADS_SLICES, d_tile_start=d_tiles, **common)
        psync.psync_async_step_device(st, torch.from_numpy(a).to(DEV))
        torch.cuda.synchronize()
        order = np.stack([oracle.order_by_arrival(a[j]) for j in range(M)])
        rc = oracle.async_apply_rows(off, np_slices(sl), order, host["theta"], host["ema"], host["state0"], host["state1"],
                                     slices=True, per_shard=True, **common)
        rtol = rtol_async(cfg.W)
    assert rc == oracle.OK
    for n, t in (("theta", theta), ("ema", ema), ("state0", s0), ("state1", s1)):
        assert_close(to_np(t), host[n], rtol, ATOL_STEP, f"guard {kernel} {n}")
    for raw in (th_raw, em_raw, s0_raw, s1_raw):
        assert bool((raw[:PAD] == SENT).all()) and bool((raw[PAD + P:] == SENT).all()), "write outside theta / state / ema"
    for raw, o, n in raws:
        assert bool(torch.isnan(raw[:o].float()).all()) and bool(torch.isnan(raw[o + n:].float()).all())
