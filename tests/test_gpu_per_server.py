"""GPU parity for the per-parameter-server step (NEXT-1: Alg. 4 per server j) and the
time-out rule (NEXT-2: PAPER.md:L259) against the CPU oracle, through the C ABI.  Kept rows, counts and
status words are compared bit-exactly; theta / state / ema within north_star's lock-step tolerance."""
from dataclasses import replace

import numpy as np
import pytest
import torch

import oracle
import paper_1702_05800_b200 as psync
from paper_1702_05800_b200 import synth

from _harness import ATOL_STEP, RTOL_STEP, STATE_NAMES, assert_close, to_np

pytestmark = pytest.mark.gpu
DEV = "cuda"

BASE = synth.Config(name="per_server", cfg_id=11, P=70_003, M=7, N=10, b=3, arrival_sigma=0.3, opt=synth.SGD,
                    gamma=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0, steps=3)


class RowsPair:
    """One parameter-server state on the GPU and on the host, stepped with kept ROWS (per server and/or
    variable count) on both sides from the same bytes."""

    def __init__(self, cfg, shard_off=None, misalign=0):
        self.cfg = cfg
        self.off = synth.shard_offsets(cfg) if shard_off is None else np.asarray(shard_off, dtype=np.int64)
        self.M = self.off.size - 1
        self.misalign = misalign

        def place(t):      # optionally put the array at an element offset that breaks 16-byte alignment
            if t is None or not misalign:
                return t
            buf = torch.empty(t.numel() + 8, dtype=t.dtype, device=DEV)
            view = buf[misalign:misalign + t.numel()]
            view.copy_(t)
            return view

        self.theta = place(synth.init_theta(cfg, DEV))
        s0, s1 = synth.init_state(cfg, DEV)
        self.state0, self.state1 = place(s0), place(s1)
        self.ema = place(self.theta.clone()) if cfg.ema_mode != synth.EMA_OFF else None
        self.d_off = torch.from_numpy(self.off).to(DEV)
        self.host = {n: to_np(getattr(self, n)) for n in STATE_NAMES}

    def make_step(self, table, d_kept, d_status, per_shard, d_n_kept=None, kept_stride=0):
        cfg = self.cfg
        return psync.make_step(self.off, cfg.N, cfg.W, table.grad_dtype, self.theta, self.ema, self.state0,
                               self.state1, opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha,
                               mu=cfg.mu, rho=cfg.rho, eps=cfg.eps, d_grads=table.d_ptrs, d_kept=d_kept,
                               d_status=d_status, per_shard=per_shard,
                               kept_stride=kept_stride, d_shard_off=self.d_off if per_shard else None,
                               d_n_kept=d_n_kept)

    def oracle_rows(self, grads, kept, per_shard, n_kept=None, status=None):
        cfg, h = self.cfg, self.host
        rc = oracle.aggregate_update_rows(self.off, cfg.N, [synth.as_numpy_grad(g) for g in grads], kept, h["theta"],
                                          h["ema"], h["state0"], h["state1"], per_shard=per_shard, n_kept=n_kept,
                                          status=status, opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma,
                                          alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
        assert rc == oracle.OK

    def compare_and_sync(self, what):
        for n in STATE_NAMES:
            g = getattr(self, n)
            if g is not None:
                assert_close(to_np(g), self.host[n], RTOL_STEP, ATOL_STEP, f"{what} {n}")
                self.host[n] = to_np(g)

    # ---- one per-server first-N step on both sides ------------------------------------------------
    def step_first_n(self, step, arrival, tags=None, t=0):
        cfg = self.cfg
        grads = [synth.gradient(cfg, step, k, DEV) for k in range(cfg.W)]
        table = psync.make_grad_table(grads)
        d_kept = torch.full((self.M, cfg.N), -1, dtype=torch.int32, device=DEV)
        d_status = torch.full((self.M,), -9, dtype=torch.int32, device=DEV)
        d_tn = torch.full((self.M,), float("nan"), dtype=torch.float32, device=DEV)
        d_tags = None if tags is None else torch.from_numpy(tags).to(DEV)
        psync.psync_select_first_n_sharded(torch.from_numpy(arrival).to(DEV), cfg.N, cfg.b, self.M, d_kept, d_status,
                                           d_tn, d_tags, t)
        st, keep = self.make_step(table, d_kept, d_status, per_shard=True)
        psync.psync_aggregate_update(st)
        torch.cuda.synchronize()
        status, kept, t_nth = oracle.select_first_n_sharded(arrival, cfg.N, cfg.b, tags=tags, t=t)
        assert np.array_equal(d_status.cpu().numpy(), status)
        assert np.array_equal(d_kept.cpu().numpy(), kept)            # failed rows untouched (-1) on both sides
        assert np.array_equal(d_tn.cpu().numpy(), t_nth, equal_nan=True)
        self.oracle_rows(grads, kept, True, status=status)
        self.compare_and_sync(f"{cfg.name} step {step}")
        return status, kept


def per_server_cfg(**kw):
    return replace(BASE, **kw)


# ------------------------------------------------------------------ per-server selection kernel
@pytest.mark.parametrize("seed", range(4))
def test_select_sharded_random_rows_ties_nonfinite_tags(seed):
    rng = np.random.default_rng(900 + seed)
    M = int(rng.integers(1, 300))
    N, b = int(rng.integers(1, 120)), int(rng.integers(0, 20))
    W = N + b
    a = rng.lognormal(0, 0.3, (M, W)).astype(np.float32)
    ties = rng.random((M, W)) < 0.3
    a[ties] = rng.choice(np.array([0.5, 1.0, 1.0, 2.0, -0.0, 0.0], np.float32), size=int(ties.sum()))
    a[rng.random((M, W)) < 0.05] = np.inf
    a[rng.random((M, W)) < 0.03] = np.nan
    if M > 2:
        a[1, :] = np.inf                                   # a server nobody reaches
    tags = np.where(rng.random((M, W)) < 0.1, 4, 5).astype(np.int32)
    for tg in (None, tags):
        d_kept = torch.full((M, N), -1, dtype=torch.int32, device=DEV)
        d_status = torch.full((M,), -9, dtype=torch.int32, device=DEV)
        d_tn = torch.full((M,), float("nan"), dtype=torch.float32, device=DEV)
        psync.psync_select_first_n_sharded(torch.from_numpy(a).to(DEV), N, b, M, d_kept, d_status, d_tn,
                                           None if tg is None else torch.from_numpy(tg).to(DEV), 5)
        status, kept, t_nth = oracle.select_first_n_sharded(a, N, b, tags=tg, t=5)
        assert np.array_equal(d_status.cpu().numpy(), status)
        assert np.array_equal(d_kept.cpu().numpy(), kept)
        assert np.array_equal(d_tn.cpu().numpy(), t_nth, equal_nan=True)


def test_select_sharded_max_workers_many_servers():
    rng = np.random.default_rng(77)
    M, N, b = 64, 1000, 24
    a = rng.lognormal(0, 0.3, (M, N + b)).astype(np.float32)
    d_kept = torch.full((M, N), -1, dtype=torch.int32, device=DEV)
    d_status = torch.full((M,), -9, dtype=torch.int32, device=DEV)
    psync.psync_select_first_n_sharded(torch.from_numpy(a).to(DEV), N, b, M, d_kept, d_status)
    status, kept, _ = oracle.select_first_n_sharded(a, N, b)
    assert (status == 0).all() and np.array_equal(d_status.cpu().numpy(), status)
    assert np.array_equal(d_kept.cpu().numpy(), kept)


# ------------------------------------------------------------------ per-server fused step
@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
@pytest.mark.parametrize("opt", [synth.SGD, synth.MOMENTUM, synth.RMSPROP_MOM])
@pytest.mark.parametrize("ema_mode", [synth.EMA_POST, synth.EMA_PRE, synth.EMA_OFF])
def test_per_server_every_template_instance_lockstep(dtype, opt, ema_mode):
    cfg = per_server_cfg(grad_dtype=dtype, opt=opt, ema_mode=ema_mode, name=f"ps_d{dtype}_o{opt}_e{ema_mode}")
    pair = RowsPair(cfg)
    for s in range(2):
        status, kept = pair.step_first_n(s, synth.arrival_times_per_server(cfg, s, server_sigma=0.3))
        assert (status == 0).all() and len({tuple(r) for r in kept.tolist()}) > 1   # servers keep different sets


@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
def test_per_server_awkward_shard_cuts(dtype):
    """Empty servers, servers shorter than one 16-byte unit, cuts at every alignment phase, a cut inside the
    last partial unit, tiles that straddle several servers."""
    P = 20_000 + 5
    off = [0, 0, 1, 3, 3, 10, 1023, 1024, 1029, 2048, 2049, 2049, 7000, 7001, 7002, 7003, 7011, 16_384, 20_001, P]
    cfg = per_server_cfg(P=P, M=len(off) - 1, grad_dtype=dtype, opt=synth.RMSPROP_MOM, N=9, b=4, name="ps_awkward")
    pair = RowsPair(cfg, shard_off=off)
    for s in range(2):
        pair.step_first_n(s, synth.arrival_times_per_server(cfg, s, server_sigma=0.3))


@pytest.mark.parametrize("P", [1, 3, 5, 8, 9, 1024, 1025])
def test_per_server_small_P(P):
    cfg = per_server_cfg(P=P, M=min(P, 3), opt=synth.MOMENTUM, ragged=False, name=f"ps_small{P}")
    RowsPair(cfg).step_first_n(0, synth.arrival_times_per_server(cfg, 0, server_sigma=0.3))


def test_per_server_failed_servers_untouched_others_update():
    cfg = per_server_cfg(opt=synth.RMSPROP_MOM, P=50_001, name="ps_failed")
    pair = RowsPair(cfg)
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    a[2, :5] = np.inf                      # server 2 sees only 8 < N = 10 workers
    a[5, :] = np.nan                       # server 5 sees nobody
    before = {n: to_np(getattr(pair, n)) for n in STATE_NAMES}
    status, kept = pair.step_first_n(0, a)
    assert status.tolist() == [0, 0, oracle.ETOOFEW, 0, 0, oracle.ETOOFEW, 0]
    for j in (2, 5):
        lo, hi = pair.off[j], pair.off[j + 1]
        for n in STATE_NAMES:              # bit-for-bit untouched
            assert np.array_equal(to_np(getattr(pair, n))[lo:hi], before[n][lo:hi])
    lo, hi = pair.off[3], pair.off[4]
    assert not np.array_equal(to_np(pair.theta)[lo:hi], before["theta"][lo:hi])


def test_per_server_stale_tags_per_row():
    cfg = per_server_cfg(P=30_000, name="ps_tags")
    pair = RowsPair(cfg)
    rng = np.random.default_rng(5)
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    tags = np.where(rng.random(a.shape) < 0.15, 2, 3).astype(np.int32)     # some late gradients of step 2
    pair.step_first_n(0, a, tags=tags, t=3)


@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
def test_per_server_unaligned_state_takes_the_scalar_path(dtype):
    cfg = per_server_cfg(P=9_001, grad_dtype=dtype, opt=synth.RMSPROP_MOM, name="ps_unaligned")
    pair = RowsPair(cfg, misalign=1)
    pair.step_first_n(0, synth.arrival_times_per_server(cfg, 0, server_sigma=0.3))


def test_identical_rows_are_bit_identical_to_the_single_kept_set_kernel():
    """Property at any size: when every server sees the same arrival times the per-server kernel must
    reproduce the shared-kept-set kernel bit for bit (same adds in the same order)."""
    cfg = per_server_cfg(P=1_000_003, M=20, N=50, b=5, opt=synth.RMSPROP_MOM, name="ps_same")
    row = synth.arrival_times(cfg, 0)
    grads = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    table = psync.make_grad_table(grads)
    out = []
    for per_shard in (True, False):
        pair = RowsPair(cfg)
        rows = pair.M if per_shard else 1
        d_kept = torch.full((rows, cfg.N), -1, dtype=torch.int32, device=DEV)
        d_status = torch.full((rows,), -9, dtype=torch.int32, device=DEV)
        a = np.tile(row, (rows, 1))
        psync.psync_select_first_n_sharded(torch.from_numpy(a).to(DEV), cfg.N, cfg.b, rows, d_kept, d_status)
        st, keep = pair.make_step(table, d_kept, d_status, per_shard=per_shard)
        psync.psync_aggregate_update(st)
        torch.cuda.synchronize()
        out.append({n: to_np(getattr(pair, n)) for n in STATE_NAMES})
    for n in STATE_NAMES:
        assert np.array_equal(out[0][n], out[1][n]), n


def test_per_server_poison_and_null_for_dropped_slices():
    """A worker dropped by server j may hold NaN in slice j; a worker dropped by EVERY server may be NULL."""
    cfg = per_server_cfg(P=40_000, M=5, N=6, b=3, name="ps_poison")
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    a[:, 4] = 99.0                                                       # worker 4 is last everywhere
    grads = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    status, kept, _ = oracle.select_first_n_sharded(a, cfg.N, cfg.b)
    off = synth.shard_offsets(cfg)
    results = []
    for poisoned in (False, True):
        gs = [g.clone() for g in grads]
        if poisoned:
            for j in range(cfg.M):
                for k in set(range(cfg.W)) - set(kept[j].tolist()):
                    gs[k][off[j]:off[j + 1]] = float("nan")
        table = psync.make_grad_table(gs)
        if poisoned:
            table.d_ptrs[4] = 0                                          # never dereferenced
        pair = RowsPair(cfg)
        d_kept = torch.full((cfg.M, cfg.N), -1, dtype=torch.int32, device=DEV)
        d_status = torch.full((cfg.M,), -9, dtype=torch.int32, device=DEV)
        psync.psync_select_first_n_sharded(torch.from_numpy(a).to(DEV), cfg.N, cfg.b, cfg.M, d_kept, d_status)
        st, keep = pair.make_step(table, d_kept, d_status, per_shard=True)
        psync.psync_aggregate_update(st)
        torch.cuda.synchronize()
        results.append(to_np(pair.theta))
    assert np.isfinite(results[1]).all() and np.array_equal(results[0], results[1])


# ------------------------------------------------------------------ time-out rule
def _timeout_gpu(a, timeout, rows, W, min_keep=1, tags=None, t=0):
    d_kept = torch.full((rows, W), -1, dtype=torch.int32, device=DEV)
    d_n = torch.full((rows,), -7, dtype=torch.int32, device=DEV)
    d_status = torch.full((rows,), -9, dtype=torch.int32, device=DEV)
    psync.psync_select_timeout(torch.from_numpy(a).to(DEV), W, timeout, d_kept, d_n, d_status, rows=rows,
                               min_keep=min_keep, d_step_tag=None if tags is None else torch.from_numpy(tags).to(DEV),
                               t=t)
    return d_kept, d_n, d_status


@pytest.mark.parametrize("seed", range(4))
def test_select_timeout_matches_oracle(seed):
    rng = np.random.default_rng(1200 + seed)
    rows, W = int(rng.integers(1, 40)), int(rng.choice([1, 5, 31, 32, 33, 106, 700, 1024]))
    a = rng.lognormal(0, 0.4, (rows, W)).astype(np.float32)
    a[rng.random((rows, W)) < 0.05] = np.inf
    a[rng.random((rows, W)) < 0.03] = np.nan
    a[rng.random((rows, W)) < 0.03] = -np.inf
    tags = np.where(rng.random((rows, W)) < 0.1, 0, 1).astype(np.int32)
    for timeout, min_keep in ((1.0, 1), (float(a[0, 0]) if np.isfinite(a[0, 0]) else 0.9, 1), (float("inf"), 1),
                              (0.01, 1), (1.2, max(1, W // 2))):
        for tg in (None, tags):
            d_kept, d_n, d_status = _timeout_gpu(a, timeout, rows, W, min_keep, tg, 1)
            kept_g, n_g, st_g = d_kept.cpu().numpy(), d_n.cpu().numpy(), d_status.cpu().numpy()
            for r in range(rows):
                st, kept = oracle.select_timeout(a[r], timeout, min_keep, tags=None if tg is None else tg[r], t=1)
                assert st_g[r] == st
                if st == oracle.OK:
                    assert n_g[r] == kept.size and np.array_equal(kept_g[r, :kept.size], kept)
                    assert (kept_g[r, kept.size:] == -1).all()
                else:
                    assert n_g[r] == 0 and (kept_g[r] == -1).all()       # the count is zeroed, the row is not written


@pytest.mark.parametrize("per_shard", [False, True])
@pytest.mark.parametrize("dtype,opt", [(synth.F32, synth.RMSPROP_MOM), (synth.BF16, synth.MOMENTUM),
                                       (synth.F32, synth.SGD)])
def test_timeout_step_divides_by_the_number_kept(per_shard, dtype, opt):
    cfg = per_server_cfg(grad_dtype=dtype, opt=opt, N=1, b=22, P=60_007, name=f"timeout_ps{int(per_shard)}")
    pair = RowsPair(cfg)
    W, rows = cfg.W, (pair.M if per_shard else 1)
    for s, timeout in enumerate((1.0, 1.3, 0.8)):
        a = synth.arrival_times_per_server(cfg, s, server_sigma=0.3)[:rows].copy()
        if per_shard and s == 1:
            a[3, :] = 50.0                                               # server 3 times out with nobody
        grads = [synth.gradient(cfg, s, k, DEV) for k in range(W)]
        table = psync.make_grad_table(grads)
        d_kept, d_n, d_status = _timeout_gpu(a, timeout, rows, W)
        st, keep = pair.make_step(table, d_kept, d_status, per_shard=per_shard, d_n_kept=d_n)
        psync.psync_aggregate_update(st)
        torch.cuda.synchronize()
        kept = np.full((rows, W), -1, np.int32)
        n_kept = np.ones(rows, np.int32)
        status = np.zeros(rows, np.int32)
        for r in range(rows):
            status[r], k = oracle.select_timeout(a[r], timeout)
            if status[r] == oracle.OK:
                kept[r, :k.size], n_kept[r] = k, k.size
        assert np.array_equal(d_status.cpu().numpy(), status)
        ok = status == 0
        assert np.array_equal(d_n.cpu().numpy()[ok], n_kept[ok]) and len(set(n_kept[ok].tolist())) >= 1
        pair.oracle_rows(grads, kept, per_shard, n_kept=n_kept, status=status)
        pair.compare_and_sync(f"{cfg.name} step {s} timeout {timeout}")


def test_timeout_infinite_equals_first_n_with_b0_bitwise():
    """timeout = +inf keeps all W arrived workers: the same adds in the same order as N = W, b = 0."""
    cfg = per_server_cfg(N=16, b=0, P=200_003, opt=synth.MOMENTUM, name="timeout_inf")
    a = synth.arrival_times(cfg, 0)
    grads = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    table = psync.make_grad_table(grads)
    out = []
    for use_timeout in (True, False):
        pair = RowsPair(cfg)
        if use_timeout:
            d_kept, d_n, d_status = _timeout_gpu(a.reshape(1, -1), float("inf"), 1, cfg.W)
            st, keep = pair.make_step(table, d_kept, d_status, per_shard=False, d_n_kept=d_n)
        else:
            d_kept = torch.full((cfg.N,), -1, dtype=torch.int32, device=DEV)
            d_status = torch.full((1,), -9, dtype=torch.int32, device=DEV)
            psync.psync_select_first_n(torch.from_numpy(a).to(DEV), cfg.N, cfg.b, d_kept, d_status)
            st, keep = pair.make_step(table, d_kept, d_status, per_shard=False)
        psync.psync_aggregate_update(st)
        torch.cuda.synchronize()
        out.append({n: to_np(getattr(pair, n)) for n in STATE_NAMES})
    for n in STATE_NAMES:
        if out[0][n] is not None:
            assert np.array_equal(out[0][n], out[1][n]), n


# ------------------------------------------------------------------ full size (bench launch configuration)
def test_full_size_cfg3_per_server_sampled():
    """cfg3 at full size with one kept row per server: sampled elements (every shard cut, the first and last
    tiles, random interior) against the oracle run on the gathered columns."""
    cfg = synth.PAPER_RMSPROP
    free, _ = torch.cuda.mem_get_info()
    if cfg.footprint_bytes * 1.15 > free:
        pytest.skip("not enough free HBM for the full-size config")
    pair = RowsPair(cfg)
    rng = np.random.default_rng(33)
    cuts = pair.off[1:-1]
    idx = np.unique(np.concatenate([np.arange(0, 4096), np.arange(cfg.P - 4096, cfg.P),
                                    *[np.arange(c - 1100, c + 1100) for c in cuts],      # the straddling tiles
                                    rng.integers(0, cfg.P, 30_000)])).astype(np.int64)
    d_idx = torch.from_numpy(idx).to(DEV)
    off_s = np.searchsorted(idx, pair.off).astype(np.int64)              # the same cuts in the gathered space
    host = {n: to_np(getattr(pair, n)[d_idx]) for n in STATE_NAMES}
    grads = [torch.empty(cfg.P, dtype=torch.float32, device=DEV) for _ in range(cfg.W)]
    table = psync.make_grad_table(grads)
    d_kept = torch.full((pair.M, cfg.N), -1, dtype=torch.int32, device=DEV)
    d_status = torch.full((pair.M,), -9, dtype=torch.int32, device=DEV)
    st, keep = pair.make_step(table, d_kept, d_status, per_shard=True)
    for s in range(2):
        for k in range(cfg.W):
            synth.gradient(cfg, s, k, DEV, out=grads[k])
        a = synth.arrival_times_per_server(cfg, s)
        psync.psync_select_first_n_sharded(torch.from_numpy(a).to(DEV), cfg.N, cfg.b, pair.M, d_kept, d_status)
        psync.psync_aggregate_update(st)
        torch.cuda.synchronize()
        status, kept, _ = oracle.select_first_n_sharded(a, cfg.N, cfg.b)
        assert (status == 0).all() and np.array_equal(d_kept.cpu().numpy(), kept)
        assert len({tuple(r) for r in kept.tolist()}) > 1
        rc = oracle.aggregate_update_rows(off_s, cfg.N, [synth.as_numpy_grad(g[d_idx]) for g in grads], kept,
                                          host["theta"], host["ema"], host["state0"], host["state1"], per_shard=True,
                                          status=status, opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma,
                                          alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho, eps=cfg.eps)
        assert rc == oracle.OK
        for n in STATE_NAMES:
            got = to_np(getattr(pair, n)[d_idx])
            assert_close(got, host[n], RTOL_STEP, ATOL_STEP, f"cfg3 per-server step {s} {n} (sampled)")
            host[n] = got
        assert bool(torch.isfinite(pair.theta).all())


def test_per_server_many_tiny_servers_every_tile_straddles():
    """M = 1000 servers of ~100 parameters: every 1024-parameter tile spans ~10 servers, so the whole vector goes
    through the element-wise path, each element with its own server's kept row."""
    cfg = per_server_cfg(P=100_003, M=1000, N=5, b=2, opt=synth.RMSPROP_MOM, name="ps_tiny_servers")
    pair = RowsPair(cfg)
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    a[::7, :4] = np.inf                       # every 7th server fails (3 < N eligible)
    status, kept = pair.step_first_n(0, a)
    assert (status[::7] == oracle.ETOOFEW).all() and (np.delete(status, np.s_[::7]) == 0).all()


def test_flat_rows_kernel_status_null_zero_count_and_garbage_count_are_failed_rows():
    """The flat-index rows kernel (no work list) with status = NULL: a row whose time-out selection failed carries a
    zero count and is skipped; a count nobody wrote (out of range) is skipped too -- never a loop over a stale count, a
    wild pointer or 0 * inf = NaN in theta."""
    cfg = per_server_cfg(opt=synth.RMSPROP_MOM, P=50_003, name="rows_null_status")
    pair = RowsPair(cfg)
    W, M = cfg.W, pair.M
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    a[3, :] = 9.0
    d_kept, d_n, d_status = _timeout_gpu(a, 1.1, M, W)
    torch.cuda.synchronize()
    assert int(d_status[3].item()) == oracle.ETOOFEW and int(d_n[3].item()) == 0
    d_n[5] = 1_000_000                                             # garbage
    grads = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    table = psync.make_grad_table(grads)
    st, keep = pair.make_step(table, d_kept, None, per_shard=True, d_n_kept=d_n)
    st.d_status = None
    psync.psync_aggregate_update(st)
    torch.cuda.synchronize()
    kept = np.full((M, W), -1, np.int32)
    n_kept = np.ones(M, np.int32)
    status = np.zeros(M, np.int32)
    for r in range(M):
        status[r], k = oracle.select_timeout(a[r], 1.1)
        if status[r] == oracle.OK:
            kept[r, :k.size], n_kept[r] = k, k.size
    status[5] = oracle.ETOOFEW                                     # the garbage row must behave like a failed one
    pair.oracle_rows(grads, kept, True, n_kept=n_kept, status=status)
    pair.compare_and_sync("rows kernel, status NULL")
    assert bool(torch.isfinite(pair.theta).all())


@pytest.mark.parametrize("per_server,slices", [(False, False), (True, False), (True, True)])
def test_parameter_server_step_timeout_rule(per_server, slices):
    """ParameterServerStep.step_timeout: the time-out rule (L259) through the plumbing object -- flat buffers or slices, one
    kept set or one per server -- against the oracle over three chained steps with different time-outs."""
    cfg = per_server_cfg(N=1, b=22, P=60_007, opt=synth.MOMENTUM, name=f"ps_timeout_{int(per_server)}{int(slices)}")
    off = synth.shard_offsets(cfg)
    M, W = off.size - 1, cfg.W
    theta = synth.init_theta(cfg, DEV)
    s0, _ = synth.init_state(cfg, DEV)
    ema = theta.clone()
    ps = psync.ParameterServerStep(off, cfg.N, cfg.b, theta, ema, s0, None, cfg.opt, cfg.ema_mode, alpha=cfg.alpha, mu=cfg.mu,
                                   per_server=per_server)
    host = {"theta": to_np(theta), "ema": to_np(ema), "state0": to_np(s0)}
    rows = M if per_server else 1
    for s, timeout in enumerate((1.0, 1.3, 0.8)):
        a = synth.arrival_times_per_server(cfg, s, server_sigma=0.3)[:rows].copy()
        grads = [synth.gradient(cfg, s, k, DEV) for k in range(W)]
        if slices:
            sl = [[g[int(off[j]):int(off[j + 1])].clone() for j in range(M)] for g in grads]
            ps.set_gradient_slices(sl)
        else:
            ps.set_gradients(grads)
        ps.step_timeout(torch.from_numpy(a if per_server else a[0]).to(DEV), timeout, cfg.gamma)
        torch.cuda.synchronize()
        kept = np.full((rows, W), -1, np.int32)
        n_kept = np.ones(rows, np.int32)
        status = np.zeros(rows, np.int32)
        for r in range(rows):
            status[r], k = oracle.select_timeout(a[r], timeout)
            if status[r] == oracle.OK:
                kept[r, :k.size], n_kept[r] = k, k.size
        assert np.array_equal(ps.d_status.cpu().numpy(), status)
        np_grads = [synth.as_numpy_grad(g) for g in grads]
        rc = oracle.aggregate_update_rows(off, cfg.N, np_grads, kept, host["theta"], host["ema"], host["state0"], None,
                                          per_shard=per_server, n_kept=n_kept, status=status, opt=cfg.opt,
                                          ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu)
        assert rc == oracle.OK
        for n, t in (("theta", theta), ("ema", ema), ("state0", s0)):
            assert_close(to_np(t), host[n], RTOL_STEP, ATOL_STEP, f"ps timeout step {s} {n}")
            host[n] = to_np(t)
