"""Pins for the oracle's per-parameter-server step (NEXT-1: Alg. 4 literally per server j)
and the time-out rule (NEXT-2: PAPER.md:L259, reading R19).

Expected values come from a hand-worked example (tests/golden/hand_worked_per_server.json), numpy's
lexsort / boolean masks / float64 mean, exact rational arithmetic, and reductions to the already pinned
single-kept-set step -- never from re-calling the function under test.
"""
import json
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from test_oracle_select import lexsort_first_n
from test_oracle_update import F, _round_f32, coeffs, f32, ulp_diff

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hand_worked_per_server.json")


def _load():
    with open(GOLDEN) as fh:
        return json.load(fh)


def _arr(x, dt=np.float32):
    return np.array([[float(v) for v in r] for r in x] if isinstance(x[0], list) else [float(v) for v in x], dtype=dt)


# ------------------------------------------------------------------ hand-worked (golden)
def test_golden_per_server_kept_sets_and_update():
    g = _load()["per_server"]
    arrival = _arr(g["arrival"])
    status, kept, t_nth = oracle.select_first_n_sharded(arrival, g["N"], g["b"])
    assert status.tolist() == [0, 0]
    assert kept.tolist() == g["kept"] and t_nth.tolist() == g["t_nth"]
    theta, ema = _arr(g["theta"]), _arr(g["ema"])
    grads = [_arr(x) for x in g["grads"]]
    rc = oracle.aggregate_update_rows(g["shard_off"], g["N"], grads, kept, theta, ema, per_shard=True, status=status,
                                      gamma_t=g["gamma"], alpha=g["alpha"])
    assert rc == oracle.OK
    assert theta.tolist() == g["theta_out"] and ema.tolist() == g["ema_post"]


def test_golden_failed_server_is_left_untouched_others_update():
    g = _load()["per_server"]
    arrival = _arr(g["failed_arrival"])
    status, kept, t_nth = oracle.select_first_n_sharded(arrival, g["N"], g["b"])
    assert status.tolist() == g["failed_status"]
    assert kept[1].tolist() == [-1, -1] and np.isnan(t_nth[1])          # failed row not written
    theta, ema = _arr(g["theta"]), _arr(g["ema"])
    grads = [_arr(x) for x in g["grads"]]
    rc = oracle.aggregate_update_rows(g["shard_off"], g["N"], grads, kept, theta, ema, per_shard=True, status=status,
                                      gamma_t=g["gamma"], alpha=g["alpha"])
    assert rc == oracle.OK
    assert theta.tolist() == g["failed_theta_out"] and ema.tolist() == g["failed_ema_post"]


def test_golden_timeout():
    g = _load()["timeout"]
    arrival = _arr(g["arrival"])
    st, kept = oracle.select_timeout(arrival, g["timeout"])
    assert st == oracle.OK and kept.tolist() == g["kept"]
    grads = [_arr(x) for x in g["grads"]]
    W = len(grads)
    rows = np.full((1, W), -1, np.int32)
    rows[0, :len(kept)] = kept
    theta = _arr(g["theta"])
    rc = oracle.aggregate_update_rows([0, 1, 2], W, grads, rows, theta, per_shard=False,
                                      n_kept=np.array([len(kept)], np.int32), ema_mode=oracle.EMA_OFF,
                                      gamma_t=g["gamma"])
    assert rc == oracle.OK
    assert np.abs(theta - _arr(g["theta_out_approx"])).max() <= 1e-7     # fl32(1/3) is not 1/3 (error 3e-8 rel.)
    # the exact (power-of-two count) variant
    st, kept = oracle.select_timeout(arrival, g["timeout_exact"])
    assert st == oracle.OK and kept.tolist() == g["kept_exact"]
    rows[:] = -1
    rows[0, :2] = kept
    theta = _arr(g["theta"])
    oracle.aggregate_update_rows([0, 2], W, grads, rows, theta, per_shard=False, n_kept=np.array([2], np.int32),
                                 ema_mode=oracle.EMA_OFF, gamma_t=g["gamma"])
    assert theta.tolist() == g["theta_out_exact"]
    # nobody in time / fewer than min_keep
    assert oracle.select_timeout(arrival, 0.25)[0] == oracle.ETOOFEW
    assert oracle.select_timeout(arrival, 1.0, min_keep=3)[0] == oracle.ETOOFEW
    assert oracle.select_timeout(arrival, 1.0, min_keep=2)[0] == oracle.OK


# ------------------------------------------------------------------ per-server selection vs numpy lexsort
@pytest.mark.parametrize("seed", range(6))
def test_per_server_rows_match_numpy_lexsort(seed):
    rng = np.random.default_rng(500 + seed)
    M, N, b = int(rng.integers(1, 9)), int(rng.integers(1, 12)), int(rng.integers(0, 5))
    W = N + b
    arrival = rng.choice(np.array([0.25, 0.5, 1.0, 1.5, 2.0, -1.0, -0.0, 0.0], np.float32), size=(M, W))
    arrival = np.where(rng.random((M, W)) < 0.5, rng.lognormal(0, 0.3, (M, W)), arrival).astype(np.float32)
    arrival[rng.random((M, W)) < 0.1] = np.float32("inf")
    arrival[rng.random((M, W)) < 0.05] = np.float32("nan")
    tags = np.where(rng.random((M, W)) < 0.15, 6, 7).astype(np.int32)
    for use_tags in (False, True):
        status, kept, t_nth = oracle.select_first_n_sharded(arrival, N, b, tags=tags if use_tags else None, t=7)
        for j in range(M):
            want, want_t = lexsort_first_n(arrival[j], N, tags[j] if use_tags else None, 7)
            if want is None:
                assert status[j] == oracle.ETOOFEW and (kept[j] == -1).all() and np.isnan(t_nth[j])
            else:
                assert status[j] == oracle.OK and kept[j].tolist() == want.tolist()
                assert float(t_nth[j]) == want_t or (want_t == 0.0 and float(t_nth[j]) == 0.0)


def test_per_server_rows_are_independent():
    """Changing server j's arrival row changes only row j of the outputs."""
    rng = np.random.default_rng(3)
    M, N, b = 5, 6, 3
    a = rng.lognormal(0, 0.3, (M, N + b)).astype(np.float32)
    s0, k0, t0 = oracle.select_first_n_sharded(a, N, b)
    a2 = a.copy()
    a2[2] = a2[2][::-1]
    s1, k1, t1 = oracle.select_first_n_sharded(a2, N, b)
    for j in (0, 1, 3, 4):
        assert k0[j].tolist() == k1[j].tolist() and t0[j] == t1[j]
    assert sorted((N + b - 1 - k0[2]).tolist()) == k1[2].tolist()


# ------------------------------------------------------------------ per-server update
def _case(rng, P, W, bf16=False):
    theta = rng.normal(0, 0.02, P).astype(f32)
    g = [rng.normal(0, 1e-3, P).astype(f32) for _ in range(W)]
    if bf16:
        g = [(x.view(np.uint32) >> 16).astype(np.uint16) for x in g]
    return theta, g


def _vals(g):
    return (g.astype(np.uint32) << 16).view(np.float32) if g.dtype == np.uint16 else g


@pytest.mark.parametrize("bf16", [False, True])
def test_per_server_sgd_against_numpy_float64_mean_per_slice(bf16):
    """Independent library statement: for each server j, theta[j] - gamma * mean over kept_j of G[j] (numpy, fp64)."""
    rng = np.random.default_rng(41 + bf16)
    P, M, N, b = 997, 6, 8, 3            # N a power of two: fl32(1/N) is exactly 1/N
    W = N + b
    off = np.array([0, 100, 100, 333, 640, 900, P])
    theta, grads = _case(rng, P, W, bf16)
    arrival = rng.lognormal(0, 0.3, (M, W)).astype(f32)
    status, kept, _ = oracle.select_first_n_sharded(arrival, N, b)
    assert len({tuple(r) for r in kept.tolist()}) > 1        # the servers really keep different sets
    th = theta.copy()
    rc = oracle.aggregate_update_rows(off, N, grads, kept, th, per_shard=True, status=status,
                                      ema_mode=oracle.EMA_OFF, gamma_t=0.125)
    assert rc == oracle.OK
    G = np.stack([_vals(g) for g in grads]).astype(np.float64)
    want = theta.astype(np.float64)
    for j in range(M):
        lo, hi = off[j], off[j + 1]
        want[lo:hi] -= 0.125 * G[kept[j], lo:hi].mean(axis=0)
    assert ulp_diff(th, want.astype(f32)).max() <= 1


def test_identical_rows_reduce_to_the_single_kept_set_step():
    """All servers seeing the same arrival times is the shared-kept-set step of reading R11 (already pinned)."""
    rng = np.random.default_rng(43)
    P, M, N, b = 513, 4, 7, 2
    W = N + b
    off = [0, 17, 300, 301, P]
    theta, grads = _case(rng, P, W)
    row = rng.lognormal(0, 0.3, W).astype(f32)
    status, kept, _ = oracle.select_first_n_sharded(np.tile(row, (M, 1)), N, b)
    st1, kept1, _ = oracle.select_first_n(row, N, b)
    assert all(kept[j].tolist() == kept1.tolist() for j in range(M))
    hp = dict(opt=oracle.RMSPROP_MOM, ema_mode=oracle.EMA_POST, gamma_t=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0)
    a = [theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)]
    c = [x.copy() for x in a]
    assert oracle.aggregate_update_rows(off, N, grads, kept, *a, per_shard=True, status=status, **hp) == oracle.OK
    assert oracle.aggregate_update(off, N, grads, kept1, *c, **hp) == oracle.OK
    for x, y in zip(a, c):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("opt", [oracle.SGD, oracle.MOMENTUM])
def test_per_server_exact_rational_brute_force(opt):
    """P <= 64, different kept rows and a failed server: exact Fractions on the exact fp32 inputs."""
    rng = np.random.default_rng(47 + opt)
    P, M, N, b = 48, 4, 5, 2
    W = N + b
    off = [0, 11, 11, 30, P]
    theta, grads = _case(rng, P, W)
    ema = (theta + rng.normal(0, 1e-3, P)).astype(f32)
    v = rng.normal(0, 1e-3, P).astype(f32)
    arrival = rng.lognormal(0, 0.3, (M, W)).astype(f32)
    arrival[3, :4] = np.inf                                   # server 3 sees only 3 < N workers
    status, kept, _ = oracle.select_first_n_sharded(arrival, N, b)
    assert status.tolist() == [0, 0, 0, oracle.ETOOFEW]
    gamma, alpha, mu = 0.045, 0.9999, 0.9
    th, em, vv = theta.copy(), ema.copy(), v.copy()
    rc = oracle.aggregate_update_rows(off, N, grads, kept, th, em, vv if opt == oracle.MOMENTUM else None,
                                      per_shard=True, status=status, opt=opt, gamma_t=gamma, alpha=alpha, mu=mu)
    assert rc == oracle.OK
    inv_N, oma, _ = coeffs(N, alpha)
    for j in range(M):
        for i in range(off[j], off[j + 1]):
            if status[j] != 0:
                assert th[i] == theta[i] and em[i] == ema[i] and vv[i] == v[i]
                continue
            G = sum((F(grads[k][i]) for k in kept[j]), Fraction(0)) * inv_N
            if opt == oracle.SGD:
                t_new = F(theta[i]) - F(f32(gamma)) * G
            else:
                v_new = F(f32(mu)) * F(v[i]) + G
                assert ulp_diff(vv[i], _round_f32(v_new)) <= 1
                t_new = F(theta[i]) - F(f32(gamma)) * v_new
            t_f = _round_f32(t_new)
            assert ulp_diff(th[i], t_f) <= 1
            e_new = F(f32(alpha)) * F(ema[i]) + oma * F(th[i])
            assert ulp_diff(em[i], _round_f32(e_new)) <= 1


def test_per_server_poison_dropped_buffers_per_slice():
    """A worker dropped by server j may hold NaN in slice j (and only there) without any effect."""
    rng = np.random.default_rng(53)
    P, M, N, b = 256, 3, 4, 2
    W = N + b
    off = [0, 80, 200, P]
    theta, grads = _case(rng, P, W)
    arrival = rng.lognormal(0, 0.3, (M, W)).astype(f32)
    status, kept, _ = oracle.select_first_n_sharded(arrival, N, b)
    clean = theta.copy()
    oracle.aggregate_update_rows(off, N, grads, kept, clean, per_shard=True, ema_mode=oracle.EMA_OFF, gamma_t=0.1)
    poisoned = [g.copy() for g in grads]
    for j in range(M):
        for k in set(range(W)) - set(kept[j].tolist()):
            poisoned[k][off[j]:off[j + 1]] = np.nan
    th = theta.copy()
    oracle.aggregate_update_rows(off, N, poisoned, kept, th, per_shard=True, ema_mode=oracle.EMA_OFF, gamma_t=0.1)
    assert np.array_equal(th, clean)


# ------------------------------------------------------------------ time-out rule
@pytest.mark.parametrize("seed", range(5))
def test_timeout_matches_numpy_mask(seed):
    rng = np.random.default_rng(700 + seed)
    W = int(rng.integers(1, 40))
    a = rng.lognormal(0, 0.4, W).astype(f32)
    a[rng.random(W) < 0.1] = np.inf
    a[rng.random(W) < 0.05] = np.nan
    a[rng.random(W) < 0.05] = -np.inf
    tags = np.where(rng.random(W) < 0.2, 1, 2).astype(np.int32)
    for tau in (f32(0.5), f32(1.0), a[0] if np.isfinite(a[0]) else f32(1.25), f32(np.inf), f32(-1.0)):
        for tg in (None, tags):
            mask = np.isfinite(a) & (a <= tau)
            if tg is not None:
                mask &= (tg == 2)
            st, kept = oracle.select_timeout(a, float(tau), tags=tg, t=2)
            if mask.sum() == 0:
                assert st == oracle.ETOOFEW and kept is None
            else:
                assert st == oracle.OK and kept.tolist() == np.flatnonzero(mask).tolist()


def test_timeout_infinite_keeps_every_arrived_worker_and_equals_the_plain_mean():
    """timeout = +inf with all workers arrived is Sync-SGD without backups: numpy's float64 mean over W."""
    rng = np.random.default_rng(61)
    P, W = 300, 16
    theta, grads = _case(rng, P, W)
    a = rng.lognormal(0, 0.3, W).astype(f32)
    st, kept = oracle.select_timeout(a, float("inf"))
    assert kept.tolist() == list(range(W))
    th = theta.copy()
    oracle.aggregate_update_rows([0, P], W, grads, kept.reshape(1, W), th, per_shard=False,
                                 n_kept=np.array([W], np.int32), ema_mode=oracle.EMA_OFF, gamma_t=0.5)
    want = theta.astype(np.float64) - 0.5 * np.stack(grads).astype(np.float64).mean(axis=0)
    assert ulp_diff(th, want.astype(f32)).max() <= 1


def test_timeout_divides_by_the_number_kept_not_by_W():
    """Constant gradient g in every buffer: the mean is g whatever the number kept (a wrong divisor shows)."""
    P, W = 64, 9
    g = np.full(P, 0.75, f32)
    grads = [g.copy() for _ in range(W)]
    a = np.arange(1, W + 1, dtype=f32)
    for tau, n in ((1.0, 1), (2.0, 2), (4.0, 4), (8.0, 8)):
        st, kept = oracle.select_timeout(a, tau)
        assert len(kept) == n
        rows = np.full((1, W), -1, np.int32)
        rows[0, :n] = kept
        th = np.zeros(P, f32)
        oracle.aggregate_update_rows([0, P], W, grads, rows, th, per_shard=False, n_kept=np.array([n], np.int32),
                                     ema_mode=oracle.EMA_OFF, gamma_t=1.0)
        assert (th == f32(-0.75)).all()


def test_rows_invalid_arguments():
    P, W = 8, 3
    theta = np.zeros(P, f32)
    grads = [np.zeros(P, f32) for _ in range(W)]
    kept = np.array([[0, 1, 2]], np.int32)
    ok = dict(per_shard=False, ema_mode=oracle.EMA_OFF)
    assert oracle.aggregate_update_rows([0, P], 2, grads, kept, theta, n_kept=np.array([0], np.int32), **ok) == oracle.EINVAL
    assert oracle.aggregate_update_rows([0, P], 2, grads, kept, theta, n_kept=np.array([4], np.int32), **ok) == oracle.EINVAL
    bad = np.array([[0, 1, 3]], np.int32)
    assert oracle.aggregate_update_rows([0, P], 3, grads, bad, theta, **ok) == oracle.EINVAL
    assert (theta == 0).all()
    assert oracle.select_timeout(np.ones(3, f32), float("nan"))[0] == oracle.EINVAL
    assert oracle.select_timeout(np.ones(3, f32), 1.0, min_keep=0)[0] == oracle.EINVAL
