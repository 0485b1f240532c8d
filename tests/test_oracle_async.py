"""Pins for the oracle's Async-SGD parameter-server step (NEXT-3: Algorithm 2).

Expected values: a hand-worked example (tests/golden/hand_worked_async.json), numpy's lexsort for the
arrival order, exact rational arithmetic with one fp32 rounding per stored value per iteration, numpy's
float64 sum for the SGD closed form, and the reduction "K async iterations = K synchronous steps with
N=1, b=0" onto the already pinned synchronous step.
"""
import itertools
import json
import os

import numpy as np
import pytest

import oracle
from test_oracle_update import F, _round_f32, coeffs, f32, ulp_diff

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hand_worked_async.json")


def _load():
    with open(GOLDEN) as fh:
        return json.load(fh)


def _arr(x):
    return np.array(x, dtype=np.float32)


def test_golden_async_pre_post_and_per_iteration_gamma():
    g = _load()
    order = oracle.order_by_arrival(_arr(g["arrival"]))
    assert order.tolist() == g["order"]
    grads = [_arr(x) for x in g["grads"]]
    for mode, key in ((oracle.EMA_PRE, "ema_pre"), (oracle.EMA_POST, "ema_post")):
        theta, ema = _arr(g["theta"]), _arr(g["ema"])
        assert oracle.async_apply([0, 1, 2], grads, order, theta, ema, ema_mode=mode, gamma_t=g["gamma"],
                                  alpha=g["alpha"]) == oracle.OK
        assert theta.tolist() == g["theta_out"] and ema.tolist() == g[key]
    theta = _arr(g["theta"])
    oracle.async_apply([0, 2], grads, order, theta, gammas=_arr(g["gammas"]), ema_mode=oracle.EMA_OFF, gamma_t=99.0)
    assert theta.tolist() == g["theta_out_gammas"]


# ------------------------------------------------------------------ arrival order
@pytest.mark.parametrize("W", [1, 2, 3, 4, 5])
def test_order_exhaustive_with_ties(W):
    for combo in itertools.product([0.0, 1.0, 2.0], repeat=W):
        a = np.array(combo, dtype=np.float32)
        assert oracle.order_by_arrival(a).tolist() == sorted(range(W), key=lambda k: (combo[k], k))


@pytest.mark.parametrize("seed", range(5))
def test_order_matches_numpy_lexsort(seed):
    rng = np.random.default_rng(800 + seed)
    W = int(rng.integers(1, 200))
    a = rng.lognormal(0, 0.3, W).astype(f32)
    ties = rng.random(W) < 0.3
    a[ties] = rng.choice(np.array([0.5, 1.0, -0.0, 0.0, -1.5], f32), size=int(ties.sum()))
    a[rng.random(W) < 0.1] = np.inf
    a[rng.random(W) < 0.05] = np.nan
    a[rng.random(W) < 0.05] = -np.inf
    idx = np.flatnonzero(np.isfinite(a))
    want = idx[np.lexsort((idx, a[idx] + f32(0.0)))]
    assert oracle.order_by_arrival(a).tolist() == want.tolist()


def test_order_is_the_first_n_selection_for_every_prefix():
    """The first N entries of the arrival order are, as a set, the first-N-of-W selection (L130)."""
    rng = np.random.default_rng(9)
    W = 23
    a = rng.lognormal(0, 0.3, W).astype(f32)
    a[[3, 7]] = a[11]
    order = oracle.order_by_arrival(a)
    for N in range(1, W + 1):
        st, kept, t_nth = oracle.select_first_n(a, N, W - N)
        assert sorted(order[:N].tolist()) == kept.tolist() and t_nth == a[order[N - 1]]


# ------------------------------------------------------------------ the K-iteration update
def _case(rng, P, W, bf16=False):
    theta = rng.normal(0, 0.02, P).astype(f32)
    g = [rng.normal(0, 1e-3, P).astype(f32) for _ in range(W)]
    if bf16:
        g = [(x.view(np.uint32) >> 16).astype(np.uint16) for x in g]
    return theta, g


def _vals(g):
    return (g.astype(np.uint32) << 16).view(np.float32) if g.dtype == np.uint16 else g


@pytest.mark.parametrize("opt", [oracle.SGD, oracle.MOMENTUM, oracle.RMSPROP_MOM])
@pytest.mark.parametrize("ema_mode", [oracle.EMA_PRE, oracle.EMA_POST, oracle.EMA_OFF])
def test_async_is_k_synchronous_steps_with_n1_b0(opt, ema_mode):
    """Alg. 2 is Alg. 4 with N=1, b=0 run once per arrival: bit-identical to the pinned synchronous step."""
    rng = np.random.default_rng(90 + 3 * opt + ema_mode)
    P, W = 257, 9
    off = [0, 100, 100, P]
    theta, grads = _case(rng, P, W, bf16=(opt == oracle.MOMENTUM))
    a = rng.lognormal(0, 0.3, W).astype(f32)
    a[4] = np.inf                                        # one worker never reports
    order = oracle.order_by_arrival(a)
    assert order.size == W - 1
    gammas = rng.uniform(0.01, 0.1, order.size).astype(f32)
    hp = dict(opt=opt, ema_mode=ema_mode, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0)
    st = [theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)]
    ref = [x.copy() for x in st]
    assert oracle.async_apply(off, grads, order, *st, gammas=gammas, **hp) == oracle.OK
    for i, k in enumerate(order):
        assert oracle.aggregate_update(off, 1, grads, np.array([k], np.int32), *ref, gamma_t=float(gammas[i]),
                                       **hp) == oracle.OK
    for x, y in zip(st, ref):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("ema_mode", [oracle.EMA_PRE, oracle.EMA_POST])
def test_async_exact_rational_brute_force_sgd(ema_mode):
    """P <= 64: exact Fractions, rounded to fp32 once per stored value per iteration (the server's state)."""
    rng = np.random.default_rng(95 + ema_mode)
    P, W = 40, 6
    theta, grads = _case(rng, P, W)
    ema0 = (theta + rng.normal(0, 1e-3, P)).astype(f32)
    a = rng.lognormal(0, 0.3, W).astype(f32)
    order = oracle.order_by_arrival(a)
    gamma, alpha = 0.045, 0.9999
    th, em = theta.copy(), ema0.copy()
    assert oracle.async_apply([0, 7, P], grads, order, th, em, ema_mode=ema_mode, gamma_t=gamma, alpha=alpha) == oracle.OK
    _, oma, _ = coeffs(1, alpha)
    for e in range(P):
        t, m = F(theta[e]), F(ema0[e])
        for k in order:
            t_new = F(_round_f32(t - F(f32(gamma)) * F(grads[k][e])))
            operand = t_new if ema_mode == oracle.EMA_POST else t
            m = F(_round_f32(F(f32(alpha)) * m + oma * operand))
            t = t_new
        assert ulp_diff(th[e], f32(float(t))) <= 1 and ulp_diff(em[e], f32(float(m))) <= 1


def test_async_sgd_constant_gamma_closed_form_numpy_sum():
    """theta(K) = theta(0) - gamma * sum of all arrived gradients, whatever the order (up to rounding)."""
    rng = np.random.default_rng(97)
    P, W = 500, 32
    theta, grads = _case(rng, P, W)
    order = oracle.order_by_arrival(rng.lognormal(0, 0.3, W).astype(f32))
    th = theta.copy()
    oracle.async_apply([0, P], grads, order, th, ema_mode=oracle.EMA_OFF, gamma_t=0.25)
    want = theta.astype(np.float64) - 0.25 * np.stack(grads).astype(np.float64).sum(axis=0)
    assert np.abs(th - want).max() <= W * 2.0 ** -24 * np.abs(want).max()      # one fp32 rounding per iteration


def test_async_differs_from_the_synchronous_mean_and_order_matters_for_momentum():
    rng = np.random.default_rng(98)
    P, W = 64, 5
    theta, grads = _case(rng, P, W)
    order = np.arange(W, dtype=np.int32)
    a = [theta.copy(), None, np.zeros(P, f32)]
    b = [theta.copy(), None, np.zeros(P, f32)]
    hp = dict(opt=oracle.MOMENTUM, ema_mode=oracle.EMA_OFF, gamma_t=0.5, mu=0.9)
    oracle.async_apply([0, P], grads, order, *a, **hp)
    oracle.async_apply([0, P], grads, order[::-1].copy(), *b, **hp)
    assert not np.array_equal(a[0], b[0])                       # arrival order matters
    c = [theta.copy(), None, np.zeros(P, f32)]
    oracle.aggregate_update([0, P], W, grads, order, *c, **hp)
    assert np.abs(a[0] - c[0]).max() > 1e-4                     # W async iterations != one synchronous step


def test_async_k0_is_a_no_op_and_invalid_arguments():
    theta = np.arange(4, dtype=f32)
    grads = [np.ones(4, f32)]
    assert oracle.async_apply([0, 4], grads, np.zeros(0, np.int32), theta, ema_mode=oracle.EMA_OFF, gamma_t=1.0) == oracle.OK
    assert theta.tolist() == [0, 1, 2, 3]
    assert oracle.async_apply([0, 4], grads, np.array([1], np.int32), theta, ema_mode=oracle.EMA_OFF) == oracle.EINVAL
    assert oracle.async_apply([0, 4], grads, np.array([0, 0], np.int32), theta, ema_mode=oracle.EMA_OFF) == oracle.EINVAL
    assert oracle.async_apply([0, 3], grads, np.array([0], np.int32), theta, ema_mode=oracle.EMA_OFF) == oracle.EINVAL


# ------------------------------------------------------------------ Alg. 2 per parameter server j (rows, slices)
def _g():
    with open(os.path.join(os.path.dirname(__file__), "golden", "hand_worked_async.json")) as fh:
        return json.load(fh)


def test_golden_per_server_orders_counts_rates_clip_factors_and_a_failed_server():
    g = _g()
    ps = g["per_server"]
    arr = lambda x: np.array(x, dtype=np.float32)                            # noqa: E731
    flat = [arr(x) for x in g["grads"]]
    sl = [[x[0:1].copy(), x[1:2].copy()] for x in flat]                       # what each server receives
    order = np.array(ps["order"], np.int32)
    n = np.array(ps["n_arrived"], np.int32)
    for grads, slices in ((flat, False), (sl, True)):
        for mode, key in ((oracle.EMA_PRE, "ema_pre"), (oracle.EMA_POST, "ema_post")):
            th, em = arr(g["theta"]), arr(g["ema"])
            assert oracle.async_apply_rows(ps["shard_off"], grads, order, th, em, slices=slices, n_arrived=n,
                                           ema_mode=mode, gamma_t=g["gamma"], alpha=g["alpha"]) == oracle.OK
            assert th.tolist() == ps["theta_out"] and em.tolist() == ps[key]
        th = arr(g["theta"])
        assert oracle.async_apply_rows(ps["shard_off"], grads, order, th, None, slices=slices, n_arrived=n,
                                       gammas=arr(g["gammas"]), ema_mode=oracle.EMA_OFF) == oracle.OK
        assert th.tolist() == ps["theta_out_gammas"]
        th = arr(g["theta"])
        assert oracle.async_apply_rows(ps["shard_off"], grads, order, th, None, slices=slices, n_arrived=n,
                                       gscales=arr(ps["gscales"]), ema_mode=oracle.EMA_OFF, gamma_t=g["gamma"]) == oracle.OK
        assert th.tolist() == ps["theta_out_scaled"]
        th, em = arr(g["theta"]), arr(g["ema"])
        assert oracle.async_apply_rows(ps["shard_off"], grads, order, th, em, slices=slices, n_arrived=n,
                                       status=np.array(ps["failed_status"], np.int32), gamma_t=g["gamma"],
                                       alpha=g["alpha"]) == oracle.OK
        assert th.tolist() == ps["failed_theta_out"] and em.tolist() == ps["failed_ema_pre"]


@pytest.mark.parametrize("opt", [oracle.SGD, oracle.MOMENTUM, oracle.RMSPROP_MOM])
@pytest.mark.parametrize("bf16", [False, True])
def test_per_server_rows_reduce_to_the_pinned_single_order_oracle_server_by_server(opt, bf16):
    """Each server's slice must equal what the already pinned oracle_async_apply computes when it is given that
    server's parameters alone, its own order, count, rates and (per-arrival) clip factors -- flat and sliced."""
    from test_oracle_update import to_bf16_bits
    rng = np.random.default_rng(810 + 2 * opt + bf16)
    P, M, W = 1501, 6, 9
    cuts = np.sort(rng.integers(0, P + 1, M - 1))
    off = np.concatenate([[0], cuts, [P]]).astype(np.int64)
    off[3] = off[2]                                                            # an empty server
    off = np.sort(off)
    theta = rng.normal(0, 0.02, P).astype(np.float32)
    grads = [rng.normal(0, 1e-3, P).astype(np.float32) for _ in range(W)]
    if bf16:
        grads = [to_bf16_bits(x) for x in grads]
    order = np.full((M, W), -1, np.int32)
    n = rng.integers(0, W + 1, M).astype(np.int32)
    for j in range(M):
        order[j, :n[j]] = rng.permutation(W)[:n[j]]
    status = np.zeros(M, np.int32)
    status[4] = oracle.ETOOFEW
    gammas = rng.uniform(0.01, 0.09, W).astype(np.float32)
    gscales = rng.uniform(0.3, 1.0, W).astype(np.float32)
    hp = dict(opt=opt, ema_mode=oracle.EMA_PRE, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0)

    def state():
        return [theta.copy(), theta.copy(), np.ones(P, np.float32) if opt else None,
                np.zeros(P, np.float32) if opt == oracle.RMSPROP_MOM else None]

    want = state()
    for j in range(M):
        lo, hi = int(off[j]), int(off[j + 1])
        if status[j] != 0 or hi == lo or n[j] == 0:
            continue
        sub = [None if a is None else a[lo:hi].copy() for a in want]
        o = order[j, :n[j]].copy()
        assert oracle.async_apply([0, hi - lo], [x[lo:hi].copy() for x in grads], o, *sub, gammas=gammas[:n[j]].copy(),
                                  gscales=gscales[o].copy(), **hp) == oracle.OK
        for a, b_ in zip(want, sub):
            if a is not None:
                a[lo:hi] = b_
    got = state()
    assert oracle.async_apply_rows(off, grads, order, *got, n_arrived=n, status=status, gammas=gammas, gscales=gscales,
                                   **hp) == oracle.OK
    sl = [[x[off[j]:off[j + 1]].copy() for j in range(M)] for x in grads]
    got_s = state()
    assert oracle.async_apply_rows(off, sl, order, *got_s, slices=True, n_arrived=n, status=status, gammas=gammas,
                                   gscales=gscales, **hp) == oracle.OK
    for a, b_, c in zip(want, got, got_s):
        if a is not None:
            assert np.array_equal(a, b_) and np.array_equal(a, c)
    assert np.array_equal(got[0][off[4]:off[5]], theta[off[4]:off[5]])         # the failed server is untouched


def test_per_server_rows_invalid_arguments():
    g = _g()
    arr = lambda x: np.array(x, dtype=np.float32)                            # noqa: E731
    flat = [arr(x) for x in g["grads"]]
    th = arr(g["theta"])
    bad = np.array([[0, 3, 1], [1, 0, -1]], np.int32)
    assert oracle.async_apply_rows([0, 1, 2], flat, bad, th, None, ema_mode=oracle.EMA_OFF) == oracle.EINVAL
    ok = np.array([[0, 2, 1], [1, 0, 2]], np.int32)
    assert oracle.async_apply_rows([0, 1, 2], flat, ok, th, None, n_arrived=np.array([3, 4], np.int32),
                                   ema_mode=oracle.EMA_OFF) == oracle.EINVAL
    assert th.tolist() == g["theta"]
