"""Pins for oracle_staleness: the bookkeeping behind Table 1 of the paper for Algorithm 2 ("Staleness of a gradient is
measured as the number of updates that have occurred between its corresponding read and update operations",
PAPER.md:L110; workers loop read -> compute -> send, Alg. 1 L58-76) and the fixed-lag simulation of section 2.1 (L114).

Expected values: a hand-worked example (tests/golden/hand_worked_staleness.json), the closed form for equally fast
workers served round-robin (every gradient sees exactly W - 1 other updates -- the order of magnitude of Table 1, where
40 workers give means of 14.5 to 39), a brute-force event replay written independently here, and numpy's statistics."""
import json
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hand_worked_staleness.json")


def _i64(x):
    return np.array(x, dtype=np.int64)


def _i32(x):
    return np.array(x, dtype=np.int32)


def test_golden_hand_worked_batches():
    g = json.load(open(GOLDEN))
    for name in ("batch1", "batch2"):
        b = g[name]
        rc, st, nxt, stats = oracle.staleness(_i64(b["read_iter"]), _i32(b["order"]), b["t0"])
        assert rc == oracle.OK and st.tolist() == b["staleness"] and nxt.tolist() == b["read_iter_out"]
        assert stats[0] == b["min"] and stats[1] == b["mean"] and stats[2] == b["median"] and stats[3] == b["max"]
        assert stats[4] == np.sqrt(b["var_times_K"] / b["count"]) and stats[5] == b["count"]
    b = g["batch2_lag5"]
    rc, st, nxt, _ = oracle.staleness(_i64(b["read_iter"]), _i32(b["order"]), b["t0"], lag=b["lag"])
    assert rc == oracle.OK and st.tolist() == b["staleness"] and nxt.tolist() == b["read_iter_out"]
    b = g["partial"]
    rc, st, nxt, stats = oracle.staleness(_i64(b["read_iter"]), _i32(b["order"]), b["t0"])
    assert rc == oracle.OK and st.tolist() == b["staleness"] and nxt.tolist() == b["read_iter_out"]
    assert stats[2] == b["median"] and stats[5] == 2


@pytest.mark.parametrize("W", [1, 2, 7, 40, 106])
def test_round_robin_workers_have_staleness_W_minus_1(W):
    """W equally fast workers, served in the same order every round: after the first round every gradient was
    computed from parameters that are exactly W - 1 updates old (each of the other workers got one update in)."""
    read = np.zeros(W, np.int64)
    order = np.arange(W, dtype=np.int32)
    t0 = 0
    for rnd in range(4):
        rc, st, read, stats = oracle.staleness(read, order, t0)
        assert rc == oracle.OK
        if rnd == 0:
            assert st.tolist() == list(range(W))              # everybody read the initial parameters
        else:
            assert (st == W - 1).all() and stats[1] == W - 1 and stats[4] == 0.0
        t0 += W


@pytest.mark.parametrize("seed", range(5))
def test_random_orders_against_an_event_replay_and_numpy(seed):
    rng = np.random.default_rng(700 + seed)
    W = int(rng.integers(2, 60))
    lag = int(rng.integers(0, 4))
    read = np.zeros(W, np.int64)
    version_read = {k: 0 for k in range(W)}                   # replay: which parameter version each worker holds
    t0 = 0
    for batch in range(6):
        K = int(rng.integers(0, W + 1))
        order = rng.permutation(W)[:K].astype(np.int32)
        rc, st, nxt, stats = oracle.staleness(read, order, t0, lag=lag)
        assert rc == oracle.OK
        # replay the events one by one: versions are numbered by the update counter
        counter = t0 + lag
        want = []
        for k in order.tolist():
            want.append(counter - version_read[k])            # updates applied since that worker's read
            counter += 1
            version_read[k] = counter                          # it reads the parameters that include its own update
        assert st.tolist() == want
        assert nxt.tolist() == [version_read[k] for k in range(W)]
        if K:
            a = np.array(want, dtype=np.float64)
            assert stats[0] == a.min() and stats[3] == a.max() and stats[5] == K
            assert stats[2] == np.median(a)
            assert abs(stats[1] - a.mean()) <= 1e-12 * max(1.0, abs(a.mean())) and abs(stats[4] - a.std()) <= 1e-12 * max(1.0, a.std())
        else:
            assert np.isnan(stats[:5]).all() and stats[5] == 0
        read, t0 = nxt, t0 + K                                 # the lag is a delay line: the counter advances by K


def test_invalid_arguments():
    r = _i64([0, 0, 0])
    assert oracle.staleness(r, _i32([0, 0]), 0)[0] == oracle.EINVAL          # a worker twice in one batch
    assert oracle.staleness(r, _i32([0, 3]), 0)[0] == oracle.EINVAL          # no such worker
    assert oracle.staleness(_i64([5, 0, 0]), _i32([0]), 0)[0] == oracle.EINVAL  # read from the future
    assert oracle.staleness(r, _i32([0]), -1)[0] == oracle.EINVAL
    assert oracle.staleness(r, _i32([0]), 0, lag=-1)[0] == oracle.EINVAL
