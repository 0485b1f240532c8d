"""Pins for the oracle's straggler statistics (NEXT-4: the procedure of PAPER.md section 3.1).
Expected values: a hand-worked example (tests/golden/hand_worked_stragglers.json) and numpy's sort / mean / median."""
import json
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hand_worked_stragglers.json")


def _arr(x):
    return np.array([[float(v) for v in r] for r in x], dtype=np.float32)


def test_golden_hand_worked():
    with open(GOLDEN) as fh:
        g = json.load(fh)
    a = _arr(g["arrival"])
    r = oracle.kth_arrival_stats(a, np.array(g["iters"]))
    assert np.array_equal(r["sorted"], _arr(g["sorted"]))
    assert r["count"].tolist() == g["count"] and r["median"].tolist() == g["median"]
    assert np.allclose(r["mean"], np.array(g["mean_num"]) / np.array(g["mean_den"]), rtol=1e-15)
    assert np.allclose(r["est_time"], np.array(g["est_time_num"]) / np.array(g["est_time_den"]), rtol=1e-15)
    assert oracle.kth_arrival_stats(a[:2].copy())["median"].tolist() == g["median_first_two_iterations"]


@pytest.mark.parametrize("seed", range(4))
def test_against_numpy_sort_mean_median(seed):
    rng = np.random.default_rng(300 + seed)
    T, W = int(rng.integers(1, 60)), int(rng.integers(1, 40))
    a = rng.lognormal(0, 0.3, (T, W)).astype(np.float32)
    a[rng.random((T, W)) < 0.02] *= 5
    a[rng.random((T, W)) < 0.1] = np.inf
    a[rng.random((T, W)) < 0.05] = np.nan
    r = oracle.kth_arrival_stats(a)
    want = np.sort(np.where(np.isfinite(a), a, np.inf), axis=1)
    assert np.array_equal(r["sorted"], want)
    for k in range(W):
        col = want[:, k][np.isfinite(want[:, k])].astype(np.float64)
        assert r["count"][k] == col.size
        if col.size:
            assert np.isclose(r["mean"][k], col.mean(), rtol=1e-14) and r["median"][k] == np.median(col)
        else:
            assert np.isnan(r["mean"][k]) and np.isnan(r["median"][k])


def test_invariants_of_order_statistics():
    """With every worker reporting: the k-th arrival is no earlier than the (k-1)-th, so mean and median grow
    with k; permuting workers within an iteration, or the iterations, changes nothing but the row order."""
    rng = np.random.default_rng(7)
    T, W = 50, 12
    a = rng.lognormal(0, 0.3, (T, W)).astype(np.float32)
    r = oracle.kth_arrival_stats(a)
    assert (np.diff(r["mean"]) >= 0).all() and (np.diff(r["median"]) >= 0).all() and (r["count"] == T).all()
    assert r["mean"][0] == a.min(axis=1).astype(np.float64).mean()
    assert np.isclose(r["mean"][-1], a.max(axis=1).astype(np.float64).mean(), rtol=1e-15)
    b = np.stack([row[rng.permutation(W)] for row in a])
    r2 = oracle.kth_arrival_stats(b)
    assert np.array_equal(r["sorted"], r2["sorted"]) and np.array_equal(r["median"], r2["median"])
    perm = rng.permutation(T)
    r3 = oracle.kth_arrival_stats(a[perm].copy())
    assert np.array_equal(r3["sorted"], r["sorted"][perm]) and np.array_equal(r3["median"], r["median"])
    assert np.allclose(r3["mean"], r["mean"], rtol=1e-14)


def test_first_n_wait_time_is_the_nth_order_statistic():
    """The time the synchronous server waits (t_Nth of the selection, L130) is column N-1 of the sorted row."""
    rng = np.random.default_rng(8)
    W = 9
    a = rng.lognormal(0, 0.3, (5, W)).astype(np.float32)
    r = oracle.kth_arrival_stats(a)
    for t in range(5):
        for N in range(1, W + 1):
            assert oracle.select_first_n(a[t].copy(), N, W - N)[2] == r["sorted"][t, N - 1]


def test_invalid_arguments():
    with pytest.raises(ValueError):
        oracle.kth_arrival_stats(np.zeros((0, 3), np.float32))
    with pytest.raises(ValueError):
        oracle.kth_arrival_stats(np.zeros(3, np.float32))


# ------------------------------------------------------------------ Fig. 5 -> Fig. 6: iterations(N), interpolated
def test_interp_iterations_paper_points():
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_fig5_points.json")) as fh:
        g = json.load(fh)
    it = oracle.interp_iterations(g["N"], g["iterations"], 106)
    for n, want in g["interpolated"].items():
        assert abs(it[int(n) - 1] - want) <= 1e-9 * want
    assert 0.55 < it[99] / it[49] < 0.56                       # "nearly halves" (L181)
    assert (it[:50] == 137500.0).all() and (it[99:] == 76200.0).all()      # held outside the measured range (R23)
    assert (np.diff(it[49:100]) < 0).all()


def test_interp_iterations_against_numpy_interp_and_fig6_product():
    rng = np.random.default_rng(11)
    N_pts = np.array([50, 70, 80, 90, 100], np.int32)
    iters = np.sort(rng.uniform(7e4, 1.4e5, 5))[::-1].copy()
    W = 106
    got = oracle.interp_iterations(N_pts, iters, W)
    want = np.interp(np.arange(1, W + 1), N_pts, iters)        # numpy holds the end values too
    assert np.allclose(got, want, rtol=1e-15, atol=0)
    a = rng.lognormal(0, 0.25, (40, W)).astype(np.float32)
    r = oracle.kth_arrival_stats(a, got)
    assert np.allclose(r["est_time"], r["mean"] * want, rtol=1e-14)
    best = int(np.argmin(r["est_time"][49:100])) + 50          # Fig. 6: the N in 50..100 with the least estimated time
    assert 50 <= best <= 100
    with pytest.raises(ValueError):
        oracle.interp_iterations([50, 50], [1.0, 2.0], 10)
    with pytest.raises(ValueError):
        oracle.interp_iterations([], [], 10)
