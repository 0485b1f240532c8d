"""Pins for oracle_aggregate_update_slices: Alg. 4 l.8-9 on what each parameter server RECEIVES -- one separate
buffer G_k[j] per (worker, server) (theta[j] owned by server j, L42).

Nothing here re-calls the function under test to check it: expected values come from a hand-worked dyadic example
(tests/golden/hand_worked_slices.json), from the already pinned flat-layout oracle when the slices are views of flat
buffers (same numbers, different addressing: must be bit-equal), from exact rational arithmetic on separately
allocated, odd-offset slices (P <= 64), and from numpy's float64 mean per slice.
"""
import json
import os

import numpy as np
import pytest

import oracle
from test_oracle_update import exact_step, f32, to_bf16_bits, bf16_bits_to_f32

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hand_worked_slices.json")


def _arr(x, dt=np.float32):
    return np.array(x, dtype=dt)


def _load():
    with open(GOLDEN) as fh:
        return json.load(fh)


def _slices(g):
    return [[_arr(s) for s in row] for row in g["slices"]]


def odd_offset_copy(a, offset_elems):
    """The same values in a fresh allocation that starts `offset_elems` elements after a 64-byte boundary."""
    raw = np.zeros(a.size + 32 + offset_elems, dtype=a.dtype)
    base = (-raw.ctypes.data // a.itemsize) % (64 // a.itemsize)       # elements up to the next 64-byte boundary
    out = raw[base + offset_elems: base + offset_elems + a.size]
    out[:] = a
    assert (raw.ctypes.data + base * a.itemsize) % 64 == 0
    return out


# ------------------------------------------------------------------ hand-worked example
def test_golden_one_kept_set_sgd_ema_post_pre_and_momentum():
    g = _load()
    kept = _arr(g["A"]["kept"], np.int32)
    for mode, key in ((oracle.EMA_POST, "ema_post"), (oracle.EMA_PRE, "ema_pre")):
        theta, ema = _arr(g["theta"]), _arr(g["theta"])
        assert oracle.aggregate_update_slices(g["shard_off"], g["N"], _slices(g), kept, theta, ema, ema_mode=mode,
                                              gamma_t=g["gamma"], alpha=g["alpha"]) == oracle.OK
        assert theta.tolist() == g["A"]["theta_out"] and ema.tolist() == g["A"][key]
    m = g["A"]["momentum"]
    theta, v = _arr(g["theta"]), _arr(m["v"])
    assert oracle.aggregate_update_slices(g["shard_off"], g["N"], _slices(g), kept, theta, None, v,
                                          opt=oracle.MOMENTUM, ema_mode=oracle.EMA_OFF, gamma_t=g["gamma"],
                                          mu=m["mu"]) == oracle.OK
    assert theta.tolist() == m["theta_out"] and v.tolist() == m["v_out"]


def test_golden_one_kept_row_per_server_and_failed_server():
    g = _load()
    kept = _arr(g["B"]["kept"], np.int32)
    theta, ema = _arr(g["theta"]), _arr(g["theta"])
    assert oracle.aggregate_update_slices(g["shard_off"], g["N"], _slices(g), kept, theta, ema, per_shard=True,
                                          gamma_t=g["gamma"], alpha=g["alpha"]) == oracle.OK
    assert theta.tolist() == g["B"]["theta_out"] and ema.tolist() == g["B"]["ema_post"]
    theta, ema = _arr(g["theta"]), _arr(g["theta"])
    assert oracle.aggregate_update_slices(g["shard_off"], g["N"], _slices(g), kept, theta, ema, per_shard=True,
                                          status=_arr(g["C"]["status"], np.int32), gamma_t=g["gamma"],
                                          alpha=g["alpha"]) == oracle.OK
    assert theta.tolist() == g["C"]["theta_out"] and ema.tolist() == g["C"]["ema_post"]


def test_golden_slices_nobody_keeps_are_never_read():
    """Server j never dereferences the slice of a worker it does not keep: None entries and NaN poison change nothing."""
    g = _load()
    kept = _arr(g["B"]["kept"], np.int32)          # server 0 keeps workers 0,1; server 1 keeps 1,2
    sl = _slices(g)
    sl[2][0] = None                                # worker 2 -> server 0: dropped there
    sl[0][1] = np.full(2, np.nan, np.float32)      # worker 0 -> server 1: dropped there
    theta, ema = _arr(g["theta"]), _arr(g["theta"])
    assert oracle.aggregate_update_slices(g["shard_off"], g["N"], sl, kept, theta, ema, per_shard=True,
                                          gamma_t=g["gamma"], alpha=g["alpha"]) == oracle.OK
    assert theta.tolist() == g["B"]["theta_out"] and ema.tolist() == g["B"]["ema_post"]
    sl[1][0] = None                                # ... but a KEPT slice must be there
    theta2 = _arr(g["theta"])
    assert oracle.aggregate_update_slices(g["shard_off"], g["N"], sl, kept, theta2, _arr(g["theta"]), per_shard=True,
                                          gamma_t=g["gamma"], alpha=g["alpha"]) == oracle.EINVAL
    assert theta2.tolist() == g["theta"]           # nothing was written


# ------------------------------------------------------------------ views of flat buffers: the pinned flat oracle
def _ragged(rng, P, M):
    cuts = np.sort(rng.integers(0, P + 1, M - 1))
    return np.concatenate([[0], cuts, [P]]).astype(np.int64)


@pytest.mark.parametrize("opt", [oracle.SGD, oracle.MOMENTUM, oracle.RMSPROP_MOM])
@pytest.mark.parametrize("ema_mode", [oracle.EMA_POST, oracle.EMA_PRE, oracle.EMA_OFF])
@pytest.mark.parametrize("bf16", [False, True])
def test_views_of_flat_buffers_are_bit_equal_to_the_flat_oracle(opt, ema_mode, bf16):
    rng = np.random.default_rng(500 + 9 * opt + 3 * ema_mode + bf16)
    P, M, N, W = 3001, 9, 6, 8
    off = _ragged(rng, P, M)
    off[4] = off[3]                                                   # one empty server
    off = np.sort(off)
    theta = rng.normal(0, 0.02, P).astype(f32)
    grads = [rng.normal(0, 1e-3, P).astype(f32) for _ in range(W)]
    if bf16:
        grads = [to_bf16_bits(g) for g in grads]
    kept = np.sort(rng.permutation(W)[:N]).astype(np.int32)
    hp = dict(opt=opt, ema_mode=ema_mode, gamma_t=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0)

    def state():
        return [theta.copy(), None if ema_mode == oracle.EMA_OFF else theta.copy(),
                None if opt == oracle.SGD else np.ones(P, f32), np.zeros(P, f32) if opt == oracle.RMSPROP_MOM else None]

    a = state()
    assert oracle.aggregate_update(off, N, grads, kept, *a, **hp) == oracle.OK
    views = [[g[off[j]:off[j + 1]] for j in range(M)] for g in grads]       # odd offsets come for free
    b = state()
    assert oracle.aggregate_update_slices(off, N, views, kept, *b, **hp) == oracle.OK
    # separately allocated copies, each at its own odd element offset
    copies = [[odd_offset_copy(v, int(rng.integers(0, 8))) for v in row] for row in views]
    c = state()
    assert oracle.aggregate_update_slices(off, N, copies, kept, *c, **hp) == oracle.OK
    for x, y, z in zip(a, b, c):
        if x is not None:
            assert np.array_equal(x, y) and np.array_equal(x, z)


def test_views_with_rows_counts_and_status_are_bit_equal_to_the_rows_oracle():
    rng = np.random.default_rng(540)
    P, M, N, W = 2003, 7, 5, 9
    off = _ragged(rng, P, M)
    theta = rng.normal(0, 0.02, P).astype(f32)
    grads = [rng.normal(0, 1e-3, P).astype(f32) for _ in range(W)]
    kept = np.full((M, W), -1, np.int32)
    n_kept = rng.integers(1, W + 1, M).astype(np.int32)
    for j in range(M):
        kept[j, :n_kept[j]] = np.sort(rng.permutation(W)[:n_kept[j]])
    status = np.zeros(M, np.int32)
    status[2] = oracle.ETOOFEW
    hp = dict(per_shard=True, n_kept=n_kept, status=status, opt=oracle.RMSPROP_MOM, gamma_t=0.045, alpha=0.9999,
              mu=0.9, rho=0.9, eps=1.0)
    a = [theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)]
    assert oracle.aggregate_update_rows(off, N, grads, kept, *a, **hp) == oracle.OK
    views = [[g[off[j]:off[j + 1]] for j in range(M)] for g in grads]
    b = [theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)]
    assert oracle.aggregate_update_slices(off, N, views, kept, *b, **hp) == oracle.OK
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    assert np.array_equal(b[0][off[2]:off[3]], theta[off[2]:off[3]])           # the failed server's slice is untouched


# ------------------------------------------------------------------ exact rationals, P <= 64, odd-offset slices
@pytest.mark.parametrize("opt", [oracle.SGD, oracle.MOMENTUM, oracle.RMSPROP_MOM])
@pytest.mark.parametrize("bf16", [False, True])
def test_exact_rational_brute_force_on_ragged_odd_offset_slices(opt, bf16):
    """Each server's slice is computed with exact rationals (exact_step of tests/test_oracle_update.py: Fraction,
    mpmath square root) from that server's own kept row and count; the oracle may differ by the one fp32 storage
    rounding of a double result that is itself within 2^-52 of exact, i.e. at most the last bit."""
    rng = np.random.default_rng(560 + 2 * opt + bf16)
    P, M, W, N = 61, 5, 6, 4
    off = np.array([0, 7, 8, 8, 33, P], np.int64)                    # ragged, one 1-element and one empty server
    theta = rng.normal(0, 0.02, P).astype(f32)
    ema = (theta + rng.normal(0, 1e-3, P)).astype(f32)
    s0 = np.abs(rng.normal(0.5, 0.2, P)).astype(f32)
    s1 = rng.normal(0, 1e-3, P).astype(f32)
    flat = [rng.normal(0, 1e-3, P).astype(f32) for _ in range(W)]
    if bf16:
        flat = [to_bf16_bits(g) for g in flat]
    vals = [bf16_bits_to_f32(g) if bf16 else g for g in flat]
    slices = [[odd_offset_copy(g[off[j]:off[j + 1]], (3 * k + j) % 7 + 1) for j in range(M)] for k, g in enumerate(flat)]
    kept = np.full((M, W), -1, np.int32)
    n_kept = np.array([4, 3, 2, 6, 1], np.int32)
    for j in range(M):
        kept[j, :n_kept[j]] = np.sort(rng.permutation(W)[:n_kept[j]])
    status = np.array([0, 0, 0, 0, oracle.ETOOFEW], np.int32)
    hp = dict(gamma=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0)
    got = [theta.copy(), ema.copy(), s0.copy() if opt else None, s1.copy() if opt == oracle.RMSPROP_MOM else None]
    assert oracle.aggregate_update_slices(off, N, slices, kept, *got, per_shard=True, n_kept=n_kept, status=status,
                                          opt=opt, ema_mode=oracle.EMA_POST, gamma_t=hp["gamma"], alpha=hp["alpha"],
                                          mu=hp["mu"], rho=hp["rho"], eps=hp["eps"]) == oracle.OK
    for j in range(M):
        lo, hi = int(off[j]), int(off[j + 1])
        if status[j] != 0:
            want = [theta[lo:hi], ema[lo:hi], s0[lo:hi], s1[lo:hi]]
        else:
            n = int(n_kept[j])
            want = exact_step(theta[lo:hi], ema[lo:hi], s0[lo:hi], s1[lo:hi], [v[lo:hi] for v in vals],
                              kept[j, :n].tolist(), n, opt, oracle.EMA_POST, **hp)
        for x, y in zip(got, want):
            if x is not None and hi > lo:
                d = np.abs(x[lo:hi].view(np.int32).astype(np.int64) - np.asarray(y, f32).view(np.int32).astype(np.int64))
                assert d.max() <= 1, (j, d.max())


@pytest.mark.parametrize("bf16", [False, True])
def test_sgd_against_numpy_float64_mean_per_slice(bf16):
    rng = np.random.default_rng(580 + bf16)
    P, M, W, N = 5003, 6, 10, 8                      # N = 8: 1/N exact, so theta' = fl32(theta - gamma * mean) to 1 ulp
    off = _ragged(rng, P, M)
    theta = rng.normal(0, 0.02, P).astype(f32)
    flat = [rng.normal(0, 1e-3, P).astype(f32) for _ in range(W)]
    if bf16:
        flat = [to_bf16_bits(g) for g in flat]
    vals = [(bf16_bits_to_f32(g) if bf16 else g).astype(np.float64) for g in flat]
    slices = [[odd_offset_copy(g[off[j]:off[j + 1]], (k + 2 * j) % 5) for j in range(M)] for k, g in enumerate(flat)]
    kept = np.stack([np.sort(rng.permutation(W)[:N]) for _ in range(M)]).astype(np.int32)
    got = theta.copy()
    assert oracle.aggregate_update_slices(off, N, slices, kept, got, per_shard=True, ema_mode=oracle.EMA_OFF,
                                          gamma_t=0.25) == oracle.OK
    for j in range(M):
        lo, hi = int(off[j]), int(off[j + 1])
        mean = np.mean(np.stack([vals[k][lo:hi] for k in kept[j]]), axis=0)
        want = (theta[lo:hi].astype(np.float64) - 0.25 * mean).astype(f32)
        d = np.abs(got[lo:hi].view(np.int32).astype(np.int64) - want.view(np.int32).astype(np.int64))
        assert d.size == 0 or d.max() <= 1


def test_transposed_table_or_flat_indexing_would_fail():
    """The table is worker-major, entry k*M + j, and element i of a slice is parameter off[j] + i: a result computed
    with the table transposed, or with slice elements addressed by their flat index, differs (sizes differ too)."""
    g = _load()
    sl = _slices(g)
    kept = _arr(g["A"]["kept"], np.int32)
    theta = _arr(g["theta"])
    oracle.aggregate_update_slices(g["shard_off"], g["N"], sl, kept, theta, None, ema_mode=oracle.EMA_OFF,
                                   gamma_t=g["gamma"])
    # server 1's two parameters come from the SECOND slices, elements 0 and 1 -- not from elements 3 and 4 of anything
    assert theta[3] == 4.0 - 0.5 * (sl[0][1][0] + sl[2][1][0]) / 2 and theta[4] == 5.0 - 0.5 * (sl[0][1][1] + sl[2][1][1]) / 2


def test_slices_invalid_arguments():
    g = _load()
    sl = _slices(g)
    theta = _arr(g["theta"])
    ok_kept = _arr([0, 2], np.int32)
    short = [[row[0], row[1][:1]] for row in sl]                     # off[M] = 4 != P = 5
    assert oracle.aggregate_update_slices([0, 3, 4], 2, short, ok_kept, theta, ema_mode=oracle.EMA_OFF) == oracle.EINVAL
    assert oracle.aggregate_update_slices(g["shard_off"], 2, sl, _arr([0, 3], np.int32), theta,
                                          ema_mode=oracle.EMA_OFF) == oracle.EINVAL
    assert oracle.aggregate_update_slices(g["shard_off"], 2, sl, _arr([[0, 2], [0, 2]], np.int32), theta,
                                          per_shard=True, n_kept=_arr([2, 0], np.int32),
                                          ema_mode=oracle.EMA_OFF) == oracle.EINVAL
    with pytest.raises(ValueError):
        oracle.aggregate_update_slices(g["shard_off"], 2, [[sl[0][0]], [sl[1][0]], [sl[2][0]]], ok_kept, theta)
    assert theta.tolist() == g["theta"]
