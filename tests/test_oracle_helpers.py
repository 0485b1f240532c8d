"""Pins for the oracle's NEXT-4 helpers: the learning-rate schedule of A.2/A.3 and the
global-norm clipping Async-Opt needs (reading R22).

Expected values: numbers worked by hand from the paper's own hyper-parameters (gamma_0 = 0.045 N, beta = 0.94), a
3-4-5 triangle, mpmath at 50 digits, numpy's float64 norm, and exact power-of-two scalings."""
import mpmath
import numpy as np
import pytest

import oracle
from test_oracle_update import f32, ulp_diff


# ------------------------------------------------------------------ learning-rate schedule
def test_lr_schedule_paper_hyperparameters_by_hand():
    """A.2 (L305): gamma_0 = 0.045 N, beta = 0.94, gamma_t = gamma_0 beta^(t N / (2T)).  With N = 100 and T = 1000
    mini-batches per epoch the exponent is t/20: every 20 iterations (two epochs of data) the rate shrinks by 0.94.
    By hand: 4.5, 4.5*0.94 = 4.23, 4.5*0.94^2 = 3.97620, 4.5*0.94^3 = 3.737628."""
    N, T = 100, 1000
    g = oracle.lr_schedule(0.045 * N, 0.94, 0, 61, N / (2.0 * T))
    want = np.array([4.5, 4.23, 3.97620, 3.737628], dtype=np.float64)
    assert np.abs(g[[0, 20, 40, 60]].astype(np.float64) - want).max() <= 2e-6      # gamma_0, beta are fp32 inputs
    assert (np.diff(g) < 0).all()
    # Async-Opt (A.3, L315): gamma_0 = 0.045, exponent t/(2T): N times slower per iteration, equal per datapoint
    ga = oracle.lr_schedule(0.045, 0.94, 0, 1, 1 / (2.0 * T))
    gs = oracle.lr_schedule(0.045, 0.94, 0, 1, N / (2.0 * T))
    assert ga[0] == gs[0] == f32(0.045)
    a_late = oracle.lr_schedule(0.045, 0.94, 100 * 37, 1, 1 / (2.0 * T))      # after 3700 async iterations
    s_late = oracle.lr_schedule(0.045, 0.94, 37, 1, N / (2.0 * T))            # after 37 sync iterations: same data seen
    assert ulp_diff(a_late, s_late).max() <= 1


@pytest.mark.parametrize("t0", [0, 1, 12345, 10**7])
def test_lr_schedule_against_mpmath(t0):
    s = 50 / (2.0 * 40037)
    got = oracle.lr_schedule(2.25, 0.94, t0, 5, s)
    with mpmath.workdps(50):
        for i in range(5):
            want = mpmath.mpf(float(f32(2.25))) * mpmath.power(mpmath.mpf(float(f32(0.94))), mpmath.mpf(t0 + i) * mpmath.mpf(s))
            assert ulp_diff(got[i], f32(float(want))) <= 1


def test_lr_schedule_edges():
    assert oracle.lr_schedule(0.1, 0.5, 0, 0, 1.0).size == 0
    assert oracle.lr_schedule(0.75, 0.5, 3, 2, 1.0).tolist() == [0.09375, 0.046875]      # exact powers of two
    assert oracle.lr_schedule(0.1, 1.0, 0, 3, 7.0).tolist() == [f32(0.1)] * 3             # beta = 1: constant
    with pytest.raises(ValueError):
        oracle.lr_schedule(0.1, 0.0, 0, 1, 1.0)
    with pytest.raises(ValueError):
        oracle.lr_schedule(0.1, 0.5, -1, 1, 1.0)


# ------------------------------------------------------------------ global-norm clipping
def test_clip_scales_3_4_5_by_hand():
    """G = [3, 4]: ||G|| = 5.  clip 2.5 -> factor 0.5 -> clipped [1.5, 2.0] of norm 2.5; clip 5 and 10 -> factor 1."""
    g = [np.array([3.0, 4.0], f32), np.array([0.0, 0.0], f32), np.array([-6.0, 8.0], f32)]
    assert oracle.clip_scales(g, 2.5).tolist() == [0.5, 1.0, 0.25]
    assert oracle.clip_scales(g, 5.0).tolist() == [1.0, 1.0, 0.5]
    assert oracle.clip_scales(g, 10.0).tolist() == [1.0, 1.0, 1.0]


@pytest.mark.parametrize("bf16", [False, True])
def test_clip_scales_against_numpy_norm(bf16):
    rng = np.random.default_rng(60 + bf16)
    P, W = 10_007, 7
    vals = [(rng.normal(0, 10.0 ** rng.integers(-4, 2), P)).astype(f32) for _ in range(W)]
    if bf16:
        grads = [(v.view(np.uint32) >> 16).astype(np.uint16) for v in vals]
        vals = [(g.astype(np.uint32) << 16).view(np.float32) for g in grads]
    else:
        grads = vals
    clip = 0.5
    got = oracle.clip_scales(grads, clip)
    for k in range(W):
        norm = np.linalg.norm(vals[k].astype(np.float64))
        want = f32(clip / max(norm, clip))
        assert ulp_diff(got[k], want) <= 1
        if norm <= clip:
            assert got[k] == 1.0
        else:   # the clipped gradient has norm clip
            assert abs(np.linalg.norm(vals[k].astype(np.float64) * float(got[k])) - clip) <= 1e-6 * clip


def test_clip_invalid_and_nonfinite():
    g = [np.array([1.0, np.inf], f32)]
    assert oracle.clip_scales(g, 1.0)[0] == 0.0                     # clip / inf
    with pytest.raises(ValueError):
        oracle.clip_scales(g, 0.0)


# ------------------------------------------------------------------ clip factors of sliced gradients
def test_clip_scales_slices_3_4_12_by_hand():
    """Worker 0: G[0] = [3], G[1] = [4, 12] on two servers: ||G|| = 13 over BOTH slices (a per-slice norm would give 3
    and sqrt(160)).  clip 6.5 -> 0.5.  Worker 1: [0], [0, 1]: norm 1 -> 1."""
    off = [0, 1, 3]
    sl = [[np.array([3.0], f32), np.array([4.0, 12.0], f32)], [np.array([0.0], f32), np.array([0.0, 1.0], f32)]]
    assert oracle.clip_scales_slices(off, sl, 6.5).tolist() == [0.5, 1.0]
    assert oracle.clip_scales_slices(off, sl, 13.0).tolist() == [1.0, 1.0]
    assert oracle.clip_scales_slices(off, sl, 0.25).tolist() == [float(f32(0.25 / 13.0)), 0.25]


@pytest.mark.parametrize("bf16", [False, True])
def test_clip_scales_slices_equal_the_pinned_flat_factors_and_numpy(bf16):
    """Slices that are cuts of flat buffers (views, and separately allocated copies at odd offsets, with an empty and a
    one-element server): bit-equal to the already pinned flat oracle; numpy's norm of the concatenation."""
    rng = np.random.default_rng(70 + bf16)
    off = np.array([0, 1, 1, 4_099, 7_000, 10_007], np.int64)
    P, W = int(off[-1]), 6
    vals = [(rng.normal(0, 10.0 ** rng.integers(-3, 1), P)).astype(f32) for _ in range(W)]
    if bf16:
        grads = [(v.view(np.uint32) >> 16).astype(np.uint16) for v in vals]
        vals = [(g.astype(np.uint32) << 16).view(np.float32) for g in grads]
    else:
        grads = vals
    clip = 0.5
    want = oracle.clip_scales(grads, clip)
    views = [[g[off[j]:off[j + 1]] for j in range(off.size - 1)] for g in grads]
    assert np.array_equal(oracle.clip_scales_slices(off, views, clip), want)
    copies = []
    for k, g in enumerate(grads):
        row = []
        for j in range(off.size - 1):
            buf = np.zeros(int(off[j + 1] - off[j]) + 8, g.dtype)
            o = (k + j) % 3
            buf[o:o + int(off[j + 1] - off[j])] = g[off[j]:off[j + 1]]
            row.append(buf[o:o + int(off[j + 1] - off[j])])
        copies.append(row)
    got = oracle.clip_scales_slices(off, copies, clip)
    assert np.array_equal(got, want)
    for k in range(W):
        norm = np.linalg.norm(np.concatenate([vals[k][off[j]:off[j + 1]] for j in range(off.size - 1)]).astype(np.float64))
        assert ulp_diff(got[k], f32(clip / max(norm, clip))) <= 1


def test_clip_scales_slices_invalid():
    off = [0, 1, 3]
    sl = [[np.array([3.0], f32), None]]
    with pytest.raises(ValueError):
        oracle.clip_scales_slices(off, sl, 1.0)                      # a missing slice of a non-empty server
    sl = [[np.array([3.0], f32), np.array([4.0, 12.0], f32)]]
    with pytest.raises(ValueError):
        oracle.clip_scales_slices(off, sl, 0.0)
    assert oracle.clip_scales_slices([0, 1, 1, 3], [[sl[0][0], None, sl[0][1]]], 6.5).tolist() == [0.5]   # empty server


# ------------------------------------------------------------------ clipped async update
def test_async_with_clip_by_hand():
    """theta = [1, 1], one arrival G = [3, 4], clip 2.5, gamma 0.5: clipped G = [1.5, 2]; theta' = [0.25, 0.0]."""
    g = [np.array([3.0, 4.0], f32)]
    theta = np.array([1.0, 1.0], f32)
    sc = oracle.clip_scales(g, 2.5)
    oracle.async_apply([0, 2], g, np.array([0], np.int32), theta, gscales=sc, ema_mode=oracle.EMA_OFF, gamma_t=0.5)
    assert theta.tolist() == [0.25, 0.0]


@pytest.mark.parametrize("opt", [oracle.SGD, oracle.MOMENTUM, oracle.RMSPROP_MOM])
def test_async_gscales_power_of_two_equals_prescaled_buffers(opt):
    """Scaling by 2^-k is exact, so passing gscales must equal scaling the buffers beforehand, bit for bit, for
    every optimizer (a scale folded into gamma instead would be wrong for momentum and RMSProp)."""
    rng = np.random.default_rng(70 + opt)
    P, W = 300, 5
    theta = rng.normal(0, 0.02, P).astype(f32)
    grads = [rng.normal(0, 1e-2, P).astype(f32) for _ in range(W)]
    order = np.array([3, 0, 4, 1, 2], np.int32)
    sc = np.array([0.5, 1.0, 0.25, 0.125, 1.0], f32)                  # indexed by iteration, like gammas
    hp = dict(opt=opt, ema_mode=oracle.EMA_PRE, gamma_t=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0)
    a = [theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)]
    b = [x.copy() for x in a]
    assert oracle.async_apply([0, P], grads, order, *a, gscales=sc, **hp) == oracle.OK
    pre = [g.copy() for g in grads]
    for i, k in enumerate(order):
        pre[k] = (grads[k] * sc[i]).astype(f32)
    assert oracle.async_apply([0, P], pre, order, *b, **hp) == oracle.OK
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    if opt != oracle.SGD:       # and it is NOT the same as scaling gamma
        c = [theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)]
        oracle.async_apply([0, P], grads, order, *c, gammas=(f32(0.045) * sc).astype(f32), **{**hp, "gamma_t": 0.0})
        assert not np.array_equal(a[0], c[0])
