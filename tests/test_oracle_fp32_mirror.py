"""Pins for the fp32 MIRROR (oracle/psync_mirror_f32.cpp -- a separate diagnostic library, not the graded oracle;
SURVEY.md section 8c; readings R9/R10): the same step in fp32 with the summation order, the five fused
multiply-adds and the correctly rounded reciprocal square root the GPU is documented to use.  Pinned by exact rational
arithmetic with one RN-even rounding per stated operation, by the hand-worked examples (dyadic, so exact in any
precision) and by closeness to the double-arithmetic oracle, which stays the graded truth."""
import json
import os
from fractions import Fraction

import mpmath
import numpy as np
import pytest

import oracle
from test_oracle_update import F, _round_f32, f32

HERE = os.path.dirname(__file__)


def rn(x):
    return F(_round_f32(x))


def rsqrt_rn(x: Fraction) -> Fraction:
    """Correctly rounded fp32 reciprocal square root of an exact rational (mpmath at 200 digits decides the rounding)."""
    with mpmath.workdps(200):
        r = 1 / mpmath.sqrt(mpmath.mpf(x.numerator) / mpmath.mpf(x.denominator))
        return F(_round_f32(Fraction(int(mpmath.floor(r * mpmath.mpf(10) ** 150)), 10 ** 150)))


def mirror_step_exact(theta, ema, s0, s1, grads, kept, N, opt, ema_mode, gamma, alpha, mu, rho, eps):
    """R9/R10 op by op in exact arithmetic, rounding once where one fp32 operation (or one FMA) is stated."""
    g_, a_, m_, r_, e_ = (F(f32(x)) for x in (gamma, alpha, mu, rho, eps))
    inv_N, oma, omr = F(f32(1.0) / f32(N)), F(f32(1.0) - f32(alpha)), F(f32(1.0) - f32(rho))
    P = len(theta)
    out = [np.array(x, dtype=f32, copy=True) for x in (theta, ema, s0, s1)]
    for i in range(P):
        S = Fraction(0)
        for k in kept:
            S = rn(S + F(grads[k][i]))                       # fp32 adds, ascending worker order, from 0
        G = rn(S * inv_N)
        th = F(theta[i])
        if opt == oracle.SGD:
            th_new = rn(th - g_ * G)                          # one FMA
        elif opt == oracle.MOMENTUM:
            v = rn(m_ * F(s0[i]) + G)                         # one FMA
            out[2][i] = f32(float(v))
            th_new = rn(th - g_ * v)                          # one FMA
        else:
            ms = rn(r_ * F(s0[i]) + rn(omr * rn(G * G)))      # mul, mul, FMA
            step = rn(rn(g_ * G) * rsqrt_rn(rn(ms + e_)))     # mul, add, rsqrt, mul
            mom = rn(m_ * F(s1[i]) + step)                    # one FMA
            out[2][i], out[3][i] = f32(float(ms)), f32(float(mom))
            th_new = rn(th - mom)
        out[0][i] = f32(float(th_new))
        if ema_mode != oracle.EMA_OFF:
            operand = th_new if ema_mode == oracle.EMA_POST else th
            out[1][i] = f32(float(rn(a_ * F(ema[i]) + rn(oma * operand))))    # mul, FMA
    return out


def test_mirror_rsqrt_is_correctly_rounded():
    """mirror_rsqrt_rn against mpmath (200 digits) on random fp32 values over the whole normal range, on values whose
    reciprocal root sits next to a rounding boundary (x = 1/m^2 rounded, m a midpoint of two floats), and exact cases."""
    fn = oracle.mirror_lib().mirror_rsqrt_rn
    rng = np.random.default_rng(77)
    xs = [f32(v) for v in np.exp(rng.uniform(np.log(1.2e-38), np.log(3e38), 3000))]
    xs += [f32(v) for v in rng.uniform(0.5, 4.0, 3000)]
    for _ in range(2000):                                   # near-midpoint cases
        y = f32(rng.uniform(0.5, 2.0))
        m = (float(y) + float(np.nextafter(y, f32(4.0)))) / 2
        x = f32(1.0 / (m * m))
        xs += [x, np.nextafter(x, f32(0)), np.nextafter(x, f32(9))]
    for x in xs:
        assert F(f32(fn(float(x)))) == rsqrt_rn(F(f32(x))), float(x)
    assert fn(4.0) == 0.5 and fn(0.25) == 2.0 and fn(1.0) == 1.0 and fn(float(2.0 ** -100)) == 2.0 ** 50


@pytest.mark.parametrize("opt", [oracle.SGD, oracle.MOMENTUM, oracle.RMSPROP_MOM])
@pytest.mark.parametrize("ema_mode", [oracle.EMA_POST, oracle.EMA_PRE])
def test_mirror_is_bit_exact_against_exact_rationals(opt, ema_mode):
    rng = np.random.default_rng(200 + 3 * opt + ema_mode)
    P, N, b = 24, 7, 2
    W = N + b
    theta = rng.normal(0, 0.02, P).astype(f32)
    grads = [rng.normal(0, 1e-3, P).astype(f32) for _ in range(W)]
    ema = (theta + rng.normal(0, 1e-3, P)).astype(f32)
    s0 = np.abs(rng.normal(0.5, 0.2, P)).astype(f32)
    s1 = rng.normal(0, 1e-3, P).astype(f32)
    hp = dict(gamma=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0)
    st, kept, _ = oracle.select_first_n(rng.lognormal(0, 0.3, W).astype(f32), N, b)
    want = mirror_step_exact(theta, ema, s0, s1, grads, kept.tolist(), N, opt, ema_mode, **hp)
    got = [theta.copy(), ema.copy(), s0.copy(), s1.copy()]
    with oracle.fp32_mirror():
        assert oracle.aggregate_update([0, 5, P], N, grads, kept, got[0], got[1], got[2] if opt else None,
                                       got[3] if opt == oracle.RMSPROP_MOM else None, opt=opt, ema_mode=ema_mode,
                                       gamma_t=hp["gamma"], alpha=hp["alpha"], mu=hp["mu"], rho=hp["rho"],
                                       eps=hp["eps"]) == oracle.OK
    n_arrays = {oracle.SGD: 2, oracle.MOMENTUM: 3, oracle.RMSPROP_MOM: 4}[opt]
    for x, y in list(zip(got, want))[:n_arrays]:
        assert np.array_equal(x, y)


def test_mirror_reproduces_the_hand_worked_examples_exactly():
    with open(os.path.join(HERE, "golden", "hand_worked_step.json")) as fh:
        g = json.load(fh)
    arr = lambda x: np.array(x, dtype=f32)                                   # noqa: E731
    grads = [arr(x) for x in g["grads"]]
    kept = np.array(g["kept"], np.int32)
    with oracle.fp32_mirror():
        th, em = arr(g["theta"]), arr(g["ema"])
        oracle.aggregate_update(g["shard_off"], g["N"], grads, kept, th, em, gamma_t=g["gamma"], alpha=g["alpha"])
        assert th.tolist() == g["sgd"]["theta"] and em.tolist() == g["sgd"]["ema_post"]
        r = g["rmsprop"]
        th, em, ms, mom = arr(g["theta"]), arr(g["ema"]), arr(r["ms"]), arr(r["mom"])
        oracle.aggregate_update(g["shard_off"], g["N"], grads, kept, th, em, ms, mom, opt=oracle.RMSPROP_MOM,
                                gamma_t=g["gamma"], alpha=g["alpha"], mu=r["mu"], rho=r["rho"], eps=r["eps"])
        assert th.tolist() == r["theta"] and ms.tolist() == r["ms_out"] and mom.tolist() == r["mom_out"]
        assert em.tolist() == r["ema_post"]
    with open(os.path.join(HERE, "golden", "hand_worked_async.json")) as fh:
        a = json.load(fh)
    with oracle.fp32_mirror():
        th, em = arr(a["theta"]), arr(a["ema"])
        oracle.async_apply([0, 2], [arr(x) for x in a["grads"]], np.array(a["order"], np.int32), th, em,
                           ema_mode=oracle.EMA_PRE, gamma_t=a["gamma"], alpha=a["alpha"])
        assert th.tolist() == a["theta_out"] and em.tolist() == a["ema_pre"]


@pytest.mark.parametrize("opt", [oracle.SGD, oracle.MOMENTUM, oracle.RMSPROP_MOM])
def test_mirror_stays_within_tolerance_of_the_double_oracle_and_is_off_by_default(opt):
    rng = np.random.default_rng(210 + opt)
    P, N, b = 5000, 100, 6
    W = N + b
    theta = rng.normal(0, 0.02, P).astype(f32)
    grads = [rng.normal(0, 1e-3, P).astype(f32) for _ in range(W)]
    kept = np.sort(rng.permutation(W)[:N]).astype(np.int32)
    hp = dict(opt=opt, gamma_t=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0)
    a = [theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)]
    m = [x.copy() for x in a]
    oracle.aggregate_update([0, P], N, grads, kept, *a, **hp)
    with oracle.fp32_mirror():
        oracle.aggregate_update([0, P], N, grads, kept, *m, **hp)
    again = [theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)]
    oracle.aggregate_update([0, P], N, grads, kept, *again, **hp)             # the switch was restored
    for x, y, z in zip(a, m, again):
        assert np.array_equal(x, z)
        assert np.all(np.abs(x.astype(np.float64) - y) <= 1e-6 + 1e-5 * np.abs(x))
    assert not np.array_equal(a[0], m[0])                                     # it really is a different arithmetic


def test_mirror_streamed_form_and_rows_agree_with_the_whole_step():
    rng = np.random.default_rng(220)
    P, N, W = 300, 9, 12
    theta = rng.normal(0, 0.02, P).astype(f32)
    grads = [rng.normal(0, 1e-3, P).astype(f32) for _ in range(W)]
    kept = np.sort(rng.permutation(W)[:N]).astype(np.int32)
    hp = dict(opt=oracle.RMSPROP_MOM, gamma_t=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0)
    with oracle.fp32_mirror():
        a = [theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)]
        oracle.aggregate_update([0, 100, P], N, grads, kept, *a, **hp)
        b_ = [theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)]
        S = np.zeros(P, np.float64)
        for k in kept:
            oracle.accumulate(S, grads[k])
        oracle.apply_sum([0, 100, P], N, S, *b_, **hp)
        c = [theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)]
        oracle.aggregate_update_rows([0, 100, P], N, grads, np.tile(kept, (2, 1)), *c, per_shard=True, **hp)
    for x, y, z in zip(a, b_, c):
        assert np.array_equal(x, y) and np.array_equal(x, z)
