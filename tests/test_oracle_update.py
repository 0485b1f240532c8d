"""Pins for the oracle's aggregate + update + EMA (Alg. 4 l.8-9, L160-162; L40).

Nothing here re-calls the oracle to check the oracle: the expected values come from the paper's
equations worked by hand (tests/golden/hand_worked_step.json), numpy's own mean, exact rational
arithmetic (fractions.Fraction; mpmath for the square root), and closed forms.
"""
import json
import os
from fractions import Fraction

import mpmath
import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "hand_worked_step.json")
f32 = np.float32


def ulp_diff(a, b):
    """Distance in fp32 units-in-the-last-place between two float32 arrays (same sign assumed near 0)."""
    ia = np.asarray(a, dtype=np.float32).view(np.int32).astype(np.int64)
    ib = np.asarray(b, dtype=np.float32).view(np.int32).astype(np.int64)
    ia = np.where(ia < 0, -(ia & 0x7FFFFFFF), ia)
    ib = np.where(ib < 0, -(ib & 0x7FFFFFFF), ib)
    return np.abs(ia - ib)


def _round_f32(x: Fraction) -> np.float32:
    """Exact RN-even rounding of a Fraction to fp32 (handles normals and subnormals)."""
    if x == 0:
        return f32(0.0)
    sign = -1 if x < 0 else 1
    ax = abs(x)
    e = ax.numerator.bit_length() - ax.denominator.bit_length()
    if Fraction(2) ** e > ax:
        e -= 1
    e = max(e, -126)                       # subnormal exponent floor
    q = ax / Fraction(2) ** (e - 23)       # significand in units of the last place
    n = q.numerator // q.denominator
    rem = q - n
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and (n & 1)):
        n += 1
    val = Fraction(n) * Fraction(2) ** (e - 23)
    return f32(sign * float(val))          # val has <= 25 significant bits: float() is exact


def F(x):
    return Fraction(float(x))


def coeffs(N, alpha=0.0, rho=0.0):
    """The real numbers both sides multiply by (reading R8): formed in fp32."""
    return F(f32(1.0) / f32(N)), F(f32(1.0) - f32(alpha)), F(f32(1.0) - f32(rho))


# ------------------------------------------------------------------ hand-worked example (golden)
def _load():
    with open(GOLDEN) as fh:
        return json.load(fh)


def _arr(x):
    return np.array(x, dtype=np.float32)


def test_golden_hand_worked_sgd_ema_post_and_pre():
    g = _load()
    grads = [_arr(x) for x in g["grads"]]
    st, kept, t_nth = oracle.select_first_n(_arr(g["arrival"]), g["N"], g["b"])
    assert st == oracle.OK and kept.tolist() == g["kept"] and t_nth == g["t_nth"]
    for mode, key in ((oracle.EMA_POST, "ema_post"), (oracle.EMA_PRE, "ema_pre")):
        theta, ema = _arr(g["theta"]), _arr(g["ema"])
        st = oracle.aggregate_update(g["shard_off"], g["N"], grads, kept, theta, ema, opt=oracle.SGD,
                                     ema_mode=mode, gamma_t=g["gamma"], alpha=g["alpha"])
        assert st == oracle.OK
        assert theta.tolist() == g["sgd"]["theta"]
        assert ema.tolist() == g["sgd"][key]
    theta, ema = _arr(g["theta"]), _arr(g["ema"])
    oracle.aggregate_update(g["shard_off"], g["N"], grads, kept, theta, ema, opt=oracle.SGD,
                            ema_mode=oracle.EMA_OFF, gamma_t=g["gamma"], alpha=g["alpha"])
    assert theta.tolist() == g["sgd"]["theta"] and ema.tolist() == g["ema"]


def test_golden_hand_worked_momentum():
    g = _load()
    m = g["momentum"]
    grads = [_arr(x) for x in g["grads"]]
    kept = np.array(g["kept"], dtype=np.int32)
    theta, ema, v = _arr(g["theta"]), _arr(g["ema"]), _arr(m["v"])
    st = oracle.aggregate_update(g["shard_off"], g["N"], grads, kept, theta, ema, state0=v, opt=oracle.MOMENTUM,
                                 gamma_t=g["gamma"], alpha=g["alpha"], mu=m["mu"])
    assert st == oracle.OK
    assert v.tolist() == m["v_out"] and theta.tolist() == m["theta"] and ema.tolist() == m["ema_post"]


def test_golden_hand_worked_rmsprop():
    g = _load()
    r = g["rmsprop"]
    grads = [_arr(x) for x in g["grads"]]
    kept = np.array(g["kept"], dtype=np.int32)
    theta, ema, ms, mom = _arr(g["theta"]), _arr(g["ema"]), _arr(r["ms"]), _arr(r["mom"])
    st = oracle.aggregate_update(g["shard_off"], g["N"], grads, kept, theta, ema, state0=ms, state1=mom,
                                 opt=oracle.RMSPROP_MOM, gamma_t=g["gamma"], alpha=g["alpha"], mu=r["mu"],
                                 rho=r["rho"], eps=r["eps"])
    assert st == oracle.OK
    assert ms.tolist() == r["ms_out"] and mom.tolist() == r["mom_out"]
    assert theta.tolist() == r["theta"] and ema.tolist() == r["ema_post"]


def test_golden_dropped_worker_is_never_read():
    """Poison: the dropped buffer full of NaN/Inf changes nothing, bit for bit (L130: 'dropped')."""
    g = _load()
    grads = [_arr(x) for x in g["grads"]]
    grads[1][:] = [np.nan, np.inf]
    kept = np.array(g["kept"], dtype=np.int32)
    theta, ema = _arr(g["theta"]), _arr(g["ema"])
    oracle.aggregate_update(g["shard_off"], g["N"], grads, kept, theta, ema, gamma_t=g["gamma"], alpha=g["alpha"])
    assert theta.tolist() == g["sgd"]["theta"] and ema.tolist() == g["sgd"]["ema_post"]


# ------------------------------------------------------------------ special cases vs library routines
def _rand_case(rng, P, W, bf16=False):
    theta = rng.normal(0, 0.02, P).astype(f32)
    grads = [rng.normal(0, 1e-3, P).astype(f32) for _ in range(W)]
    if bf16:
        grads = [to_bf16_bits(x) for x in grads]
    return theta, grads


def to_bf16_bits(x):
    """fp32 -> bf16 bit patterns, round-to-nearest-even (input preparation, not method arithmetic)."""
    u = x.astype(f32).view(np.uint32).astype(np.uint64)
    r = ((u + 0x7FFF + ((u >> 16) & 1)) >> 16).astype(np.uint16)
    return r


def bf16_bits_to_f32(h):
    return (h.astype(np.uint32) << 16).view(f32)


def test_b0_is_plain_mean_numpy():
    """b = 0: theta' = theta - gamma * mean_k G_k, with numpy's float64 mean as the library routine."""
    rng = np.random.default_rng(3)
    P, N = 1000, 16                       # N a power of two: 1/N exact, so only fp32 storage rounding remains
    theta, grads = _rand_case(rng, P, N)
    st, kept, _ = oracle.select_first_n(rng.lognormal(0, 0.3, N).astype(f32), N, 0)
    th = theta.copy()
    oracle.aggregate_update([0, P], N, grads, kept, th, ema_mode=oracle.EMA_OFF, gamma_t=0.25)
    expect = (theta.astype(np.float64) - 0.25 * np.stack(grads).astype(np.float64).mean(axis=0)).astype(f32)
    assert ulp_diff(th, expect).max() <= 1
    assert (ulp_diff(th, expect) == 0).mean() > 0.99


def test_n1_applies_only_the_earliest_worker():
    rng = np.random.default_rng(4)
    P, W = 257, 7
    theta, grads = _rand_case(rng, P, W)
    arrival = rng.lognormal(0, 0.3, W).astype(f32)
    st, kept, _ = oracle.select_first_n(arrival, 1, W - 1)
    k = int(np.argmin(arrival))
    assert kept.tolist() == [k]
    th = theta.copy()
    oracle.aggregate_update([0, 100, P], 1, grads, kept, th, ema_mode=oracle.EMA_OFF, gamma_t=0.5)
    expect = (theta.astype(np.float64) - 0.5 * grads[k].astype(np.float64)).astype(f32)
    assert np.array_equal(th, expect)     # one product and one subtraction of exact doubles: bit-exact


def test_permutation_invariance_with_arrival_times():
    rng = np.random.default_rng(5)
    P, N, b = 300, 10, 3
    W = N + b
    theta, grads = _rand_case(rng, P, W)
    arrival = rng.permutation(np.linspace(0.5, 2.5, W)).astype(f32)
    _, kept, _ = oracle.select_first_n(arrival, N, b)
    th1 = theta.copy()
    oracle.aggregate_update([0, P], N, grads, kept, th1, ema_mode=oracle.EMA_OFF, gamma_t=0.045)
    pi = rng.permutation(W)
    _, kept2, _ = oracle.select_first_n(arrival[pi].copy(), N, b)
    th2 = theta.copy()
    oracle.aggregate_update([0, P], N, [grads[p] for p in pi], kept2, th2, ema_mode=oracle.EMA_OFF, gamma_t=0.045)
    assert set(pi[kept2].tolist()) == set(kept.tolist())
    assert ulp_diff(th1, th2).max() <= 1  # double sums in another order: at most the last fp32 bit moves


def test_shard_layout_invariance_and_streamed_form():
    rng = np.random.default_rng(6)
    P, N, W = 1237, 5, 6
    theta, grads = _rand_case(rng, P, W)
    kept = np.array([0, 1, 3, 4, 5], dtype=np.int32)
    kw = dict(opt=oracle.RMSPROP_MOM, gamma_t=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0)
    outs = []
    for off in ([0, P], [0, 1, 2, 700, 700, P], list(range(0, P, 97)) + [P]):
        th, ema, ms, mom = theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)
        assert oracle.aggregate_update(off, N, grads, kept, th, ema, ms, mom, **kw) == oracle.OK
        outs.append((th, ema, ms, mom))
    for o in outs[1:]:
        for a, b in zip(outs[0], o):
            assert np.array_equal(a, b)
    # streamed form (accumulate one kept worker at a time, then apply) is bit-identical
    S = np.zeros(P, np.float64)
    for k in kept:
        assert oracle.accumulate(S, grads[k]) == oracle.OK
    th, ema, ms, mom = theta.copy(), theta.copy(), np.ones(P, f32), np.zeros(P, f32)
    assert oracle.apply_sum([0, 500, P], N, S, th, ema, ms, mom, **kw) == oracle.OK
    for a, b in zip(outs[0], (th, ema, ms, mom)):
        assert np.array_equal(a, b)


def test_invalid_arguments():
    P = 8
    theta = np.zeros(P, f32)
    grads = [np.zeros(P, f32)] * 3
    kept = np.array([0, 1], dtype=np.int32)
    assert oracle.aggregate_update([0, 4, 7], 2, grads, kept, theta, ema_mode=oracle.EMA_OFF) == oracle.EINVAL
    assert oracle.aggregate_update([0, 5, 4, P], 2, grads, kept, theta, ema_mode=oracle.EMA_OFF) == oracle.EINVAL
    assert oracle.aggregate_update([0, P], 2, grads, kept, theta, ema_mode=oracle.EMA_POST) == oracle.EINVAL
    assert oracle.aggregate_update([0, P], 2, grads, kept, theta, ema_mode=oracle.EMA_OFF,
                                   opt=oracle.MOMENTUM) == oracle.EINVAL
    bad = np.array([0, 3], dtype=np.int32)
    assert oracle.aggregate_update([0, P], 2, grads, bad, theta, ema_mode=oracle.EMA_OFF) == oracle.EINVAL
    assert np.array_equal(theta, np.zeros(P, f32))


# ------------------------------------------------------------------ exact rational brute force, P <= 64
def exact_step(theta, ema, s0, s1, grads, kept, N, opt, ema_mode, gamma, alpha, mu, rho, eps):
    """Alg. 4 l.8-9 in exact arithmetic on the exact fp32 inputs; returns fp32-rounded new arrays.
    Written independently in Python from DESIGN.md's equations; sqrt via mpmath at 200 digits."""
    inv_N, oma, omr = coeffs(N, alpha, rho)
    P = len(theta)
    out = [np.empty(P, f32) for _ in range(4)]
    for i in range(P):
        S = sum((F(grads[k][i]) for k in kept), Fraction(0))
        G = S * inv_N
        th = F(theta[i])
        if opt == oracle.SGD:
            th_new = th - F(f32(gamma)) * G
            n0 = n1 = None
        elif opt == oracle.MOMENTUM:
            v = F(f32(mu)) * F(s0[i]) + G
            th_new = th - F(f32(gamma)) * v
            n0, n1 = v, None
        else:
            ms = F(f32(rho)) * F(s0[i]) + omr * G * G
            with mpmath.workdps(200):
                root = mpmath.sqrt(mpmath.mpf(ms.numerator) / mpmath.mpf(ms.denominator) + mpmath.mpf(float(f32(eps))))
                step = mpmath.mpf(float(f32(gamma))) * (mpmath.mpf(G.numerator) / mpmath.mpf(G.denominator)) / root
                # a 200-digit decimal is exact enough to be treated as a rational for fp32 rounding
                step = Fraction(int(mpmath.floor(step * mpmath.mpf(10) ** 150)), 10 ** 150)
            mom = F(f32(mu)) * F(s1[i]) + step
            th_new = th - mom
            n0, n1 = ms, mom
        th_f = _round_f32(th_new)
        out[0][i] = th_f
        if n0 is not None:
            out[2][i] = _round_f32(n0)
        if n1 is not None:
            out[3][i] = _round_f32(n1)
        if ema_mode != oracle.EMA_OFF:
            operand = F(th_f) if ema_mode == oracle.EMA_POST else th
            out[1][i] = _round_f32(F(f32(alpha)) * F(ema[i]) + oma * operand)
    return out


@pytest.mark.parametrize("opt", [oracle.SGD, oracle.MOMENTUM, oracle.RMSPROP_MOM])
@pytest.mark.parametrize("ema_mode", [oracle.EMA_POST, oracle.EMA_PRE])
@pytest.mark.parametrize("bf16", [False, True])
def test_exact_rational_brute_force(opt, ema_mode, bf16):
    rng = np.random.default_rng(10 + opt * 7 + ema_mode * 3 + bf16)
    P, N, b = 64, 7, 2
    W = N + b
    theta, grads = _rand_case(rng, P, W, bf16=bf16)
    gvals = [bf16_bits_to_f32(g) for g in grads] if bf16 else grads
    ema = (theta + rng.normal(0, 1e-3, P)).astype(f32)
    s0 = np.abs(rng.normal(0.5, 0.2, P)).astype(f32)
    s1 = rng.normal(0, 1e-3, P).astype(f32)
    hp = dict(gamma=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0)
    for step in range(3):                 # lock-step: both sides start each step from the same stored state
        arrival = rng.lognormal(0, 0.3, W).astype(f32)
        st, kept, _ = oracle.select_first_n(arrival, N, b)
        exp = exact_step(theta, ema, s0, s1, gvals, kept.tolist(), N, opt, ema_mode, **hp)
        th, em, a0, a1 = theta.copy(), ema.copy(), s0.copy(), s1.copy()
        st = oracle.aggregate_update([0, 13, 13, 40, P], N, grads, kept, th, em,
                                     a0 if opt != oracle.SGD else None, a1 if opt == oracle.RMSPROP_MOM else None,
                                     opt=opt, ema_mode=ema_mode, gamma_t=hp["gamma"], alpha=hp["alpha"],
                                     mu=hp["mu"], rho=hp["rho"], eps=hp["eps"])
        assert st == oracle.OK
        pairs = [(th, exp[0]), (em, exp[1])]
        if opt != oracle.SGD:
            pairs.append((a0, exp[2]))
        if opt == oracle.RMSPROP_MOM:
            pairs.append((a1, exp[3]))
        for got, want in pairs:
            d = ulp_diff(got, want)
            # double arithmetic then one fp32 rounding vs exact then one rounding: equal except for
            # rare double-rounding cases, which move the last bit only
            assert d.max() <= 1 and (d == 0).mean() >= 0.95
        theta, ema, s0, s1 = th, em, a0, a1


def test_coefficient_reading_r8_is_within_tolerance_of_decimal_coefficients():
    """1-alpha formed in fp32 (R8) vs the decimal 1-0.9999: the EMA differs far below 1e-5 relative."""
    rng = np.random.default_rng(12)
    P = 64
    theta = rng.normal(0, 0.02, P).astype(f32)
    ema = (theta + rng.normal(0, 1e-3, P)).astype(f32)
    e = ema.copy()
    oracle.ema_update(e, theta, 0.9999)
    dec = Fraction(9999, 10000)
    want = np.array([float(dec * F(ema[i]) + (1 - dec) * F(theta[i])) for i in range(P)])
    assert np.allclose(e, want, rtol=1e-6, atol=1e-9)


# ------------------------------------------------------------------ closed forms
def _run_const(opt, T, g, theta0, N=4, **hp):
    P = len(theta0)
    grads = [np.full(P, g, f32)] * N
    kept = np.arange(N, dtype=np.int32)
    th, ema = theta0.copy(), theta0.copy()
    s0 = np.full(P, hp.pop("ms0", 0.0), f32)
    s1 = np.zeros(P, f32)
    for _ in range(T):
        oracle.aggregate_update([0, P], N, grads, kept, th, ema, s0 if opt != oracle.SGD else None,
                                s1 if opt == oracle.RMSPROP_MOM else None, opt=opt, **hp)
    return th, ema, s0, s1


def test_closed_form_sgd_constant_gradient():
    theta0 = np.linspace(-1, 1, 33).astype(f32)
    T, g, gamma = 50, 0.125, 0.0625       # dyadic: every step is exact
    th, *_ = _run_const(oracle.SGD, T, g, theta0, gamma_t=gamma, alpha=0.5)
    assert np.array_equal(th, (theta0.astype(np.float64) - T * gamma * g).astype(f32))
    th, *_ = _run_const(oracle.SGD, 5, g, theta0, gamma_t=0.0, alpha=0.5)
    assert np.array_equal(th, theta0)     # gamma = 0 leaves theta bit-unchanged


def test_closed_form_momentum_constant_gradient():
    theta0 = np.linspace(-1, 1, 33).astype(f32)
    T, g, gamma, mu = 30, 1e-3, 0.01, 0.9
    th, _, v, _ = _run_const(oracle.MOMENTUM, T, g, theta0, gamma_t=gamma, alpha=0.5, mu=mu)
    g_, mu_, gamma_ = float(f32(g)), float(f32(mu)), float(f32(gamma))
    v_T = g_ * (1 - mu_ ** T) / (1 - mu_)
    disp = gamma_ * g_ * sum((1 - mu_ ** s) / (1 - mu_) for s in range(1, T + 1))
    assert np.allclose(v, v_T, rtol=T * 2.0 ** -23, atol=0)
    assert np.allclose(th, theta0.astype(np.float64) - disp, rtol=0, atol=T * 2.0 ** -24 * 1.0)


def test_closed_form_rmsprop_second_moment():
    theta0 = np.zeros(17, f32)
    T, g, rho = 25, 0.5, 0.9
    _, _, ms, _ = _run_const(oracle.RMSPROP_MOM, T, g, theta0, gamma_t=0.01, alpha=0.5, mu=0.0, rho=rho, eps=1.0,
                             ms0=2.0)
    rho_ = float(f32(rho))
    omr = float(f32(1.0) - f32(rho))
    # ms_T = rho^T ms_0 + (1-rho) g^2 (1-rho^T)/(1-rho), with the fp32-formed (1-rho) of reading R8
    want = rho_ ** T * 2.0 + omr * g * g * (1 - rho_ ** T) / (1 - rho_)
    assert np.allclose(ms, want, rtol=T * 2.0 ** -23, atol=0)


def test_reduction_momentum_mu0_is_sgd_and_rmsprop_rho1_is_sgd():
    rng = np.random.default_rng(13)
    P, N, W = 200, 6, 8
    theta, grads = _rand_case(rng, P, W)
    kept = np.array([0, 2, 3, 4, 6, 7], dtype=np.int32)
    ref = theta.copy()
    oracle.aggregate_update([0, P], N, grads, kept, ref, ema_mode=oracle.EMA_OFF, opt=oracle.SGD, gamma_t=0.045)
    th, v = theta.copy(), rng.normal(0, 1, P).astype(f32)
    oracle.aggregate_update([0, P], N, grads, kept, th, state0=v, ema_mode=oracle.EMA_OFF, opt=oracle.MOMENTUM,
                            gamma_t=0.045, mu=0.0)
    assert ulp_diff(th, ref).max() <= 1   # v is rounded to fp32 storage but theta uses the unrounded v
    assert np.array_equal(th, ref)
    # rho = 1, ms0 = 0, eps = 1, mu = 0: ms stays 0, sqrt(0 + 1) = 1, mom = gamma G  ->  SGD
    th, ms, mom = theta.copy(), np.zeros(P, f32), rng.normal(0, 1, P).astype(f32)
    oracle.aggregate_update([0, P], N, grads, kept, th, state0=ms, state1=mom, ema_mode=oracle.EMA_OFF,
                            opt=oracle.RMSPROP_MOM, gamma_t=0.045, mu=0.0, rho=1.0, eps=1.0)
    assert np.array_equal(ms, np.zeros(P, f32))
    assert np.array_equal(th, ref)


def test_rmsprop_mu0_single_step_vs_library_sqrt():
    rng = np.random.default_rng(14)
    P, N = 100, 4
    theta, grads = _rand_case(rng, P, N)
    kept = np.arange(N, dtype=np.int32)
    ms0 = np.abs(rng.normal(1, 0.1, P)).astype(f32)
    th, ms, mom = theta.copy(), ms0.copy(), np.zeros(P, f32)
    oracle.aggregate_update([0, P], N, grads, kept, th, state0=ms, state1=mom, ema_mode=oracle.EMA_OFF,
                            opt=oracle.RMSPROP_MOM, gamma_t=0.045, mu=0.0, rho=0.9, eps=1.0)
    G = np.stack(grads).astype(np.float64).sum(0) * 0.25
    ms_w = float(f32(0.9)) * ms0.astype(np.float64) + float(f32(1) - f32(0.9)) * G * G
    th_w = theta.astype(np.float64) - float(f32(0.045)) * G / np.sqrt(ms_w + 1.0)
    assert ulp_diff(ms, ms_w.astype(f32)).max() <= 1
    assert ulp_diff(th, th_w.astype(f32)).max() <= 1


# ------------------------------------------------------------------ EMA
def test_ema_constant_theta_closed_form():
    """theta constant (zero gradients): ema_T = alpha^T ema_0 + (1 - alpha^T) theta (north_star)."""
    rng = np.random.default_rng(15)
    P, T, alpha = 50, 200, 0.999
    theta = rng.uniform(-0.1, 0.1, P).astype(f32)
    ema0 = rng.uniform(-0.1, 0.1, P).astype(f32)
    zero = [np.zeros(P, f32)] * 3
    kept = np.array([0, 1], dtype=np.int32)
    for mode in (oracle.EMA_POST, oracle.EMA_PRE):
        th, ema = theta.copy(), ema0.copy()
        for _ in range(T):
            oracle.aggregate_update([0, P], 2, zero, kept, th, ema, ema_mode=mode, gamma_t=0.1, alpha=alpha)
        assert np.array_equal(th, theta)
        a = float(f32(alpha))
        # with the fp32-formed (1-alpha) the fixed point is theta*(1-alpha)_f32/(1-alpha_f32) ~ theta(1 +- 6e-5)
        oma = float(f32(1) - f32(alpha))
        fix = theta.astype(np.float64) * oma / (1 - a)
        want = a ** T * ema0.astype(np.float64) + (1 - a ** T) * fix
        assert np.allclose(ema, want, rtol=0, atol=T * 2.0 ** -24 * 0.1)
        want_ideal = a ** T * ema0.astype(np.float64) + (1 - a ** T) * theta.astype(np.float64)
        assert np.allclose(ema, want_ideal, rtol=1e-4, atol=1e-6)
    e = ema0.copy()
    for _ in range(T):
        oracle.ema_update(e, theta, alpha)
    assert np.array_equal(e, ema)         # the standalone EMA call is the same recurrence


def test_ema_alpha_edge_cases():
    rng = np.random.default_rng(16)
    theta = rng.normal(0, 1, 40).astype(f32)
    ema0 = rng.normal(0, 1, 40).astype(f32)
    e = ema0.copy()
    oracle.ema_update(e, theta, 1.0)
    assert np.array_equal(e, ema0)        # alpha = 1: unchanged
    oracle.ema_update(e, theta, 0.0)
    assert np.array_equal(e, theta)       # alpha = 0: ema = theta


def test_ema_post_equals_off_then_standalone_ema():
    rng = np.random.default_rng(17)
    P, N = 90, 3
    theta, grads = _rand_case(rng, P, N)
    kept = np.arange(N, dtype=np.int32)
    th1, e1 = theta.copy(), theta.copy()
    oracle.aggregate_update([0, P], N, grads, kept, th1, e1, ema_mode=oracle.EMA_POST, gamma_t=0.1, alpha=0.99)
    th2, e2 = theta.copy(), theta.copy()
    oracle.aggregate_update([0, P], N, grads, kept, th2, None, ema_mode=oracle.EMA_OFF, gamma_t=0.1, alpha=0.99)
    oracle.ema_update(e2, th2, 0.99)
    assert np.array_equal(th1, th2) and np.array_equal(e1, e2)


def test_ema_pre_is_post_shifted_by_one_step():
    """Reading R3: with ema(-1) = theta(0), PRE after step t+1 equals POST after step t."""
    rng = np.random.default_rng(18)
    P, N, T = 30, 2, 6
    theta0 = rng.normal(0, 0.02, P).astype(f32)
    gs = [[rng.normal(0, 1e-2, P).astype(f32) for _ in range(N)] for _ in range(T)]
    kept = np.arange(N, dtype=np.int32)
    thA, eA = theta0.copy(), theta0.copy()      # POST
    thB, eB = theta0.copy(), theta0.copy()      # PRE
    post_hist = []
    for t in range(T):
        oracle.aggregate_update([0, P], N, gs[t], kept, thA, eA, ema_mode=oracle.EMA_POST, gamma_t=0.1, alpha=0.9)
        post_hist.append(eA.copy())
    # PRE folds theta(0) once more at t=0 (a no-op when ema = theta(0)): compare from there on
    for t in range(T):
        oracle.aggregate_update([0, P], N, gs[t], kept, thB, eB, ema_mode=oracle.EMA_PRE, gamma_t=0.1, alpha=0.9)
        if t >= 1:
            assert ulp_diff(eB, post_hist[t - 1]).max() <= 1
    assert np.array_equal(thA, thB)


# ------------------------------------------------------------------ exact-arithmetic aggregate
def test_exact_inputs_sum_is_order_independent():
    """Gradients that are small integers / 2^k with N a power of two: every partial sum is exact in
    fp32 and in double, so the result is the same for ANY summation order and precision."""
    rng = np.random.default_rng(19)
    P, N = 500, 8
    grads = [(rng.integers(-64, 65, P) / 256.0).astype(f32) for _ in range(N)]
    theta = (rng.integers(-512, 513, P) / 1024.0).astype(f32)
    kept = np.arange(N, dtype=np.int32)
    th = theta.copy()
    oracle.aggregate_update([0, P], N, grads, kept, th, ema_mode=oracle.EMA_OFF, gamma_t=0.5)
    want = theta - f32(0.5) * (np.sum(np.stack(grads), axis=0, dtype=f32) * f32(0.125))
    assert np.array_equal(th, want.astype(f32))
