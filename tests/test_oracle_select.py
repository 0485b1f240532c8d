"""Pins for the oracle's first-N-of-(N+b) selection (Alg. 4 l.3-6 L148-158).

The oracle sorts (time, index) pairs with std::sort; these tests pin it to things that are not
itself: numpy's stable lexsort, exhaustive enumeration, and the properties the definition implies.
"""
import itertools

import numpy as np
import pytest

import oracle
from paper_1702_05800_b200 import synth


def lexsort_first_n(arrival, N, tags=None, t=0):
    """Independent library routine: numpy lexsort on (time, index) over eligible workers."""
    W = len(arrival)
    idx = np.arange(W)
    elig = np.isfinite(arrival)
    if tags is not None:
        elig &= (tags == t)
    idx = idx[elig]
    if len(idx) < N:
        return None, None
    times = arrival[idx] + np.float32(0.0)  # -0.0 -> +0.0, so that lexsort sees IEEE equality
    order = np.lexsort((idx, times))        # primary key: times, secondary: idx
    first = idx[order[:N]]
    return np.sort(first).astype(np.int32), float(arrival[idx[order[N - 1]]])


def test_hand_example():
    a = np.array([0.5, 2.0, 1.0], dtype=np.float32)
    st, kept, t_nth = oracle.select_first_n(a, 2, 1)
    assert st == oracle.OK and kept.tolist() == [0, 2] and t_nth == 1.0


@pytest.mark.parametrize("W", [1, 2, 3, 4, 5, 6])
def test_exhaustive_permutations(W):
    """All orderings of W distinct times, every N: kept = the N workers holding the N smallest."""
    base = np.arange(1, W + 1, dtype=np.float32) * np.float32(0.25)
    for perm in itertools.permutations(range(W)):
        a = base[list(perm)].copy()
        for N in range(1, W + 1):
            st, kept, t_nth = oracle.select_first_n(a, N, W - N)
            assert st == oracle.OK
            expect = sorted(k for k in range(W) if perm[k] < N)
            assert kept.tolist() == expect
            assert t_nth == base[N - 1]


@pytest.mark.parametrize("W", [1, 2, 3, 4, 5])
def test_exhaustive_ties(W):
    """All 3^W assignments from {0,1,2} (massive ties): brute force = stable sort by time."""
    for combo in itertools.product([0.0, 1.0, 2.0], repeat=W):
        a = np.array(combo, dtype=np.float32)
        stable = sorted(range(W), key=lambda k: (combo[k], k))
        for N in range(1, W + 1):
            st, kept, t_nth = oracle.select_first_n(a, N, W - N)
            assert st == oracle.OK
            assert kept.tolist() == sorted(stable[:N])
            assert t_nth == combo[stable[N - 1]]


def test_all_equal_times_keep_lowest_indices():
    for W, N in [(5, 4), (106, 100), (1024, 1000), (33, 1)]:
        a = np.full(W, 1.5, dtype=np.float32)
        st, kept, _ = oracle.select_first_n(a, N, W - N)
        assert st == oracle.OK and kept.tolist() == list(range(N))


def test_b0_keeps_everyone():
    rng = np.random.default_rng(1)
    for N in (1, 2, 31, 32, 33, 100, 1024):
        a = rng.lognormal(0, 0.3, N).astype(np.float32)
        st, kept, t_nth = oracle.select_first_n(a, N, 0)
        assert st == oracle.OK and kept.tolist() == list(range(N)) and t_nth == a.max()


def test_n1_is_argmin_first_on_ties():
    rng = np.random.default_rng(2)
    for W in (1, 2, 7, 64, 300):
        a = rng.integers(0, 5, W).astype(np.float32)  # many ties
        st, kept, t_nth = oracle.select_first_n(a, 1, W - 1)
        assert st == oracle.OK and kept.tolist() == [int(np.argmin(a))] and t_nth == a.min()


@pytest.mark.parametrize("seed", range(20))
def test_random_vs_lexsort_with_ties_inf_nan_tags(seed):
    rng = np.random.default_rng(100 + seed)
    W = int(rng.integers(1, 1025))
    a = rng.lognormal(0, 0.3, W).astype(np.float32)
    # force ties, zeros of both signs, negatives and non-finite values
    q = rng.integers(0, 4, W)
    a = np.where(q == 0, np.round(a * 4) / 4, a).astype(np.float32)
    for val in (np.inf, -np.inf, np.nan, 0.0, -0.0, -1.25):
        a[rng.integers(0, W, max(1, W // 50))] = val
    tags = None
    t = int(rng.integers(0, 5))
    if seed % 2:
        tags = np.where(rng.random(W) < 0.9, t, t - 1).astype(np.int32)
    for N in sorted({1, max(1, W // 2), max(1, W - 3), W}):
        st, kept, t_nth = oracle.select_first_n(a, N, W - N, tags=tags, t=t)
        exp_kept, exp_t = lexsort_first_n(a, N, tags, t)
        if exp_kept is None:
            assert st == oracle.ETOOFEW and kept is None
        else:
            assert st == oracle.OK
            assert np.array_equal(kept, exp_kept)
            assert t_nth == exp_t


def test_properties_partition_and_nesting():
    rng = np.random.default_rng(7)
    for W in (5, 55, 106, 108, 110):
        a = rng.lognormal(0, 0.25, W).astype(np.float32)
        prev = set()
        for N in range(1, W + 1):
            st, kept, t_nth = oracle.select_first_n(a, N, W - N)
            assert st == oracle.OK and len(kept) == N
            assert (np.diff(kept) > 0).all()                      # strictly ascending
            dropped = np.setdiff1d(np.arange(W), kept)
            if len(dropped):
                assert a[kept].max() <= a[dropped].min()          # nobody dropped arrived earlier
            assert t_nth == a[kept].max()
            assert prev <= set(kept.tolist())                     # kept(N) is nested in kept(N+1)
            prev = set(kept.tolist())


def test_permutation_equivariance():
    rng = np.random.default_rng(8)
    W, N = 106, 100
    a = rng.permutation(np.linspace(0.5, 3.0, W)).astype(np.float32)  # distinct
    _, kept, _ = oracle.select_first_n(a, N, W - N)
    pi = rng.permutation(W)                     # new position p holds old worker pi[p]
    _, kept_p, _ = oracle.select_first_n(a[pi].copy(), N, W - N)
    assert set(pi[kept_p].tolist()) == set(kept.tolist())


def test_too_few_and_invalid():
    a = np.array([1.0, np.inf, np.nan, 2.0], dtype=np.float32)
    st, kept, _ = oracle.select_first_n(a, 3, 1)
    assert st == oracle.ETOOFEW and kept is None
    st, kept, _ = oracle.select_first_n(a, 2, 2)
    assert st == oracle.OK and kept.tolist() == [0, 3]
    tags = np.array([3, 3, 3, 2], dtype=np.int32)     # worker 3 sent a stale gradient (t' != t)
    st, _, _ = oracle.select_first_n(a, 2, 2, tags=tags, t=3)
    assert st == oracle.ETOOFEW
    assert oracle.lib().oracle_select_first_n(None, None, 0, 1, 0, None, None) == oracle.EINVAL
    st, _, _ = oracle.select_first_n(np.zeros(0, dtype=np.float32), 0, 0)
    assert st == oracle.EINVAL


def test_negative_zero_equals_positive_zero():
    a = np.array([0.0, -0.0, 0.0, -1.0], dtype=np.float32)
    st, kept, t_nth = oracle.select_first_n(a, 2, 2)
    assert kept.tolist() == [0, 3] and t_nth == 0.0   # -0.0 at index 1 does not beat +0.0 at index 0
    a = np.array([-0.0, 0.0], dtype=np.float32)
    st, kept, _ = oracle.select_first_n(a, 1, 1)
    assert kept.tolist() == [0]
    a = np.array([0.0, -0.0], dtype=np.float32)
    st, kept, _ = oracle.select_first_n(a, 1, 1)
    assert kept.tolist() == [0]


def test_config_arrivals_shapes():
    """The synthetic arrival recipe: W finite positive fp32 values, reproducible from the seed."""
    for cfg in synth.CONFIGS.values():
        a0 = synth.arrival_times(cfg, 0)
        assert a0.dtype == np.float32 and a0.shape == (cfg.W,) and np.isfinite(a0).all() and (a0 > 0).all()
        assert np.array_equal(a0, synth.arrival_times(cfg, 0))
        assert not np.array_equal(a0, synth.arrival_times(cfg, 1))
        st, kept, _ = oracle.select_first_n(a0, cfg.N, cfg.b)
        assert st == oracle.OK and len(kept) == cfg.N
