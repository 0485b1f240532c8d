"""GPU parity for K1 (psync_select_first_n) against the CPU oracle: bit-exact kept lists.
PAPER.md:L130, Alg. 4 l.3-6 (L148-158)."""
import itertools

import numpy as np
import pytest
import torch

import oracle
import paper_1702_05800_b200 as psync

pytestmark = pytest.mark.gpu
DEV = "cuda"


def gpu_select(arrival, N, b, tags=None, t=0, sentinel=-7):
    d_arr = torch.from_numpy(np.ascontiguousarray(arrival, dtype=np.float32)).to(DEV)
    d_tags = None if tags is None else torch.from_numpy(tags).to(DEV)
    d_kept = torch.full((N,), sentinel, dtype=torch.int32, device=DEV)
    d_status = torch.full((1,), 12345, dtype=torch.int32, device=DEV)
    d_tn = torch.full((1,), -99.0, dtype=torch.float32, device=DEV)
    psync.psync_select_first_n(d_arr, N, b, d_kept, d_status, d_tn, d_tags, t)
    torch.cuda.synchronize()
    return int(d_status.item()), d_kept.cpu().numpy(), float(d_tn.item())


def check(arrival, N, b, tags=None, t=0):
    st_o, kept_o, tn_o = oracle.select_first_n(np.ascontiguousarray(arrival, dtype=np.float32), N, b, tags=tags, t=t)
    st_g, kept_g, tn_g = gpu_select(arrival, N, b, tags, t)
    assert st_g == st_o
    if st_o == oracle.OK:
        assert np.array_equal(kept_g, kept_o)
        assert tn_g == tn_o
    else:
        assert (kept_g == -7).all() and tn_g == -99.0   # outputs untouched on ETOOFEW


def test_exhaustive_small():
    for W in range(1, 6):
        base = np.arange(1, W + 1, dtype=np.float32) * np.float32(0.25)
        for perm in itertools.permutations(range(W)):
            for N in range(1, W + 1):
                check(base[list(perm)], N, W - N)


def test_exhaustive_ties_small():
    for W in range(1, 5):
        for combo in itertools.product([0.0, 1.0, 2.0], repeat=W):
            for N in range(1, W + 1):
                check(np.array(combo, dtype=np.float32), N, W - N)


@pytest.mark.parametrize("seed", range(30))
def test_random_with_ties_nonfinite_tags(seed):
    rng = np.random.default_rng(1000 + seed)
    W = int(rng.integers(1, 1025)) if seed % 3 else [1024, 1023, 33, 32, 31, 65, 64, 1, 2, 993][seed // 3]
    a = rng.lognormal(0, 0.3, W).astype(np.float32)
    q = rng.integers(0, 4, W)
    a = np.where(q == 0, np.round(a * 4) / 4, a).astype(np.float32)
    for val in (np.inf, -np.inf, np.nan, 0.0, -0.0, -1.25, 1e-42, -1e-42, 3.4e38):
        a[rng.integers(0, W, max(1, W // 60))] = val
    tags, t = None, int(rng.integers(0, 5))
    if seed % 2:
        tags = np.where(rng.random(W) < 0.9, t, t - 1).astype(np.int32)
    for N in sorted({1, max(1, W // 2), max(1, W - 3), max(1, W - 1), W}):
        check(a, N, W - N, tags, t)


def test_all_equal_and_b0_and_n1():
    for W, N in [(5, 4), (106, 100), (1024, 1000), (1024, 1024), (1024, 1), (33, 1), (1, 1)]:
        check(np.full(W, 1.5, dtype=np.float32), N, W - N)
    rng = np.random.default_rng(5)
    for N in (1, 31, 32, 33, 100, 1024):
        check(rng.lognormal(0, 0.3, N).astype(np.float32), N, 0)
    for W in (2, 7, 64, 300, 1024):
        check(rng.integers(0, 5, W).astype(np.float32), 1, W - 1)


def test_negative_zero_and_denormals():
    check(np.array([0.0, -0.0, 0.0, -1.0], dtype=np.float32), 2, 2)
    check(np.array([-0.0, 0.0], dtype=np.float32), 1, 1)
    check(np.array([0.0, -0.0], dtype=np.float32), 1, 1)
    check(np.array([1e-45, -1e-45, 0.0, -0.0, 1e-40], dtype=np.float32), 3, 2)
    st, kept, tn = gpu_select(np.array([-0.0, 5.0], dtype=np.float32), 1, 1)
    assert kept.tolist() == [0] and tn == 0.0 and not np.signbit(np.float32(tn))


def test_too_few_leaves_outputs_untouched():
    a = np.array([1.0, np.inf, np.nan, 2.0], dtype=np.float32)
    check(a, 3, 1)
    check(a, 2, 2)
    check(a, 2, 2, tags=np.array([3, 3, 3, 2], dtype=np.int32), t=3)


def test_paper_configs_all_steps():
    from paper_1702_05800_b200 import synth
    for cfg in synth.CONFIGS.values():
        for s in range(cfg.steps):
            check(synth.arrival_times(cfg, s), cfg.N, cfg.b)
    for cfg in synth.sweep_configs()[:8]:
        for s in range(cfg.steps):
            check(synth.arrival_times(cfg, s), cfg.N, cfg.b)


def test_host_argument_errors_enqueue_nothing():
    d = torch.zeros(8, dtype=torch.float32, device=DEV)
    k = torch.zeros(8, dtype=torch.int32, device=DEV)
    s = torch.full((1,), 77, dtype=torch.int32, device=DEV)
    L = psync.binding.lib()
    assert L.psync_select_first_n(d.data_ptr(), None, 0, 0, 1, k.data_ptr(), None, s.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_select_first_n(d.data_ptr(), None, 0, 1, -1, k.data_ptr(), None, s.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_select_first_n(d.data_ptr(), None, 0, 1000, 25, k.data_ptr(), None, s.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_select_first_n(None, None, 0, 1, 1, k.data_ptr(), None, s.data_ptr(), None) == psync.PSYNC_EINVAL
    torch.cuda.synchronize()
    assert int(s.item()) == 77
