"""GPU parity for K2 / K3 (psync_aggregate_update, psync_ema) against the CPU oracle, element by
element, at sizes spanning several tiles and a ragged tail.  PAPER.md Alg. 4 l.8-9 (L160-162), L40."""
from dataclasses import replace

import numpy as np
import pytest
import torch

import oracle
import paper_1702_05800_b200 as psync
from paper_1702_05800_b200 import synth

from _harness import ATOL_STEP, RTOL_BF16, RTOL_STEP, STATE_NAMES, Pair, assert_close, to_np

pytestmark = pytest.mark.gpu
DEV = "cuda"

BASE = synth.Config(name="unit", cfg_id=9, P=70_003, M=7, N=10, b=3, arrival_sigma=0.3, opt=synth.SGD, gamma=0.045,
                    alpha=0.9999, mu=0.9, rho=0.9, eps=1.0, steps=3)


def rtol_for(cfg):
    return RTOL_BF16 if cfg.grad_dtype == synth.BF16 else RTOL_STEP


@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
@pytest.mark.parametrize("opt", [synth.SGD, synth.MOMENTUM, synth.RMSPROP_MOM])
@pytest.mark.parametrize("ema_mode", [synth.EMA_POST, synth.EMA_PRE, synth.EMA_OFF])
def test_every_template_instance_lockstep(dtype, opt, ema_mode):
    cfg = replace(BASE, grad_dtype=dtype, opt=opt, ema_mode=ema_mode, name=f"unit_d{dtype}_o{opt}_e{ema_mode}")
    # fp32 gradients are held to the fp32 tolerance even here; bf16 inputs are widened exactly, so they too
    # meet the tight bound -- the loose 2e-3 is only the ceiling north_star allows
    Pair(cfg).run(3, lockstep=True, rtol=RTOL_STEP, atol=ATOL_STEP)


@pytest.mark.parametrize("variant", [1, 5, 6, 7])   # 5: cp.async.bulk ring; 6: 256-bit loads; 7: per-thread cp.async ring (2, 3, 4, 8 were removed)
@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
def test_every_variant(variant, dtype):
    cfg = replace(BASE, grad_dtype=dtype, opt=synth.RMSPROP_MOM, N=21, b=2, P=200_001, name=f"variant{variant}")
    Pair(cfg, variant=variant).run(2, lockstep=True)


@pytest.mark.parametrize("P", [0, 1, 3, 4, 5, 7, 8, 9, 31, 1023, 1024, 1025, 4096 + 6])
@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
def test_small_and_ragged_sizes(P, dtype):
    cfg = replace(BASE, P=P, M=min(3, max(1, P)), grad_dtype=dtype, opt=synth.MOMENTUM, name=f"small{P}")
    if P == 0:
        th = torch.zeros(0, dtype=torch.float32, device=DEV)
        step, keep = psync.make_step([0, 0], 2, 2, dtype, th, th.clone(), th.clone(), None, opt=synth.MOMENTUM,
                                     d_grads=torch.zeros(2, dtype=torch.int64, device=DEV),
                                     d_kept=torch.zeros(2, dtype=torch.int32, device=DEV))
        assert psync.psync_aggregate_update(step) == psync.PSYNC_OK
        return
    Pair(cfg).run(2, lockstep=True)


@pytest.mark.parametrize("N,b", [(1, 0), (1, 4), (2, 0), (7, 0), (8, 1), (9, 0), (16, 2), (17, 3), (100, 6)])
def test_worker_counts_cross_unroll_boundaries(N, b):
    cfg = replace(BASE, N=N, b=b, P=20_011, opt=synth.RMSPROP_MOM, name=f"N{N}b{b}")
    Pair(cfg).run(2, lockstep=True)


def test_max_workers_1024():
    cfg = replace(BASE, N=1000, b=24, P=4099, opt=synth.SGD, name="W1024")
    Pair(cfg).run(1, lockstep=True)


def _views_with_offset(P, W, dtype, offset_elems):
    """Buffers whose base is offset from the allocation by offset_elems elements (misaligned when odd)."""
    tdt = torch.float32 if dtype == synth.F32 else torch.bfloat16
    gen = torch.Generator(device=DEV)
    gen.manual_seed(99)
    out = []
    for _ in range(W):
        raw = torch.empty(P + 16, dtype=torch.float32, device=DEV).normal_(0, 1e-3, generator=gen).to(tdt)
        out.append(raw[offset_elems:offset_elems + P])
    return out


@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
@pytest.mark.parametrize("which", ["grads", "theta", "one_grad"])
def test_unaligned_pointers_take_the_scalar_path(dtype, which):
    P, N, b = 10_007, 5, 2
    W = N + b
    cfg = replace(BASE, P=P, N=N, b=b, M=1, grad_dtype=dtype, opt=synth.RMSPROP_MOM, name="unaligned")
    grads = _views_with_offset(P, W, dtype, 1 if which == "grads" else 0)
    if which == "one_grad":
        grads[3] = _views_with_offset(P, 1, dtype, 1)[0]
    theta = None
    if which == "theta":
        theta = torch.empty(P + 4, dtype=torch.float32, device=DEV).normal_(0, 0.02)[1:P + 1]
    pair = Pair(cfg, theta=theta)
    arrival = np.array([0.1, 0.2, 9.0, 0.3, 0.4, 8.0, 0.5], dtype=np.float32)   # keeps 0,1,3,4,6
    st, kept, _ = pair.gpu_step(grads, arrival)
    st_o, kept_o, _ = pair.oracle_step(grads, arrival)
    assert st == 0 and np.array_equal(kept, kept_o) and kept.tolist() == [0, 1, 3, 4, 6]
    pair.compare(RTOL_STEP, ATOL_STEP, "unaligned")


def test_exact_arithmetic_inputs_are_bit_identical():
    """Dyadic gradients, N a power of two: every fp32 partial sum is exact, so the CUDA result must
    equal the oracle bit for bit (any dropped term, wrong divisor or reordering shows)."""
    P, N, b = 50_000 + 3, 8, 2
    W = N + b
    rng = np.random.default_rng(3)
    grads = [torch.from_numpy((rng.integers(-64, 65, P) / 256.0).astype(np.float32)).to(DEV) for _ in range(W)]
    theta = torch.from_numpy((rng.integers(-512, 513, P) / 1024.0).astype(np.float32)).to(DEV)
    cfg = replace(BASE, P=P, N=N, b=b, M=3, opt=synth.SGD, gamma=0.5, alpha=0.5, name="exact")
    pair = Pair(cfg, theta=theta)
    arrival = synth.arrival_times(cfg, 0)
    pair.gpu_step(grads, arrival)
    pair.oracle_step(grads, arrival)
    assert np.array_equal(to_np(pair.ps.theta), pair.host["theta"])
    assert np.array_equal(to_np(pair.ps.ema), pair.host["ema"])


def test_dropped_buffers_are_never_read_poison():
    cfg = replace(BASE, P=30_001, N=6, b=3, opt=synth.RMSPROP_MOM, name="poison")
    arrival = synth.arrival_times(cfg, 0)
    _, kept, _ = oracle.select_first_n(arrival, cfg.N, cfg.b)
    dropped = sorted(set(range(cfg.W)) - set(kept.tolist()))
    outs = []
    for poison in (False, True):
        pair = Pair(cfg)
        grads = pair.gradients(0)
        if poison:
            for k in dropped:
                grads[k].fill_(float("nan"))
        pair.gpu_step(grads, arrival)
        outs.append([to_np(getattr(pair.ps, n)) for n in ("theta", "ema", "state0", "state1")])
    for a, b_ in zip(*outs):
        assert np.array_equal(a, b_) and np.isfinite(a).all()


def test_null_pointer_for_dropped_worker_is_fine():
    """A dropped worker's table entry may even be NULL: it is never dereferenced."""
    cfg = replace(BASE, P=5_000, N=3, b=1, M=1, name="nullptr")
    pair = Pair(cfg)
    grads = pair.gradients(0)
    arrival = np.array([0.3, 0.1, 50.0, 0.2], dtype=np.float32)
    pair.ps.set_gradients(grads)
    pair.ps.table.d_ptrs[2] = 0
    pair.ps.step(torch.from_numpy(arrival).to(DEV), cfg.gamma)
    torch.cuda.synchronize()
    pair.oracle_step(grads, arrival)
    pair.compare(RTOL_STEP, ATOL_STEP, "nullptr")


def test_bitwise_invariance_shard_layout_launch_variant_and_rerun():
    cfg = replace(BASE, P=123_457, N=13, b=2, opt=synth.RMSPROP_MOM, name="invariance")
    arrival = synth.arrival_times(cfg, 0)
    ref = None
    P = cfg.P
    layouts = [None, [0, P], [0, 1, 2, 77_777, 77_777, P]]
    # the four launch variants differ in load width (128 / 256 bit: 1024 / 2048 parameters per tile) and staging
    # (registers / cp.async.bulk ring / per-thread cp.async ring): the fixed-order fp32 sum must give the same bits in all of them.  (grid_ctas
    # is accepted and ignored by this kernel, so it is not a dimension here.)
    runs = [(lay, 0, 0) for lay in layouts] + [(None, 0, v) for v in (1, 5, 6, 7)]
    runs.append((None, 0, 0))   # the same launch again
    for lay, grid, variant in runs:
        pair = Pair(cfg, shard_off=lay, grid_ctas=grid, variant=variant)
        pair.gpu_step(pair.gradients(0), arrival)
        out = [to_np(getattr(pair.ps, n)) for n in ("theta", "ema", "state0", "state1")] + [pair.ps.d_kept.cpu().numpy()]
        if ref is None:
            ref = out
        for a, b_ in zip(ref, out):
            assert np.array_equal(a, b_), f"layout={lay} grid={grid} variant={variant}"


def test_status_not_ok_leaves_state_untouched():
    cfg = replace(BASE, P=9_001, N=4, b=1, opt=synth.RMSPROP_MOM, name="toofew")
    pair = Pair(cfg)
    before = [to_np(getattr(pair.ps, n)) for n in ("theta", "ema", "state0", "state1")]
    arrival = np.array([0.1, np.inf, np.nan, 0.2, 0.3], dtype=np.float32)
    st, _, _ = pair.gpu_step(pair.gradients(0), arrival)
    assert st == psync.PSYNC_ETOOFEW
    for a, n in zip(before, ("theta", "ema", "state0", "state1")):
        assert np.array_equal(a, to_np(getattr(pair.ps, n)))
    st_o, _, _ = pair.oracle_step(pair.gradients(0), arrival)
    assert st_o == oracle.ETOOFEW


def test_stale_tags_are_dropped():
    """Alg. 4 l.5-6: a gradient tagged t' != t is dropped even if it arrived first."""
    cfg = replace(BASE, P=6_001, N=3, b=2, name="tags")
    pair = Pair(cfg)
    grads = pair.gradients(0)
    arrival = np.array([0.01, 0.5, 0.6, 0.7, 0.02], dtype=np.float32)
    tags = np.array([6, 7, 7, 7, 7], dtype=np.int32)
    st, kept, tn = pair.gpu_step(grads, arrival, tags=tags, t=7)
    st_o, kept_o, tn_o = pair.oracle_step(grads, arrival, tags=tags, t=7)
    assert st == 0 and kept.tolist() == [1, 2, 4] == kept_o.tolist() and tn == tn_o
    pair.compare(RTOL_STEP, ATOL_STEP, "tags")


def test_psync_ema_matches_oracle_and_fused_post():
    rng = np.random.default_rng(4)
    for P in (1, 5, 4096, 100_003):
        theta = torch.from_numpy(rng.normal(0, 0.02, P).astype(np.float32)).to(DEV)
        ema = torch.from_numpy(rng.normal(0, 0.02, P).astype(np.float32)).to(DEV)
        want = to_np(ema)
        oracle.ema_update(want, to_np(theta), 0.9999)
        psync.psync_ema(ema, theta, 0.9999)
        torch.cuda.synchronize()
        assert_close(to_np(ema), want, RTOL_STEP, ATOL_STEP, f"psync_ema P={P}")
    # EMA_OFF fused step + psync_ema == EMA_POST fused step, bit for bit
    cfg = replace(BASE, P=40_001, opt=synth.MOMENTUM, name="ema_split")
    arrival = synth.arrival_times(cfg, 0)
    a = Pair(cfg)
    a.gpu_step(a.gradients(0), arrival)
    b_ = Pair(replace(cfg, ema_mode=synth.EMA_OFF))
    ema_b = b_.ps.theta.clone()
    b_.gpu_step(b_.gradients(0), arrival)
    psync.psync_ema(ema_b, b_.ps.theta, cfg.alpha)
    torch.cuda.synchronize()
    assert np.array_equal(to_np(a.ps.theta), to_np(b_.ps.theta))
    assert np.array_equal(to_np(a.ps.ema), to_np(ema_b))


def test_ema_constant_theta_closed_form_on_gpu():
    """gamma = 0: theta never moves and ema_T = alpha^T ema_0 + (1 - alpha^T) theta (north_star)."""
    P, T, alpha = 2_000, 100, 0.999
    cfg = replace(BASE, P=P, N=2, b=1, M=1, gamma=0.0, alpha=alpha, name="ema_closed")
    pair = Pair(cfg)
    theta0 = to_np(pair.ps.theta)
    pair.ps.ema.copy_(torch.from_numpy(np.random.default_rng(6).uniform(-0.1, 0.1, P).astype(np.float32)))
    ema0 = to_np(pair.ps.ema)
    grads = pair.gradients(0)
    for s in range(T):
        pair.gpu_step(grads, synth.arrival_times(cfg, s))
    assert np.array_equal(to_np(pair.ps.theta), theta0)
    a = float(np.float32(alpha))
    want = a ** T * ema0.astype(np.float64) + (1 - a ** T) * theta0.astype(np.float64)
    assert_close(to_np(pair.ps.ema), want, 1e-4, 1e-6, "ema closed form")


def test_b0_plain_mean_and_n1_earliest_on_gpu():
    cfg = replace(BASE, P=12_345, N=16, b=0, M=1, gamma=0.25, ema_mode=synth.EMA_OFF, name="b0")
    pair = Pair(cfg)
    theta0 = to_np(pair.ps.theta).astype(np.float64)
    grads = pair.gradients(0)
    pair.gpu_step(grads, synth.arrival_times(cfg, 0))
    mean = np.stack([to_np(g) for g in grads]).astype(np.float64).mean(axis=0)
    assert_close(to_np(pair.ps.theta), theta0 - float(np.float32(0.25)) * mean, RTOL_STEP, ATOL_STEP, "b=0 mean")
    cfg = replace(BASE, P=12_345, N=1, b=6, M=1, gamma=0.5, ema_mode=synth.EMA_OFF, name="n1")
    pair = Pair(cfg)
    theta0 = to_np(pair.ps.theta).astype(np.float64)
    grads = pair.gradients(0)
    arrival = synth.arrival_times(cfg, 0)
    _, kept, _ = pair.gpu_step(grads, arrival)
    k = int(np.argmin(arrival))
    assert kept.tolist() == [k]
    assert np.array_equal(to_np(pair.ps.theta), (theta0 - 0.5 * to_np(grads[k]).astype(np.float64)).astype(np.float32))


def test_permutation_invariance_on_gpu():
    cfg = replace(BASE, P=8_191, N=10, b=3, M=1, name="perm")
    arrival = np.random.default_rng(8).permutation(np.linspace(0.5, 2.5, cfg.W)).astype(np.float32)
    a = Pair(cfg)
    grads = a.gradients(0)
    _, kept_a, _ = a.gpu_step(grads, arrival)
    pi = np.random.default_rng(9).permutation(cfg.W)
    b_ = Pair(cfg)
    _, kept_b, _ = b_.gpu_step([grads[p] for p in pi], arrival[pi].copy())
    assert set(pi[kept_b].tolist()) == set(kept_a.tolist())
    assert_close(to_np(b_.ps.theta), to_np(a.ps.theta), RTOL_STEP, ATOL_STEP, "permutation")


def test_argument_errors_return_einval_and_touch_nothing():
    cfg = replace(BASE, P=1_000, N=3, b=1, M=2, opt=synth.RMSPROP_MOM, name="einval")
    pair = Pair(cfg)
    pair.ps.set_gradients(pair.gradients(0))
    before = to_np(pair.ps.theta)
    good = dict(shard_off=pair.shard_off, N=3, W=4, grad_dtype=0, theta=pair.ps.theta, ema=pair.ps.ema,
                state0=pair.ps.state0, state1=pair.ps.state1, opt=2, ema_mode=0, d_grads=pair.ps.table.d_ptrs,
                d_kept=pair.ps.d_kept, d_status=pair.ps.d_status)
    bad_cases = [dict(shard_off=[0, 600, 999]), dict(shard_off=[0, 700, 600, 1000]), dict(N=0), dict(W=2),
                 dict(W=2000, N=1500), dict(grad_dtype=5), dict(opt=3), dict(ema_mode=-1), dict(ema=None),
                 dict(state0=None), dict(state1=None), dict(d_grads=None), dict(d_kept=None), dict(variant=99),
                 dict(grid_ctas=-1)]
    for bad in bad_cases:
        kw = dict(good)
        kw.update(bad)
        step, keep = psync.make_step(**kw)
        assert psync.psync_aggregate_update(step, check=False) == psync.PSYNC_EINVAL, bad
    for removed in (2, 3, 4, 8):             # ids of tile shapes whose kernels were removed after their A/B
        step, keep = psync.make_step(**dict(good, variant=removed))
        assert psync.psync_aggregate_update(step, check=False) == psync.PSYNC_EUNSUPPORTED, removed
    torch.cuda.synchronize()
    assert np.array_equal(before, to_np(pair.ps.theta))
    assert psync.psync_ema(pair.ps.ema, pair.ps.theta, 0.9) == psync.PSYNC_OK


@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
@pytest.mark.parametrize("P,pad", [(1, 4), (7, 8), (1021, 16), (4099, 64), (50_001, 8), (50_001, 3)])
def test_guard_bands_no_out_of_bounds_access(dtype, P, pad):
    """compute-sanitizer is closed on this GPU pool, so bounds are checked by hand: every array is a slice
    of a larger allocation whose guard bands hold NaN (gradients: an out-of-bounds READ would poison the
    result and fail parity) or a sentinel (theta/state/ema: an out-of-bounds WRITE would change it).
    pad=3 makes every base pointer misaligned (scalar path); the others keep the 128-bit path."""
    N, b = 6, 2
    W = N + b
    cfg = replace(BASE, P=P, N=N, b=b, M=1, grad_dtype=dtype, opt=synth.RMSPROP_MOM, name="guard")
    tdt = torch.float32 if dtype == synth.F32 else torch.bfloat16
    gen = torch.Generator(device=DEV)
    gen.manual_seed(5)
    SENT = 12345.0

    def banded(fill, dt, draw_std):
        raw = torch.full((P + 2 * pad,), fill, dtype=dt, device=DEV)
        core = raw[pad:pad + P]
        core.copy_(torch.empty(P, dtype=torch.float32, device=DEV).normal_(0, draw_std, generator=gen).to(dt))
        return raw, core

    grads_raw, grads = zip(*[banded(float("nan"), tdt, 1e-3) for _ in range(W)])
    th_raw, th = banded(SENT, torch.float32, 0.02)
    em_raw, em = banded(SENT, torch.float32, 0.02)
    s0_raw, s0 = banded(SENT, torch.float32, 0.02)
    s0.abs_()
    s1_raw, s1 = banded(SENT, torch.float32, 1e-3)
    pair = Pair(cfg, theta=th)
    pair.ps.ema, pair.ps.state0, pair.ps.state1 = em, s0, s1
    pair.sync_host_from_gpu()
    arrival = synth.arrival_times(cfg, 0)
    st, kept, _ = pair.gpu_step(list(grads), arrival)
    st_o, kept_o, _ = pair.oracle_step(list(grads), arrival)
    assert st == 0 and np.array_equal(kept, kept_o)
    pair.compare(RTOL_STEP, ATOL_STEP, "guard bands")
    for raw in (th_raw, em_raw, s0_raw, s1_raw):
        assert bool((raw[:pad] == SENT).all()) and bool((raw[pad + P:] == SENT).all()), "write outside the array"
    for raw in grads_raw:
        assert bool(torch.isnan(raw[:pad].float()).all()) and bool(torch.isnan(raw[pad + P:].float()).all())


def test_device_rsqrt_rn_equals_frsqrt_rn_exhaustively_and_the_mirror_on_a_sample():
    """The RMSProp step's RN(1/sqrt(x)) (reading R10): the device routine (refinement of __frsqrt_rn without range
    reduction inside [2^-60, 2^60), __frsqrt_rn outside) against __frsqrt_rn on EVERY fp32 bit pattern of the fast range
    and on the rest of the positive floats by stride, and against the CPU mirror's correctly rounded rsqrt (pinned by
    exact arithmetic in tests/test_oracle_fp32_mirror.py) on a random sample."""
    from paper_1702_05800_b200 import binding as B
    bad = torch.zeros(1, dtype=torch.int64, device=DEV)
    lo, hi = 0x21800000, 0x5D800000                      # 2^-60 ... 2^60: every bit pattern (1.0e9 inputs)
    B.psync_selftest_rsqrt(bad, hi - lo, first_bits=lo)
    # the packed unchecked form (what Alg. 2's kernels run) is valid on the wider band [2^-63, 2^65): the kernel checks
    # it against __frsqrt_rn wherever its range flag stays clear -- cover the two bands outside [2^-60, 2^60) entirely
    B.psync_selftest_rsqrt(bad, lo - 0x20000000 + (1 << 15), first_bits=0x20000000 - (1 << 15))
    B.psync_selftest_rsqrt(bad, 0x60000000 - hi + (1 << 15), first_bits=hi)
    B.psync_selftest_rsqrt(bad, 1 << 16, first_bits=lo - (1 << 15))          # across the lower edge
    B.psync_selftest_rsqrt(bad, 1 << 16, first_bits=hi - (1 << 15))          # across the upper edge
    B.psync_selftest_rsqrt(bad, 1 << 24, first_bits=0)                       # zero, denormals, tiny normals
    B.psync_selftest_rsqrt(bad, 1 << 24, first_bits=0x7F000000)              # huge, +inf, NaNs
    B.psync_selftest_rsqrt(bad, 1 << 20, first_bits=0x80000000)              # -0 and negatives
    torch.cuda.synchronize()
    assert int(bad.item()) == 0
    rng = np.random.default_rng(9)
    x = np.concatenate([np.exp(rng.uniform(np.log(1e-30), np.log(1e30), 200_000)),
                        rng.uniform(0.9, 1.2, 100_000)]).astype(np.float32)
    d_y = torch.empty(x.size, dtype=torch.float32, device=DEV)
    B.psync_selftest_rsqrt(bad, x.size, d_x=torch.from_numpy(x).to(DEV), d_y=d_y)
    torch.cuda.synchronize()
    fn = oracle.mirror_lib().mirror_rsqrt_rn
    want = np.array([fn(float(v)) for v in x], dtype=np.float32)
    assert int(bad.item()) == 0 and np.array_equal(d_y.cpu().numpy().view(np.uint32), want.view(np.uint32))


def test_steps_in_flight_on_a_side_stream_keep_their_gradients_alive():
    """Eight set_gradients() / step() pairs enqueued on a side stream with no synchronisation, the caller dropping every
    reference to the gradient tensors as it goes (more pairs than the plumbing object keeps tables for): the table
    records the side stream on the pointer table and on every gradient tensor, so torch's allocator cannot hand a block
    to the next batch while a kernel may still read it.  Same bits as the same steps run one at a time."""
    cfg = replace(BASE, P=300_007, N=6, b=2, opt=synth.MOMENTUM, name="side_stream")
    arr = [synth.arrival_times(cfg, s) for s in range(8)]
    ref = Pair(cfg)
    for s in range(8):
        ref.gpu_step(ref.gradients(s), arr[s])
    pair = Pair(cfg)
    side = torch.cuda.Stream()
    d_arr = [torch.from_numpy(a).to(DEV) for a in arr]
    torch.cuda.synchronize()
    for s in range(8):
        grads = pair.gradients(s)                    # allocated and filled on the current stream
        pair.ps.set_gradients(grads)                 # the pointer table is copied on the current stream too
        side.wait_stream(torch.cuda.current_stream())
        pair.ps.step(d_arr[s], cfg.gamma, stream=side)
        assert side.cuda_stream in pair.ps.table._recorded
        del grads                                    # the only other reference is the table's
    torch.cuda.synchronize()
    for n in STATE_NAMES:
        a, b_ = getattr(ref.ps, n), getattr(pair.ps, n)
        if a is not None:
            assert np.array_equal(to_np(a), to_np(b_)), n
