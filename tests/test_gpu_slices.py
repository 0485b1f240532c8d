"""GPU parity for the shard-aware kernel (K2s): the per-(worker, server) slice layout PSYNC_GRADS_SLICES -- what
parameter server j RECEIVES, Alg. 4 as the program of one server (theta[j] owned by server j,
L42) -- and the (server, tile) work list, against the CPU oracle through the C ABI.  theta / state / ema within
north_star's lock-step tolerance of oracle.aggregate_update_slices; bit-identity with the flat kernel is a property
checked at any size; the full-size cfg3 case compares EVERY element."""
from dataclasses import replace

import numpy as np
import pytest
import torch

import oracle
import paper_1702_05800_b200 as psync
from paper_1702_05800_b200 import synth

from _harness import ATOL_STEP, RTOL_BF16, RTOL_STEP, STATE_NAMES, assert_close, to_np

pytestmark = pytest.mark.gpu
DEV = "cuda"

BASE = synth.Config(name="slices", cfg_id=14, P=70_003, M=7, N=10, b=3, arrival_sigma=0.3, opt=synth.SGD,
                    gamma=0.045, alpha=0.9999, mu=0.9, rho=0.9, eps=1.0, steps=3)


def cut_slices(flat, off, offset_of=None):
    """Separately allocated copies of flat[off[j]:off[j+1]], slice (k, j) placed `offset_of(k, j)` elements after an
    allocation boundary (0 = as the allocator gives it: 512-byte aligned)."""
    out = []
    for k, g in enumerate(flat):
        row = []
        for j in range(len(off) - 1):
            lo, hi = int(off[j]), int(off[j + 1])
            o = 0 if offset_of is None else int(offset_of(k, j))
            buf = torch.empty(hi - lo + o + 16, dtype=g.dtype, device=g.device)
            view = buf[o:o + hi - lo]
            view.copy_(g[lo:hi])
            row.append(view)
        out.append(row)
    return out


def np_slices(slices):
    return [[None if t is None else synth.as_numpy_grad(t) for t in row] for row in slices]


class SlicesPair:
    """One parameter-server state on the GPU and on the host, stepped from per-(worker, server) slices."""

    def __init__(self, cfg, shard_off=None, state_misalign=0):
        self.cfg = cfg
        self.off = synth.shard_offsets(cfg) if shard_off is None else np.asarray(shard_off, dtype=np.int64)
        self.M = self.off.size - 1

        def place(t):
            if t is None or not state_misalign:
                return t
            buf = torch.empty(t.numel() + 8, dtype=t.dtype, device=DEV)
            view = buf[state_misalign:state_misalign + t.numel()]
            view.copy_(t)
            return view

        self.theta = place(synth.init_theta(cfg, DEV))
        s0, s1 = synth.init_state(cfg, DEV)
        self.state0, self.state1 = place(s0), place(s1)
        self.ema = place(self.theta.clone()) if cfg.ema_mode != synth.EMA_OFF else None
        self.d_off = torch.from_numpy(self.off).to(DEV)
        self.d_tiles = psync.psync_shard_worklist(self.d_off, cfg.grad_dtype)
        self.host = {n: to_np(getattr(self, n)) for n in STATE_NAMES}

    def make_step(self, table, d_kept, d_status=None, per_shard=False, d_n_kept=None, layout=psync.PSYNC_GRADS_SLICES,
                  variant=0):
        cfg = self.cfg
        return psync.make_step(self.off, cfg.N, cfg.W, table.grad_dtype, self.theta, self.ema, self.state0, self.state1,
                               opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu,
                               rho=cfg.rho, eps=cfg.eps, d_grads=table.d_ptrs, d_kept=d_kept, d_status=d_status,
                               per_shard=per_shard, d_shard_off=self.d_off, d_n_kept=d_n_kept, grad_layout=layout,
                               d_tile_start=self.d_tiles, variant=variant)

    def oracle(self, slices, kept, per_shard=False, n_kept=None, status=None):
        cfg, h = self.cfg, self.host
        rc = oracle.aggregate_update_slices(self.off, cfg.N, np_slices(slices), kept, h["theta"], h["ema"], h["state0"],
                                            h["state1"], per_shard=per_shard, n_kept=n_kept, status=status, opt=cfg.opt,
                                            ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu,
                                            rho=cfg.rho, eps=cfg.eps)
        assert rc == oracle.OK

    def compare_and_sync(self, what, rtol=RTOL_STEP):
        for n in STATE_NAMES:
            g = getattr(self, n)
            if g is not None:
                assert_close(to_np(g), self.host[n], rtol, ATOL_STEP, f"{what} {n}")
                self.host[n] = to_np(g)

    def step_first_n(self, step, offset_of=None, rtol=RTOL_STEP):
        """One shared kept set (selection kernel) + the shard-aware update from freshly cut slices."""
        cfg = self.cfg
        flat = [synth.gradient(cfg, step, k, DEV) for k in range(cfg.W)]
        slices = cut_slices(flat, self.off, offset_of)
        table = psync.make_slice_table(slices)
        arrival = synth.arrival_times(cfg, step)
        d_kept = torch.full((cfg.N,), -1, dtype=torch.int32, device=DEV)
        d_status = torch.full((1,), -9, dtype=torch.int32, device=DEV)
        st, keep = self.make_step(table, d_kept, d_status)
        psync.psync_step_device(st, torch.from_numpy(arrival).to(DEV))
        torch.cuda.synchronize()
        s, kept, _ = oracle.select_first_n(arrival, cfg.N, cfg.b)
        assert s == oracle.OK and int(d_status.item()) == 0 and np.array_equal(d_kept.cpu().numpy(), kept)
        self.oracle(slices, kept)
        self.compare_and_sync(f"{cfg.name} step {step}", rtol)


RAGGED = [0, 1, 1, 4_099, 20_000, 20_003, 51_111, 70_003]        # a 1-element, an empty and a 3-element server


# ------------------------------------------------------------------ work list
@pytest.mark.parametrize("M,dtype", [(1, synth.F32), (20, synth.F32), (1000, synth.BF16), (5000, synth.F32)])
def test_worklist_is_the_prefix_sum_of_tiles_per_server(M, dtype):
    rng = np.random.default_rng(M)
    lens = rng.integers(0, 9000, M)
    lens[rng.random(M) < 0.1] = 0
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    T = psync.binding.PSYNC_TILE_UNITS * (8 if dtype == synth.BF16 else 4)
    want = np.concatenate([[0], np.cumsum(-(-lens // T))]).astype(np.int64)     # numpy, not the oracle: integer work
    got = psync.psync_shard_worklist(torch.from_numpy(off).to(DEV), dtype)
    torch.cuda.synchronize()
    assert np.array_equal(got.cpu().numpy(), want)


# ------------------------------------------------------------------ every template instance, lock-step
@pytest.mark.parametrize("dtype", [synth.F32, synth.BF16])
@pytest.mark.parametrize("opt", [synth.SGD, synth.MOMENTUM, synth.RMSPROP_MOM])
@pytest.mark.parametrize("ema_mode", [synth.EMA_POST, synth.EMA_PRE, synth.EMA_OFF])
def test_every_template_instance_lockstep_on_ragged_slices(dtype, opt, ema_mode):
    cfg = replace(BASE, grad_dtype=dtype, opt=opt, ema_mode=ema_mode, name=f"slices_d{dtype}_o{opt}_e{ema_mode}")
    pair = SlicesPair(cfg, shard_off=RAGGED)
    for s in range(3):
        # step 0: allocator-aligned slices (theta's slice is NOT co-aligned: ragged cuts); step 1: every slice of a
        # server at the same odd offset (head peel, one phase); step 2: offsets differ between workers (mixed phases)
        offs = [None, lambda k, j: (3 * j + 1) % 8, lambda k, j: (5 * k + 3 * j) % 8][s]
        pair.step_first_n(s, offs, rtol=RTOL_BF16 if dtype == synth.BF16 else RTOL_STEP)


@pytest.mark.parametrize("state_misalign", [1, 3])
def test_unaligned_theta_state_and_ema_bases(state_misalign):
    cfg = replace(BASE, opt=synth.RMSPROP_MOM, name="slices_state_misaligned")
    pair = SlicesPair(cfg, shard_off=RAGGED, state_misalign=state_misalign)
    pair.step_first_n(0)
    pair.step_first_n(1, lambda k, j: (k + j) % 4)


@pytest.mark.parametrize("P,M", [(5, 2), (31, 3), (1024, 1), (1025, 1), (4096 + 7, 2), (300_007, 13)])
def test_sizes_around_tile_and_unit_boundaries(P, M):
    cfg = replace(BASE, P=P, M=M, N=5, b=2, opt=synth.MOMENTUM, name=f"slices_P{P}")
    pair = SlicesPair(cfg)
    pair.step_first_n(0)
    pair.step_first_n(1, lambda k, j: (k + 2 * j + 1) % 4)


# ------------------------------------------------------------------ kept rows, counts, failed servers, NULL entries
def test_one_kept_row_per_server_failed_server_and_null_entries_of_dropped_slices():
    cfg = replace(BASE, opt=synth.RMSPROP_MOM, name="slices_rows")
    pair = SlicesPair(cfg, shard_off=RAGGED)
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    a[4, :6] = np.inf                                               # server 4 cannot collect N gradients
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    slices = cut_slices(flat, pair.off, lambda k, j: (k * j) % 4)
    status, kept, _ = oracle.select_first_n_sharded(a, cfg.N, cfg.b)
    assert status[4] == oracle.ETOOFEW
    for j in range(pair.M):                                         # what server j drops is poisoned, then withheld
        for k in range(cfg.W):
            if status[j] != oracle.OK or k not in kept[j]:
                slices[k][j].fill_(float("nan"))
    d_kept = torch.full((pair.M, cfg.N), -1, dtype=torch.int32, device=DEV)
    d_status = torch.full((pair.M,), -9, dtype=torch.int32, device=DEV)
    table = psync.make_slice_table(slices)
    st, keep = pair.make_step(table, d_kept, d_status, per_shard=True)
    psync.psync_step_device(st, torch.from_numpy(a).to(DEV))
    torch.cuda.synchronize()
    assert np.array_equal(d_status.cpu().numpy(), status) and np.array_equal(d_kept.cpu().numpy(), kept)
    pair.oracle(slices, kept, per_shard=True, status=status)
    pair.compare_and_sync("rows + poison")
    assert np.array_equal(pair.host["theta"][pair.off[4]:pair.off[5]],
                          to_np(synth.init_theta(cfg, DEV))[pair.off[4]:pair.off[5]])   # failed server untouched
    # second step: the dropped entries are NULL pointers
    a = synth.arrival_times_per_server(cfg, 1, server_sigma=0.3)
    status, kept, _ = oracle.select_first_n_sharded(a, cfg.N, cfg.b)
    slices = cut_slices([synth.gradient(cfg, 1, k, DEV) for k in range(cfg.W)], pair.off)
    sparse = [[t if (status[j] == oracle.OK and k in kept[j]) else None for j, t in enumerate(row)]
              for k, row in enumerate(slices)]
    table = psync.make_slice_table(sparse)
    st, keep = pair.make_step(table, d_kept, d_status, per_shard=True)
    psync.psync_step_device(st, torch.from_numpy(a).to(DEV))
    torch.cuda.synchronize()
    pair.oracle(sparse, kept, per_shard=True, status=status)
    pair.compare_and_sync("rows + NULL entries")


def test_timeout_rule_per_server_counts_on_slices_and_garbage_count_is_a_failed_row():
    cfg = replace(BASE, opt=synth.MOMENTUM, name="slices_timeout")
    pair = SlicesPair(cfg, shard_off=RAGGED)
    W, M = cfg.W, pair.M
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    a[5, :] = 9.0                                                   # nobody reaches server 5 in time
    d_kept = torch.full((M, W), -1, dtype=torch.int32, device=DEV)
    d_n = torch.full((M,), 77_777, dtype=torch.int32, device=DEV)   # garbage until the kernel writes it
    d_status = torch.full((M,), -9, dtype=torch.int32, device=DEV)
    psync.psync_select_timeout(torch.from_numpy(a).to(DEV), W, 1.1, d_kept, d_n, d_status, rows=M)
    kept = np.full((M, W), -1, np.int32)
    n_kept = np.zeros(M, np.int32)
    status = np.zeros(M, np.int32)
    for r in range(M):
        status[r], k = oracle.select_timeout(a[r], 1.1)
        if status[r] == oracle.OK:
            kept[r, :k.size], n_kept[r] = k, k.size
    torch.cuda.synchronize()
    assert np.array_equal(d_status.cpu().numpy(), status) and np.array_equal(d_n.cpu().numpy(), n_kept)
    assert status[5] == oracle.ETOOFEW and n_kept[5] == 0            # ETOOFEW writes a zero count
    slices = cut_slices([synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)], pair.off, lambda k, j: j % 3)
    table = psync.make_slice_table(slices)
    # status = NULL: the failed row is recognised by its zero count alone (nothing is written, no NaN from 1/0)
    st, keep = pair.make_step(table, d_kept, None, per_shard=True, d_n_kept=d_n)
    psync.psync_aggregate_update(st)
    torch.cuda.synchronize()
    pair.oracle(slices, kept, per_shard=True, n_kept=np.maximum(n_kept, 1), status=status)
    pair.compare_and_sync("time-out on slices, status NULL")
    # a count nobody wrote (out of range) is a failed row too
    d_n[2] = 123_456
    before = {n: to_np(getattr(pair, n)) for n in STATE_NAMES}
    st, keep = pair.make_step(table, d_kept, None, per_shard=True, d_n_kept=d_n)
    psync.psync_aggregate_update(st)
    torch.cuda.synchronize()
    lo, hi = int(pair.off[2]), int(pair.off[3])
    for n in STATE_NAMES:
        if before[n] is not None:
            assert np.array_equal(to_np(getattr(pair, n))[lo:hi], before[n][lo:hi])


# ------------------------------------------------------------------ properties that hold at any size
def _run(pair, table, kept_np, layout, per_shard=False, variant=0):
    d_kept = torch.from_numpy(np.ascontiguousarray(kept_np)).to(DEV)
    st, keep = pair.make_step(table, d_kept, None, per_shard=per_shard, layout=layout, variant=variant)
    psync.psync_aggregate_update(st)
    torch.cuda.synchronize()
    return [to_np(getattr(pair, n)) for n in STATE_NAMES]


@pytest.mark.parametrize("dtype,opt", [(synth.F32, synth.RMSPROP_MOM), (synth.BF16, synth.MOMENTUM)])
def test_slices_are_bit_identical_to_the_flat_kernel_on_the_same_numbers(dtype, opt):
    """Same fixed-order fp32 sum, same update: cutting the flat buffers into separately allocated (and misaligned)
    slices must not change one bit.  Also the flat layout driven through the work list (views of flat buffers)."""
    cfg = replace(BASE, P=1_000_003, M=20, N=50, b=5, grad_dtype=dtype, opt=opt, name="slices_vs_flat")
    off = synth.shard_offsets(cfg)
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    kept = np.sort(np.random.default_rng(3).permutation(cfg.W)[:cfg.N]).astype(np.int32)
    ref = _run(SlicesPair(cfg, off), psync.make_grad_table(flat), kept, psync.PSYNC_GRADS_FLAT)       # K2, flat stream
    for offs in (None, lambda k, j: 1 + (j % 3), lambda k, j: (k + j) % 4):
        table = psync.make_slice_table(cut_slices(flat, off, offs))
        out = _run(SlicesPair(cfg, off), table, kept, psync.PSYNC_GRADS_SLICES)
        for a, b_ in zip(ref, out):
            assert a is None or np.array_equal(a, b_)
    views = psync.make_slice_table([[g[off[j]:off[j + 1]] for j in range(cfg.M)] for g in flat])
    out = _run(SlicesPair(cfg, off), views, kept, psync.PSYNC_GRADS_SLICES)
    for a, b_ in zip(ref, out):
        assert a is None or np.array_equal(a, b_)
    # flat buffers + one kept row per server (identical rows) through the work list == the flat stream
    rows = np.tile(kept, (cfg.M, 1))
    out = _run(SlicesPair(cfg, off), psync.make_grad_table(flat), rows, psync.PSYNC_GRADS_FLAT, per_shard=True)
    for a, b_ in zip(ref, out):
        assert a is None or np.array_equal(a, b_)


def test_many_tiny_servers_through_the_work_list_match_the_oracle_and_the_flat_rows_kernel():
    """M = 1000 servers of ~300 parameters: in the flat index space every 1024-element tile straddles servers (the
    rows kernel goes element by element there); the work list gives every server its own tiles."""
    cfg = replace(BASE, P=300_017, M=1000, N=9, b=3, opt=synth.RMSPROP_MOM, name="slices_tiny_servers")
    pair = SlicesPair(cfg)
    a = synth.arrival_times_per_server(cfg, 0, server_sigma=0.3)
    status, kept, _ = oracle.select_first_n_sharded(a, cfg.N, cfg.b)
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]
    out = _run(pair, psync.make_grad_table(flat), kept, psync.PSYNC_GRADS_FLAT, per_shard=True)          # work list
    h = pair.host
    assert oracle.aggregate_update_rows(pair.off, cfg.N, [synth.as_numpy_grad(g) for g in flat], kept, h["theta"],
                                        h["ema"], h["state0"], h["state1"], per_shard=True, opt=cfg.opt,
                                        ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu,
                                        rho=cfg.rho, eps=cfg.eps) == oracle.OK
    pair.compare_and_sync("tiny servers")
    other = SlicesPair(cfg)
    other.d_tiles = None                                            # no work list: the flat rows kernel
    ref = _run(other, psync.make_grad_table(flat), kept, psync.PSYNC_GRADS_FLAT, per_shard=True)
    for x, y in zip(ref, out):
        assert x is None or np.array_equal(x, y)
    third = SlicesPair(cfg)
    sl = _run(third, psync.make_slice_table(cut_slices(flat, pair.off, lambda k, j: (k + j) % 4)), kept,
              psync.PSYNC_GRADS_SLICES, per_shard=True)
    for x, y in zip(ref, sl):
        assert x is None or np.array_equal(x, y)


def test_slices_step_is_capturable_in_a_cuda_graph_and_replays_bit_identically():
    """psync_step_device on the slices layout makes no synchronising call: capture three steps, replay, compare with the
    same three steps enqueued directly."""
    cfg = replace(BASE, opt=synth.MOMENTUM, name="slices_graph")
    flat = [synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)]

    def run(use_graph):
        pair = SlicesPair(cfg, shard_off=RAGGED)
        table = psync.make_slice_table(cut_slices(flat, pair.off, lambda k, j: (k + j) % 3))
        d_kept = torch.full((cfg.N,), -1, dtype=torch.int32, device=DEV)
        d_status = torch.full((1,), -9, dtype=torch.int32, device=DEV)
        st, keep = pair.make_step(table, d_kept, d_status)
        arr = [torch.from_numpy(synth.arrival_times(cfg, s)).to(DEV) for s in range(3)]
        stream = torch.cuda.Stream()
        stream.wait_stream(torch.cuda.current_stream())
        if use_graph:
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                for s in range(3):
                    psync.psync_step_device(st, arr[s], t=s, stream=torch.cuda.current_stream())
            before = [to_np(getattr(pair, n)) for n in STATE_NAMES]
            g.replay()
            torch.cuda.synchronize()
            assert not np.array_equal(before[0], to_np(pair.theta))          # capture did not run the kernels, replay did
        else:
            for s in range(3):
                psync.psync_step_device(st, arr[s], t=s, stream=stream)
            torch.cuda.synchronize()
        return [to_np(getattr(pair, n)) for n in STATE_NAMES], keep, table

    a, _, _ = run(False)
    b_, _, _ = run(True)
    for x, y in zip(a, b_):
        assert x is None or np.array_equal(x, y)


def test_abi_validation_of_the_slices_layout():
    cfg = replace(BASE, P=4096, M=2, N=3, b=1, ragged=False, name="slices_abi")
    pair = SlicesPair(cfg)
    slices = cut_slices([synth.gradient(cfg, 0, k, DEV) for k in range(cfg.W)], pair.off)
    table = psync.make_slice_table(slices)
    d_kept = torch.arange(3, dtype=torch.int32, device=DEV)
    before = to_np(pair.theta)
    st, keep = pair.make_step(table, d_kept)
    st.d_tile_start = None
    assert psync.psync_aggregate_update(st, check=False) == psync.PSYNC_EINVAL
    st, keep = pair.make_step(table, d_kept)
    st.d_shard_off = None
    assert psync.psync_aggregate_update(st, check=False) == psync.PSYNC_EINVAL
    st, keep = pair.make_step(table, d_kept, variant=2)
    assert psync.psync_aggregate_update(st, check=False) == psync.PSYNC_EUNSUPPORTED
    st, keep = pair.make_step(table, d_kept)
    st.grad_layout = 7
    assert psync.psync_aggregate_update(st, check=False) == psync.PSYNC_EINVAL
    torch.cuda.synchronize()
    assert np.array_equal(to_np(pair.theta), before)
    geo = psync.psync_launch_geometry(pair.make_step(table, d_kept)[0])
    assert geo["grid"] == 4 and geo["block"] == 256 and geo["tile_elems"] == 1024
    # a work list built for the other gradient dtype (2048-parameter tiles): detected on the device, nothing is touched
    pair.d_tiles = psync.psync_shard_worklist(pair.d_off, synth.BF16)
    st, keep = pair.make_step(table, d_kept)
    assert psync.psync_aggregate_update(st, check=False) == psync.PSYNC_OK
    torch.cuda.synchronize()
    assert np.array_equal(to_np(pair.theta), before)


# ------------------------------------------------------------------ the headline config at FULL size, every element
def test_cfg3_full_size_separately_allocated_slices_some_misaligned_every_element():
    """cfg3 (P = 25,165,824, M = 20 ragged, N = 100, b = 6, RMSProp + EMA): 2,120 separately allocated slices, every
    seventh one placed 4 bytes off; two lock-step steps; ALL 25 M elements of theta / ms / mom / ema compared with
    the oracle's streamed form (oracle.accumulate over the kept workers in ascending order, then apply_sum)."""
    cfg = synth.PAPER_RMSPROP
    free, _ = torch.cuda.mem_get_info()
    if cfg.footprint_bytes * 1.2 > free:
        pytest.skip("not enough free HBM for the full-size config")
    pair = SlicesPair(cfg)
    off = pair.off
    slices = [[None] * cfg.M for _ in range(cfg.W)]
    for k in range(cfg.W):
        for j in range(cfg.M):
            o = 1 if (k * cfg.M + j) % 7 == 0 else 0
            buf = torch.empty(int(off[j + 1] - off[j]) + 8, dtype=torch.float32, device=DEV)
            slices[k][j] = buf[o:o + int(off[j + 1] - off[j])]
    table = psync.make_slice_table(slices)
    d_kept = torch.full((cfg.N,), -1, dtype=torch.int32, device=DEV)
    d_status = torch.full((1,), -9, dtype=torch.int32, device=DEV)
    st, keep = pair.make_step(table, d_kept, d_status)
    tmp = torch.empty(cfg.P, dtype=torch.float32, device=DEV)
    S = np.zeros(cfg.P, np.float64)
    h = pair.host
    for s in range(2):
        for k in range(cfg.W):
            synth.gradient(cfg, s, k, DEV, out=tmp)
            for j in range(cfg.M):
                slices[k][j].copy_(tmp[off[j]:off[j + 1]])
        arrival = synth.arrival_times(cfg, s)
        psync.psync_step_device(st, torch.from_numpy(arrival).to(DEV), t=s)
        torch.cuda.synchronize()
        stt, kept, _ = oracle.select_first_n(arrival, cfg.N, cfg.b)
        assert stt == oracle.OK and np.array_equal(d_kept.cpu().numpy(), kept)
        S[:] = 0.0
        for k in kept:                                               # what the servers received, D2H slice by slice
            host_k = np.concatenate([synth.as_numpy_grad(slices[k][j]) for j in range(cfg.M)])
            assert oracle.accumulate(S, host_k) == oracle.OK
        assert oracle.apply_sum(off, cfg.N, S, h["theta"], h["ema"], h["state0"], h["state1"], opt=cfg.opt,
                                ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu, rho=cfg.rho,
                                eps=cfg.eps) == oracle.OK
        pair.compare_and_sync(f"cfg3 full size, slices, step {s}")


def test_cfg3_full_size_1000_servers_one_kept_row_each_through_the_work_list_sampled():
    """cfg3's P, N, b and optimizer cut into M = 1000 ragged servers (25 k parameters each), every server with its own
    kept row (per-server arrival times), flat buffers through the work list -- the launch `bench.py --mode per_server
    --servers 1000` times.  Sampled columns (every server boundary, the first and last tiles, 40 k random elements)
    against the oracle's per-server rows on the gathered columns; two lock-step steps."""
    cfg = replace(synth.PAPER_RMSPROP, M=1000, name="cfg3_M1000")
    free, _ = torch.cuda.mem_get_info()
    if cfg.footprint_bytes * 1.15 > free:
        pytest.skip("not enough free HBM for the full-size config")
    pair = SlicesPair(cfg)
    off = pair.off
    rng = np.random.default_rng(1000)
    idx = np.unique(np.concatenate([np.arange(0, 4096), np.arange(cfg.P - 4096, cfg.P), off[1:-1], off[1:-1] - 1,
                                    off[1:-1] + 1, rng.integers(0, cfg.P, 40_000)])).astype(np.int64)
    idx = idx[(idx >= 0) & (idx < cfg.P)]
    d_idx = torch.from_numpy(idx).to(DEV)
    off_s = np.searchsorted(idx, off).astype(np.int64)             # the same servers, cut in the sampled index space
    host = {n: to_np(getattr(pair, n)[d_idx]) for n in STATE_NAMES}
    grads = [torch.empty(cfg.P, dtype=torch.float32, device=DEV) for _ in range(cfg.W)]
    table = psync.make_grad_table(grads)
    d_kept = torch.full((cfg.M, cfg.N), -1, dtype=torch.int32, device=DEV)
    d_status = torch.full((cfg.M,), -9, dtype=torch.int32, device=DEV)
    st, keep = pair.make_step(table, d_kept, d_status, per_shard=True, layout=psync.PSYNC_GRADS_FLAT)
    geo = psync.psync_launch_geometry(st)
    assert geo["grid"] == int(np.sum(-(-np.diff(off) // 1024))) and geo["block"] == 256      # the work list's grid
    for s in range(2):
        for k in range(cfg.W):
            synth.gradient(cfg, s, k, DEV, out=grads[k])
        a = synth.arrival_times_per_server(cfg, s, server_sigma=0.3)
        a[7, :20] = np.inf                                          # server 7 cannot collect N gradients
        psync.psync_step_device(st, torch.from_numpy(a).to(DEV), t=s)
        torch.cuda.synchronize()
        status, kept, _ = oracle.select_first_n_sharded(a, cfg.N, cfg.b)
        assert status[7] == oracle.ETOOFEW and np.array_equal(d_status.cpu().numpy(), status)
        assert np.array_equal(d_kept.cpu().numpy()[status == 0], kept[status == 0])
        g_s = [synth.as_numpy_grad(g[d_idx]) for g in grads]
        assert oracle.aggregate_update_rows(off_s, cfg.N, g_s, kept, host["theta"], host["ema"], host["state0"],
                                            host["state1"], per_shard=True, status=status, opt=cfg.opt,
                                            ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu,
                                            rho=cfg.rho, eps=cfg.eps) == oracle.OK
        for n in STATE_NAMES:
            got = to_np(getattr(pair, n)[d_idx])
            assert_close(got, host[n], RTOL_STEP, ATOL_STEP, f"cfg3 M=1000 step {s} {n} (sampled)")
            host[n] = got
        assert bool(torch.isfinite(pair.theta).all())


def test_parameter_server_step_class_drives_slices_and_per_server_rows():
    """The convenience class (plumbing only): per-(worker, server) slices + Alg. 4 per server j in one call per step."""
    cfg = replace(BASE, opt=synth.RMSPROP_MOM, name="slices_class")
    off = np.asarray(RAGGED, dtype=np.int64)
    theta = synth.init_theta(cfg, DEV)
    s0, s1 = synth.init_state(cfg, DEV)
    ema = theta.clone()
    ps = psync.ParameterServerStep(off, cfg.N, cfg.b, theta, ema, s0, s1, cfg.opt, cfg.ema_mode, alpha=cfg.alpha,
                                   mu=cfg.mu, rho=cfg.rho, eps=cfg.eps, per_server=True)
    host = {"theta": to_np(theta), "ema": to_np(ema), "state0": to_np(s0), "state1": to_np(s1)}
    for s in range(2):
        flat = [synth.gradient(cfg, s, k, DEV) for k in range(cfg.W)]
        a = synth.arrival_times_per_server(replace(cfg, M=off.size - 1), s, server_sigma=0.3)
        if s == 0:
            slices = cut_slices(flat, off, lambda k, j: (k + 2 * j) % 4)
            ps.set_gradient_slices(slices)
        else:
            ps.set_gradients(flat)                                  # flat buffers through the same work list
        ps.step(torch.from_numpy(a).to(DEV), cfg.gamma, t=s)
        torch.cuda.synchronize()
        status, kept, t_nth = oracle.select_first_n_sharded(a, cfg.N, cfg.b)
        assert np.array_equal(ps.d_status.cpu().numpy(), status) and np.array_equal(ps.d_kept.cpu().numpy(), kept)
        assert np.array_equal(ps.d_t_nth.cpu().numpy(), t_nth)
        assert oracle.aggregate_update_rows(off, cfg.N, [synth.as_numpy_grad(g) for g in flat], kept, host["theta"],
                                            host["ema"], host["state0"], host["state1"], per_shard=True, status=status,
                                            opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha,
                                            mu=cfg.mu, rho=cfg.rho, eps=cfg.eps) == oracle.OK
        for n, t in (("theta", theta), ("ema", ema), ("state0", s0), ("state1", s1)):
            assert_close(to_np(t), host[n], RTOL_STEP, ATOL_STEP, f"class step {s} {n}")
            host[n] = to_np(t)


# ------------------------------------------------------------------ seeded random cases: shapes nobody thought of
@pytest.mark.parametrize("seed", range(24))
def test_random_shard_layouts_alignments_rows_and_counts(seed):
    """Random M, shard lengths (many empty / shorter than the head peel / around one tile), slice offsets (0-7 elements,
    per worker and server), N, b, dtype, optimizer, EMA mode, kept-row mode (shared / per server / per-row counts) and
    failed rows; gradients chosen directly (no selection kernel), lock-step against oracle.aggregate_update_slices."""
    rng = np.random.default_rng(4000 + seed)
    M = int(rng.choice([1, 2, 3, 5, 17, 60]))
    lens = rng.choice([0, 1, 2, 3, 5, 31, 33, 100, 1023, 1024, 1025, 2049, 5000], size=M,
                      p=[.08, .06, .06, .06, .06, .06, .06, .1, .08, .08, .1, .1, .1])
    if lens.sum() == 0:
        lens[0] = 7
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    P = int(off[-1])
    W = int(rng.integers(1, 40))
    N = int(rng.integers(1, W + 1))
    dtype = int(rng.integers(0, 2))
    opt = int(rng.integers(0, 3))
    ema_mode = int(rng.integers(0, 3))
    cfg = replace(BASE, P=P, M=M, N=N, b=W - N, grad_dtype=dtype, opt=opt, ema_mode=ema_mode, ragged=False,
                  name=f"fuzz{seed}")
    pair = SlicesPair(cfg, shard_off=off, state_misalign=int(rng.choice([0, 0, 1, 2])))
    mode = int(rng.integers(0, 3))                  # 0: one shared row; 1: one row per server; 2: rows with counts
    per_shard = mode > 0
    rows = M if per_shard else 1
    stride = W if mode == 2 else N
    kept = np.full((rows, stride), -1, np.int32)
    n_kept = np.full(rows, N, np.int32)
    for r in range(rows):
        n_kept[r] = int(rng.integers(1, W + 1)) if mode == 2 else N
        kept[r, :n_kept[r]] = np.sort(rng.permutation(W)[:n_kept[r]])
    status = np.zeros(rows, np.int32)
    if per_shard and M > 1:
        status[int(rng.integers(0, M))] = oracle.ETOOFEW
    same_phase = bool(rng.integers(0, 2))
    phase = rng.integers(0, 8, size=M)
    tdt = torch.float32 if dtype == synth.F32 else torch.bfloat16
    flat = [(torch.randn(P, device=DEV) * 1e-3).to(tdt) for _ in range(W)]
    slices = cut_slices(flat, off, (lambda k, j: int(phase[j])) if same_phase else (lambda k, j: int((phase[j] + 3 * k) % 8)))
    table = psync.make_slice_table(slices)
    st, keep = pair.make_step(table, torch.from_numpy(kept).to(DEV), torch.from_numpy(status).to(DEV),
                              per_shard=per_shard, d_n_kept=torch.from_numpy(n_kept).to(DEV) if mode == 2 else None)
    psync.psync_aggregate_update(st)
    torch.cuda.synchronize()
    pair.oracle(slices, kept, per_shard=per_shard, n_kept=n_kept if mode == 2 else None, status=status)
    pair.compare_and_sync(f"fuzz {seed}: M={M} P={P} W={W} N={N} dtype={dtype} opt={opt} ema={ema_mode} mode={mode}",
                          RTOL_BF16 if dtype == synth.BF16 else RTOL_STEP)


# ------------------------------------------------------------------ host-buffer step from per-(worker, server) slices
@pytest.mark.parametrize("dtype,chunk", [(synth.F32, 4096), (synth.BF16, 0)])
def test_step_host_from_host_slices_matches_the_oracle(dtype, chunk):
    """psync_step_host with grad_layout = SLICES: h_grads is W x M host slices (what each server received); the kept
    workers' slices are gathered chunk by chunk (chunks straddle servers, an empty and a one-element server, slices at odd
    element offsets in host memory); the dropped workers' slices are not even there."""
    cfg = replace(BASE, grad_dtype=dtype, opt=synth.RMSPROP_MOM, name=f"host_slices_d{dtype}")
    pair = SlicesPair(cfg, shard_off=RAGGED)
    nbytes = psync.psync_step_host_workspace_bytes(cfg.N, cfg.W, cfg.grad_dtype, chunk)
    d_work = torch.empty(nbytes, dtype=torch.uint8, device=DEV)
    h_theta = torch.empty(cfg.P, dtype=torch.float32).pin_memory()
    h_kept = np.full(cfg.N, -1, dtype=np.int32)
    for s in range(2):
        flat = [synth.gradient(cfg, s, k, "cpu") for k in range(cfg.W)]
        arrival = synth.arrival_times(cfg, s)
        st_o, kept, t_nth_o = oracle.select_first_n(arrival, cfg.N, cfg.b)
        h_sl = cut_slices(flat, pair.off, lambda k, j: (k + 2 * j) % 5)
        dropped = sorted(set(range(cfg.W)) - set(kept.tolist()))
        for k in dropped:
            h_sl[k] = [None] * pair.M
        step, keep = psync.make_step(pair.off, cfg.N, cfg.W, cfg.grad_dtype, pair.theta, pair.ema, pair.state0, pair.state1,
                                     opt=cfg.opt, ema_mode=cfg.ema_mode, gamma_t=cfg.gamma, alpha=cfg.alpha, mu=cfg.mu,
                                     rho=cfg.rho, eps=cfg.eps, grad_layout=psync.PSYNC_GRADS_SLICES)
        st, t_nth = psync.psync_step_host(step, arrival, h_sl, d_work, h_theta_out=h_theta, h_kept=h_kept,
                                          chunk_elems=chunk)
        assert st == st_o == 0 and np.array_equal(h_kept, kept) and t_nth == t_nth_o
        pair.oracle(h_sl, kept)
        pair.compare_and_sync(f"host slices step {s}", RTOL_BF16 if dtype == synth.BF16 else RTOL_STEP)
        assert np.array_equal(h_theta.numpy(), to_np(pair.theta))
    # a KEPT worker's slice missing: PSYNC_EINVAL before anything is updated
    before = to_np(pair.theta)
    h_sl[int(kept[0])][3] = None
    st, _ = psync.psync_step_host(step, arrival, h_sl, d_work, chunk_elems=chunk, check=False)
    assert st == psync.PSYNC_EINVAL and np.array_equal(to_np(pair.theta), before)


def test_slice_table_validates_lengths_presence_and_worker_count():
    """The kernels read len_j elements through every kept slice pointer: the binding refuses a slice of another length
    (a short one would be an out-of-bounds device read), a table with no slice at all, and reports W (not W*M)."""
    off = np.array([0, 5, 5, 12], dtype=np.int64)
    mk = lambda n: torch.zeros(n, dtype=torch.float32, device=DEV)
    good = [[mk(5), None, mk(7)], [mk(5), mk(0), mk(7)]]
    t = psync.make_slice_table(good, off)
    assert t.W == 2 and t.d_ptrs.numel() == 6
    assert psync.make_slice_table(good).W == 2                       # without a shard table: no length check
    with pytest.raises(ValueError, match="worker 1 for server 2"):
        psync.make_slice_table([[mk(5), None, mk(7)], [mk(5), None, mk(6)]], off)
    with pytest.raises(ValueError, match="servers"):
        psync.make_slice_table(good, off[:3])
    with pytest.raises(ValueError, match="no gradient slice"):
        psync.make_slice_table([[None, None, None]], off)
    srv = psync.ParameterServerStep(off, 2, 0, mk(12), mk(12), None, None, psync.PSYNC_SGD, psync.PSYNC_EMA_POST, alpha=0.5)
    with pytest.raises(ValueError, match="worker 0 for server 0"):
        srv.set_gradient_slices([[mk(4), mk(0), mk(7)], [mk(5), mk(0), mk(7)]])
