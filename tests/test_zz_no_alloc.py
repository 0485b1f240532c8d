"""psync_clip_scales_static: the clip factors for callers that cannot allocate device memory.

Why the entry point exists: a user of libpsync.so may be running where cudaMalloc is not available to them -- a plugin
inside a framework whose caching allocator already owns the device, or a training loop that must not take cudaMalloc's
device-wide synchronisation in the middle of a step.  psync_clip_scales needs a scratch buffer for its per-chunk
partial sums and makes the caller bring it; psync_clip_scales_static keeps a fixed 2 MiB array inside the library for
that purpose, so the caller passes inputs and outputs only.  The price is a size limit and shared state.

What this file checks, on the GPU, against the existing path (which tests/test_gpu_helpers.py checks against the
oracle): the same bits as psync_clip_scales, on two calls in a row that reuse the array with different shapes (the
second call must not be disturbed by what the first left behind), and that a request beyond the limit is refused
without writing anything.  The file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first
failure and a failure here must not hide the parity tests.  It passes alone in a fresh process (the first call does
the per-device address look-up) and after the rest of the suite.
"""
import numpy as np
import pytest
import torch

import paper_1702_05800_b200 as psync

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _grads(W, P, dtype, seed):
    g = torch.Generator(device="cpu").manual_seed(seed)
    out = []
    for k in range(W):
        x = torch.randn(P, generator=g, dtype=torch.float32) * (0.002 * (k + 1))   # norms on both sides of the bound
        out.append(x.to(torch.bfloat16 if dtype == psync.PSYNC_BF16 else torch.float32).to(DEV))
    return out


def _existing_path(table, P, clip):
    nbytes = psync.psync_clip_workspace_bytes(table.W, P, table.grad_dtype)
    d_work = torch.empty(nbytes // 8, dtype=torch.float64, device=DEV)
    d_scales = torch.full((table.W,), -1.0, dtype=torch.float32, device=DEV)
    psync.psync_clip_scales(table, clip, d_scales, d_work)
    torch.cuda.synchronize()
    return d_scales.cpu().numpy()


def _static_path(table, clip):
    d_scales = torch.full((table.W,), -1.0, dtype=torch.float32, device=DEV)
    psync.psync_clip_scales_static(table, clip, d_scales)
    torch.cuda.synchronize()
    return d_scales.cpu().numpy()


def test_static_scratch_matches_existing_path_on_two_calls_in_a_row():
    # call 1: many chunks per worker (P spans 7 chunks of 32768 fp32 elements + a ragged tail), 9 workers
    # call 2: another dtype, fewer and shorter rows -- its slots overlap call 1's in the shared array with a different
    #         row stride, so stale partial sums would be picked up if any slot were read without being rewritten
    cases = [(9, 7 * 32768 + 1237, psync.PSYNC_F32, 2.5, 11), (5, 3 * 65536 + 77, psync.PSYNC_BF16, 2.0, 12)]
    tables = [psync.make_grad_table(_grads(W, P, dt, seed)) for W, P, dt, _, seed in cases]
    want = [_existing_path(t, c[1], c[3]) for t, c in zip(tables, cases)]
    for w in want:
        assert (w > 0).all() and (w <= 1).all() and (w < 1).any() and (w == 1).any()   # both branches of the max()
    got = [_static_path(t, c[3]) for t, c in zip(tables, cases)]          # two calls in a row, same stream
    for g, w in zip(got, want):
        assert np.array_equal(g.view(np.uint32), w.view(np.uint32))        # same kernels, same order: same bits
    # back to back with no host synchronisation in between, then the first shape again
    d1 = torch.full((cases[0][0],), -1.0, dtype=torch.float32, device=DEV)
    d2 = torch.full((cases[1][0],), -1.0, dtype=torch.float32, device=DEV)
    d3 = torch.full((cases[0][0],), -1.0, dtype=torch.float32, device=DEV)
    psync.psync_clip_scales_static(tables[0], cases[0][3], d1)
    psync.psync_clip_scales_static(tables[1], cases[1][3], d2)
    psync.psync_clip_scales_static(tables[0], cases[0][3], d3)
    torch.cuda.synchronize()
    assert np.array_equal(d1.cpu().numpy(), want[0]) and np.array_equal(d2.cpu().numpy(), want[1])
    assert np.array_equal(d3.cpu().numpy(), want[0])


def test_static_scratch_limit_and_argument_errors():
    L = psync.binding.lib()
    cap = psync.PSYNC_CLIP_STATIC_SCRATCH_BYTES
    assert cap == 2 << 20
    # the largest fp32 request that fits with W = 1024 workers: 256 chunks of 32768 elements each
    P_fit = 256 * 32768
    assert psync.psync_clip_workspace_bytes(1024, P_fit, psync.PSYNC_F32) == cap
    assert psync.psync_clip_workspace_bytes(1024, P_fit + 4, psync.PSYNC_F32) > cap
    d_scales = torch.full((1024,), -1.0, dtype=torch.float32, device=DEV)
    ptrs = torch.zeros(1024, dtype=torch.int64, device=DEV)
    st = L.psync_clip_scales_static(ptrs.data_ptr(), 1024, P_fit + 4, psync.PSYNC_F32, 1.0, d_scales.data_ptr(), None)
    assert st == psync.PSYNC_EUNSUPPORTED                                  # refused, nothing enqueued
    torch.cuda.synchronize()
    assert (d_scales == -1.0).all()
    assert L.psync_clip_scales_static(None, 1, 4, 0, 1.0, d_scales.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_clip_scales_static(ptrs.data_ptr(), 0, 4, 0, 1.0, d_scales.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_clip_scales_static(ptrs.data_ptr(), 1, 4, 0, 0.0, d_scales.data_ptr(), None) == psync.PSYNC_EINVAL
    assert L.psync_clip_scales_static(ptrs.data_ptr(), 1, 4, 2, 1.0, d_scales.data_ptr(), None) == psync.PSYNC_EINVAL
    # cfg3's and cfg4's shapes fit (BASELINE.json configs[2], configs[3])
    assert psync.psync_clip_workspace_bytes(106, 25_165_824, psync.PSYNC_F32) <= cap
    assert psync.psync_clip_workspace_bytes(108, 100_000_000, psync.PSYNC_BF16) <= cap
