"""Thin ctypes binding over libpsync.so (include/psync.h).  Argument marshalling ONLY: every step
of the path (selection, aggregation, update, EMA) runs in the CUDA kernels behind the C ABI.

torch is used for device memory and streams.  There is no CPU fallback: if the shared library is
missing or a tensor is not on a CUDA device the call raises.  This module never imports oracle/.
"""
from __future__ import annotations

import ctypes
from dataclasses import dataclass, field
from pathlib import Path
from typing import Optional, Sequence

import numpy as np
import torch

PKG = Path(__file__).resolve().parent
LIB_PATH = PKG / "libpsync.so"

PSYNC_OK, PSYNC_EINVAL, PSYNC_ETOOFEW, PSYNC_EUNSUPPORTED, PSYNC_ECUDA = 0, -1, -2, -3, -4
PSYNC_F32, PSYNC_BF16 = 0, 1
PSYNC_SGD, PSYNC_MOMENTUM, PSYNC_RMSPROP_MOM = 0, 1, 2
PSYNC_EMA_POST, PSYNC_EMA_PRE, PSYNC_EMA_OFF = 0, 1, 2
PSYNC_GRADS_FLAT, PSYNC_GRADS_SLICES = 0, 1
PSYNC_MAX_WORKERS = 1024
PSYNC_TILE_UNITS = 256

EXPORTS = ("psync_version", "psync_status_string", "psync_select_first_n", "psync_select_first_n_sharded",
           "psync_select_timeout", "psync_aggregate_update", "psync_shard_worklist", "psync_ema", "psync_order_by_arrival", "psync_order_by_arrival_sharded", "psync_clip_slices_workspace_bytes", "psync_clip_scales_slices", "psync_async_apply", "psync_async_step_device", "psync_staleness", "psync_staleness_sharded", "psync_step_device", "psync_clip_workspace_bytes",
           "psync_clip_scales", "psync_clip_scales_static", "psync_lr_schedule", "psync_lr_schedule_counted", "psync_kth_arrival_stats", "psync_interp_iterations",
           "psync_step_host_workspace_bytes", "psync_step_host", "psync_host_ctx_create", "psync_host_ctx_destroy",
           "psync_step_host_ctx", "psync_async_step_host", "psync_launch_geometry", "psync_probe_read",
           "psync_probe_copy", "psync_probe_pipe", "psync_selftest_rsqrt")


class PsyncError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {status_string(status)} ({status})")


class psync_step(ctypes.Structure):
    """Mirror of `struct psync_step` in include/psync.h (field order and types must match)."""
    _fields_ = [
        ("P", ctypes.c_int64), ("M", ctypes.c_int32), ("h_shard_off", ctypes.c_void_p),
        ("N", ctypes.c_int32), ("W", ctypes.c_int32), ("d_grads", ctypes.c_void_p),
        ("grad_dtype", ctypes.c_int32), ("d_kept", ctypes.c_void_p), ("d_status", ctypes.c_void_p),
        ("d_theta", ctypes.c_void_p), ("d_ema", ctypes.c_void_p), ("d_state0", ctypes.c_void_p),
        ("d_state1", ctypes.c_void_p), ("opt", ctypes.c_int32), ("ema_mode", ctypes.c_int32),
        ("gamma_t", ctypes.c_float), ("alpha", ctypes.c_float), ("mu", ctypes.c_float), ("rho", ctypes.c_float),
        ("eps", ctypes.c_float), ("grid_ctas", ctypes.c_int32), ("variant", ctypes.c_int32),
        ("per_shard", ctypes.c_int32), ("kept_stride", ctypes.c_int32), ("d_shard_off", ctypes.c_void_p),
        ("d_n_kept", ctypes.c_void_p), ("grad_layout", ctypes.c_int32), ("d_tile_start", ctypes.c_void_p),
    ]


_lib: Optional[ctypes.CDLL] = None


def lib() -> ctypes.CDLL:
    """Loads libpsync.so; raises if it has not been built (run __graft_entry__.build())."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise FileNotFoundError(f"{LIB_PATH} is missing: build it with `python -m paper_1702_05800_b200.build` "
                                    "(there is no CPU fallback)")
        L = ctypes.CDLL(str(LIB_PATH))
        vp, i32, i64, f32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_float
        L.psync_version.restype = ctypes.c_int
        L.psync_status_string.argtypes = [ctypes.c_int]
        L.psync_status_string.restype = ctypes.c_char_p
        L.psync_select_first_n.argtypes = [vp, vp, i32, i32, i32, vp, vp, vp, vp]
        L.psync_select_first_n.restype = ctypes.c_int
        L.psync_select_first_n_sharded.argtypes = [vp, vp, i32, i32, i32, i32, vp, vp, vp, vp]
        L.psync_select_first_n_sharded.restype = ctypes.c_int
        L.psync_select_timeout.argtypes = [vp, vp, i32, i32, i32, f32, i32, vp, vp, vp, vp]
        L.psync_select_timeout.restype = ctypes.c_int
        L.psync_aggregate_update.argtypes = [ctypes.POINTER(psync_step), vp]
        L.psync_aggregate_update.restype = ctypes.c_int
        L.psync_shard_worklist.argtypes = [vp, i32, i32, vp, vp]
        L.psync_shard_worklist.restype = ctypes.c_int
        L.psync_step_device.argtypes = [ctypes.POINTER(psync_step), vp, vp, i32, vp, vp]
        L.psync_step_device.restype = ctypes.c_int
        L.psync_order_by_arrival.argtypes = [vp, i32, vp, vp, vp]
        L.psync_order_by_arrival.restype = ctypes.c_int
        L.psync_order_by_arrival_sharded.argtypes = [vp, i32, i32, vp, vp, vp]
        L.psync_order_by_arrival_sharded.restype = ctypes.c_int
        L.psync_staleness.argtypes = [vp, i32, vp, vp, i32, vp, i32, vp, vp, vp, vp]
        L.psync_staleness.restype = ctypes.c_int
        L.psync_staleness_sharded.argtypes = [vp, i32, i32, vp, vp, i32, vp, i32, vp, vp, vp, vp]
        L.psync_staleness_sharded.restype = ctypes.c_int
        L.psync_async_apply.argtypes = [ctypes.POINTER(psync_step), vp, vp, vp]
        L.psync_async_step_device.argtypes = [ctypes.POINTER(psync_step), vp, vp, vp, vp]
        L.psync_async_step_device.restype = ctypes.c_int
        L.psync_clip_workspace_bytes.argtypes = [i32, i64, i32]
        L.psync_clip_workspace_bytes.restype = ctypes.c_size_t
        L.psync_clip_scales.argtypes = [vp, i32, i64, i32, f32, vp, vp, ctypes.c_size_t, vp]
        L.psync_clip_scales.restype = ctypes.c_int
        L.psync_clip_scales_static.argtypes = [vp, i32, i64, i32, f32, vp, vp]
        L.psync_clip_scales_static.restype = ctypes.c_int
        L.psync_clip_slices_workspace_bytes.argtypes = [i32, i32, vp, i32]
        L.psync_clip_slices_workspace_bytes.restype = ctypes.c_size_t
        L.psync_clip_scales_slices.argtypes = [vp, i32, i32, vp, vp, i32, f32, vp, vp, ctypes.c_size_t, vp]
        L.psync_clip_scales_slices.restype = ctypes.c_int
        L.psync_kth_arrival_stats.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp, vp, vp]
        L.psync_kth_arrival_stats.restype = ctypes.c_int
        L.psync_interp_iterations.argtypes = [vp, vp, i32, i32, vp, vp]
        L.psync_interp_iterations.restype = ctypes.c_int
        L.psync_lr_schedule.argtypes = [f32, f32, i64, i32, ctypes.c_double, vp, vp]
        L.psync_lr_schedule.restype = ctypes.c_int
        L.psync_lr_schedule_counted.argtypes = [f32, f32, vp, i64, vp, i32, i32, ctypes.c_double, vp, vp]
        L.psync_lr_schedule_counted.restype = ctypes.c_int
        L.psync_async_apply.restype = ctypes.c_int
        L.psync_ema.argtypes = [vp, vp, i64, f32, vp]
        L.psync_ema.restype = ctypes.c_int
        L.psync_step_host_workspace_bytes.argtypes = [i32, i32, i32, i64]
        L.psync_step_host_workspace_bytes.restype = ctypes.c_size_t
        L.psync_step_host.argtypes = [ctypes.POINTER(psync_step), vp, vp, i32, vp, vp, vp, vp, vp, ctypes.c_size_t,
                                      i64, vp]
        L.psync_step_host.restype = ctypes.c_int
        L.psync_host_ctx_create.argtypes = [ctypes.POINTER(ctypes.c_void_p)]
        L.psync_host_ctx_create.restype = ctypes.c_int
        L.psync_host_ctx_destroy.argtypes = [vp]
        L.psync_host_ctx_destroy.restype = ctypes.c_int
        L.psync_step_host_ctx.argtypes = [vp, ctypes.POINTER(psync_step), vp, vp, i32, vp, vp, vp, vp, vp,
                                          ctypes.c_size_t, i64, vp]
        L.psync_step_host_ctx.restype = ctypes.c_int
        L.psync_async_step_host.argtypes = [vp, ctypes.POINTER(psync_step), vp, vp, vp, vp, vp, vp, vp, ctypes.c_size_t,
                                            i64, vp]
        L.psync_async_step_host.restype = ctypes.c_int
        L.psync_launch_geometry.argtypes = [ctypes.POINTER(psync_step), vp, vp, vp, vp]
        L.psync_launch_geometry.restype = ctypes.c_int
        L.psync_probe_read.argtypes = [vp, i64, vp, vp]
        L.psync_probe_read.restype = ctypes.c_int
        L.psync_probe_copy.argtypes = [vp, vp, i64, vp]
        L.psync_probe_copy.restype = ctypes.c_int
        L.psync_probe_pipe.argtypes = [i32, i64, vp, ctypes.POINTER(ctypes.c_int64), vp]
        L.psync_probe_pipe.restype = ctypes.c_int
        L.psync_selftest_rsqrt.argtypes = [vp, ctypes.c_uint32, i64, vp, vp, vp]
        L.psync_selftest_rsqrt.restype = ctypes.c_int
        _lib = L
    return _lib


def status_string(status: int) -> str:
    return lib().psync_status_string(status).decode()


def psync_version() -> int:
    return lib().psync_version()


def _dptr(t: Optional[torch.Tensor], dtype=None, name="tensor") -> Optional[int]:
    if t is None:
        return None
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"{name}: expected {dtype}, got {t.dtype}")
    return t.data_ptr()


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def psync_select_first_n(d_arrival: torch.Tensor, N: int, b: int, d_kept: torch.Tensor, d_status: torch.Tensor,
                         d_t_nth: Optional[torch.Tensor] = None, d_step_tag: Optional[torch.Tensor] = None,
                         t: int = 0, stream=None, check: bool = True) -> int:
    """Enqueues the selection kernel (include/psync.h: psync_select_first_n)."""
    if d_arrival.numel() < N + b or d_kept.numel() < max(N, 0):
        raise ValueError("d_arrival needs N+b elements and d_kept N elements")
    if d_step_tag is not None and d_step_tag.numel() < N + b:
        raise ValueError("d_step_tag needs N+b elements")
    st = lib().psync_select_first_n(_dptr(d_arrival, torch.float32, "d_arrival"),
                                    _dptr(d_step_tag, torch.int32, "d_step_tag"), t, N, b,
                                    _dptr(d_kept, torch.int32, "d_kept"), _dptr(d_t_nth, torch.float32, "d_t_nth"),
                                    _dptr(d_status, torch.int32, "d_status"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_select_first_n")
    return st


def psync_select_first_n_sharded(d_arrival: torch.Tensor, N: int, b: int, M: int, d_kept: torch.Tensor,
                                 d_status: torch.Tensor, d_t_nth: Optional[torch.Tensor] = None,
                                 d_step_tag: Optional[torch.Tensor] = None, t: int = 0, stream=None,
                                 check: bool = True) -> int:
    """Alg. 4 per parameter server j (include/psync.h: psync_select_first_n_sharded):
    d_arrival [M][N+b] -> d_kept [M][N], d_status [M], d_t_nth [M]."""
    W = N + b
    if d_arrival.numel() < M * W or d_kept.numel() < M * max(N, 0) or d_status.numel() < M:
        raise ValueError("need d_arrival [M][N+b], d_kept [M][N], d_status [M]")
    if d_step_tag is not None and d_step_tag.numel() < M * W:
        raise ValueError("d_step_tag needs M*(N+b) elements")
    if d_t_nth is not None and d_t_nth.numel() < M:
        raise ValueError("d_t_nth needs M elements")
    st = lib().psync_select_first_n_sharded(_dptr(d_arrival, torch.float32, "d_arrival"),
                                            _dptr(d_step_tag, torch.int32, "d_step_tag"), t, N, b, M,
                                            _dptr(d_kept, torch.int32, "d_kept"),
                                            _dptr(d_t_nth, torch.float32, "d_t_nth"),
                                            _dptr(d_status, torch.int32, "d_status"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_select_first_n_sharded")
    return st


def psync_select_timeout(d_arrival: torch.Tensor, W: int, timeout: float, d_kept: torch.Tensor,
                         d_n_kept: torch.Tensor, d_status: torch.Tensor, rows: int = 1, min_keep: int = 1,
                         d_step_tag: Optional[torch.Tensor] = None, t: int = 0, stream=None,
                         check: bool = True) -> int:
    """Time-out rule (include/psync.h: psync_select_timeout): d_arrival [rows][W] ->
    d_kept [rows][W] (first d_n_kept[r] entries), d_n_kept [rows], d_status [rows]."""
    if d_arrival.numel() < rows * W or d_kept.numel() < rows * W or d_n_kept.numel() < rows or d_status.numel() < rows:
        raise ValueError("need d_arrival [rows][W], d_kept [rows][W], d_n_kept [rows], d_status [rows]")
    if d_step_tag is not None and d_step_tag.numel() < rows * W:
        raise ValueError("d_step_tag needs rows*W elements")
    st = lib().psync_select_timeout(_dptr(d_arrival, torch.float32, "d_arrival"),
                                    _dptr(d_step_tag, torch.int32, "d_step_tag"), t, W, rows, timeout, min_keep,
                                    _dptr(d_kept, torch.int32, "d_kept"), _dptr(d_n_kept, torch.int32, "d_n_kept"),
                                    _dptr(d_status, torch.int32, "d_status"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_select_timeout")
    return st


@dataclass
class GradTable:
    """Device array of W device pointers (worker k -> its gradient buffer) + the tensors kept alive."""
    d_ptrs: torch.Tensor
    buffers: Sequence[torch.Tensor]
    grad_dtype: int
    n_workers: Optional[int] = None       # set for slice tables, whose `buffers` holds W*M entries
    _recorded: set = field(default_factory=set, repr=False)   # side streams the tensors were recorded on

    def record_stream(self, stream) -> None:
        """Tells torch's caching allocator that `stream` (a torch.cuda.Stream other than the one the tensors were
        allocated on) reads the pointer table AND every gradient tensor, so none of those blocks is handed out again
        before the work enqueued on `stream` so far has finished -- even if the caller drops its references.  Done
        once per (table, stream); non-torch stream handles cannot be recorded and are the caller's to order."""
        if stream is None or not hasattr(stream, "cuda_stream") or stream.cuda_stream in self._recorded:
            return
        self.d_ptrs.record_stream(stream)
        seen = set()
        for t in self.buffers:
            if t is not None and t.untyped_storage().data_ptr() not in seen:     # views of one arena: once
                seen.add(t.untyped_storage().data_ptr())
                t.record_stream(stream)
        self._recorded.add(stream.cuda_stream)

    @property
    def W(self) -> int:
        return len(self.buffers) if self.n_workers is None else self.n_workers


def make_grad_table(buffers: Sequence[torch.Tensor]) -> GradTable:
    dt = buffers[0].dtype
    if dt not in (torch.float32, torch.bfloat16):
        raise TypeError("gradient buffers must be float32 or bfloat16")
    for g in buffers:
        if g.dtype != dt or not g.is_cuda or not g.is_contiguous():
            raise ValueError("gradient buffers must be contiguous CUDA tensors of one dtype")
    ptrs = torch.tensor([g.data_ptr() for g in buffers], dtype=torch.int64).to(buffers[0].device)
    return GradTable(ptrs, list(buffers), PSYNC_F32 if dt == torch.float32 else PSYNC_BF16)


def make_slice_table(slices: Sequence[Sequence[Optional[torch.Tensor]]], shard_off=None) -> GradTable:
    """Device pointer table [W*M] for PSYNC_GRADS_SLICES: slices[k][j] is worker k's G_k[j], its own CUDA tensor of
    len_j elements (any element alignment; None -> a NULL entry, legal where server j does not keep worker k).
    With shard_off (int64 [M+1]) every present slice is checked to hold exactly len_j = off[j+1] - off[j] elements: the
    kernels read len_j elements through every kept pointer, so a short slice would be an out-of-bounds device read."""
    W, M = len(slices), len(slices[0]) if len(slices) else 0
    first = next((t for row in slices for t in row if t is not None), None)
    if first is None:
        raise ValueError("no gradient slice is present (every entry is None)")
    dt = first.dtype
    if dt not in (torch.float32, torch.bfloat16):
        raise TypeError("gradient slices must be float32 or bfloat16")
    off = None
    if shard_off is not None:
        off = np.ascontiguousarray(shard_off, dtype=np.int64)
        if off.size != M + 1:
            raise ValueError(f"shard_off has {off.size - 1} servers, the slice rows have {M}")
    ptrs = []
    for k, row in enumerate(slices):
        if len(row) != M:
            raise ValueError("every worker needs M slices")
        for j, t in enumerate(row):
            if t is not None and (t.dtype != dt or not t.is_cuda or not t.is_contiguous() or t.device != first.device):
                raise ValueError("gradient slices must be contiguous CUDA tensors of one dtype on one device")
            if t is not None and off is not None and t.numel() != int(off[j + 1] - off[j]):
                raise ValueError(f"slice of worker {k} for server {j} has {t.numel()} elements, "
                                 f"the shard table says {int(off[j + 1] - off[j])}")
            ptrs.append(0 if t is None else t.data_ptr())
    d_ptrs = torch.tensor(ptrs, dtype=torch.int64).to(first.device)
    return GradTable(d_ptrs, [t for row in slices for t in row], PSYNC_F32 if dt == torch.float32 else PSYNC_BF16, W)


def psync_shard_worklist(d_shard_off: torch.Tensor, grad_dtype: int, d_tile_start: Optional[torch.Tensor] = None,
                         stream=None) -> torch.Tensor:
    """(server, tile) work list of the shard-aware kernel (include/psync.h: psync_shard_worklist).  Returns the device
    int64 [M+1] table (allocated here unless given); it depends only on the shard layout and the gradient dtype."""
    M = d_shard_off.numel() - 1
    if d_tile_start is None:
        d_tile_start = torch.empty(M + 1, dtype=torch.int64, device=d_shard_off.device)
    if d_tile_start.numel() < M + 1:
        raise ValueError("d_tile_start needs M+1 elements")
    st = lib().psync_shard_worklist(_dptr(d_shard_off, torch.int64, "d_shard_off"), M, grad_dtype,
                                    _dptr(d_tile_start, torch.int64, "d_tile_start"), _stream(stream))
    if st != PSYNC_OK:
        raise PsyncError(st, "psync_shard_worklist")
    return d_tile_start


def make_step(shard_off, N: int, W: int, grad_dtype: int, theta: torch.Tensor, ema: Optional[torch.Tensor] = None,
              state0: Optional[torch.Tensor] = None, state1: Optional[torch.Tensor] = None, opt: int = PSYNC_SGD,
              ema_mode: int = PSYNC_EMA_POST, gamma_t: float = 0.0, alpha: float = 0.0, mu: float = 0.0,
              rho: float = 0.0, eps: float = 0.0, d_grads: Optional[torch.Tensor] = None,
              d_kept: Optional[torch.Tensor] = None, d_status: Optional[torch.Tensor] = None, grid_ctas: int = 0,
              variant: int = 0, per_shard: bool = False, kept_stride: int = 0,
              d_shard_off: Optional[torch.Tensor] = None, d_n_kept: Optional[torch.Tensor] = None,
              grad_layout: int = PSYNC_GRADS_FLAT, d_tile_start: Optional[torch.Tensor] = None):
    """Fills a psync_step.  Returns (struct, keepalive) -- hold on to both until the call returns."""
    off = np.ascontiguousarray(shard_off, dtype=np.int64)
    s = psync_step()
    s.P = theta.numel()
    s.M = off.size - 1
    s.h_shard_off = off.ctypes.data
    s.N, s.W = N, W
    s.d_grads = _dptr(d_grads, torch.int64, "d_grads")
    s.grad_dtype = grad_dtype
    s.d_kept = _dptr(d_kept, torch.int32, "d_kept")
    s.d_status = _dptr(d_status, torch.int32, "d_status")
    s.d_theta = _dptr(theta, torch.float32, "theta")
    s.d_ema = _dptr(ema, torch.float32, "ema")
    s.d_state0 = _dptr(state0, torch.float32, "state0")
    s.d_state1 = _dptr(state1, torch.float32, "state1")
    for nm, a in (("ema", ema), ("state0", state0), ("state1", state1)):
        if a is not None and a.numel() != theta.numel():
            raise ValueError(f"{nm} must have P elements")
    s.opt, s.ema_mode = opt, ema_mode
    s.gamma_t, s.alpha, s.mu, s.rho, s.eps = gamma_t, alpha, mu, rho, eps
    s.grid_ctas, s.variant = grid_ctas, variant
    s.per_shard, s.kept_stride = int(per_shard), kept_stride
    s.d_shard_off = _dptr(d_shard_off, torch.int64, "d_shard_off")
    s.d_n_kept = _dptr(d_n_kept, torch.int32, "d_n_kept")
    s.grad_layout = grad_layout
    s.d_tile_start = _dptr(d_tile_start, torch.int64, "d_tile_start")
    if d_shard_off is not None and d_shard_off.numel() != off.size:
        raise ValueError("d_shard_off must have M+1 elements")
    if d_tile_start is not None and d_tile_start.numel() != off.size:
        raise ValueError("d_tile_start must have M+1 elements")
    if grad_layout == PSYNC_GRADS_SLICES and d_grads is not None and d_grads.numel() < W * (off.size - 1):
        raise ValueError("PSYNC_GRADS_SLICES: d_grads needs W*M entries")
    rows = s.M if per_shard else 1
    stride = kept_stride if kept_stride > 0 else (W if d_n_kept is not None else N)
    if 1 <= N <= W <= PSYNC_MAX_WORKERS:       # out-of-range N / W are the C side's PSYNC_EINVAL to report
        for nm, a, need in (("d_kept", d_kept, rows * stride), ("d_status", d_status, rows),
                            ("d_n_kept", d_n_kept, rows)):
            if a is not None and a.numel() < need:
                raise ValueError(f"{nm} needs {need} elements")
    return s, (off, d_grads, d_kept, d_status, theta, ema, state0, state1, d_shard_off, d_n_kept, d_tile_start)


def psync_aggregate_update(step: psync_step, stream=None, check: bool = True) -> int:
    """Enqueues the fused aggregate+update+EMA kernel (Alg. 4 l.8-9, L160-162)."""
    st = lib().psync_aggregate_update(ctypes.byref(step), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_aggregate_update")
    return st


def psync_step_device(step: psync_step, d_arrival: torch.Tensor, d_t_nth: Optional[torch.Tensor] = None,
                      d_step_tag: Optional[torch.Tensor] = None, t: int = 0, stream=None, check: bool = True) -> int:
    """Selection + fused update in one call (include/psync.h: psync_step_device; Alg. 4)."""
    rows = step.M if step.per_shard else 1
    if d_arrival.numel() < rows * step.W:
        raise ValueError("d_arrival needs rows*W elements")
    if d_step_tag is not None and d_step_tag.numel() < rows * step.W:
        raise ValueError("d_step_tag needs rows*W elements")
    if d_t_nth is not None and d_t_nth.numel() < rows:
        raise ValueError("d_t_nth needs one element per row")
    st = lib().psync_step_device(ctypes.byref(step), _dptr(d_arrival, torch.float32, "d_arrival"),
                                 _dptr(d_step_tag, torch.int32, "d_step_tag"), t,
                                 _dptr(d_t_nth, torch.float32, "d_t_nth"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_step_device")
    return st


def psync_order_by_arrival(d_arrival: torch.Tensor, W: int, d_order: torch.Tensor, d_n_arrived: torch.Tensor,
                           stream=None, check: bool = True) -> int:
    """Arrival order of Alg. 2 (include/psync.h: psync_order_by_arrival)."""
    if d_arrival.numel() < W or d_order.numel() < W or d_n_arrived.numel() < 1:
        raise ValueError("need d_arrival [W], d_order [W], d_n_arrived [1]")
    st = lib().psync_order_by_arrival(_dptr(d_arrival, torch.float32, "d_arrival"), W,
                                      _dptr(d_order, torch.int32, "d_order"),
                                      _dptr(d_n_arrived, torch.int32, "d_n_arrived"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_order_by_arrival")
    return st


def psync_order_by_arrival_sharded(d_arrival: torch.Tensor, W: int, M: int, d_order: torch.Tensor,
                                   d_n_arrived: torch.Tensor, stream=None, check: bool = True) -> int:
    """Arrival order of Alg. 2 per parameter server j (include/psync.h: psync_order_by_arrival_sharded)."""
    if d_arrival.numel() < M * W or d_order.numel() < M * W or d_n_arrived.numel() < M:
        raise ValueError("need d_arrival [M][W], d_order [M][W], d_n_arrived [M]")
    st = lib().psync_order_by_arrival_sharded(_dptr(d_arrival, torch.float32, "d_arrival"), W, M,
                                              _dptr(d_order, torch.int32, "d_order"),
                                              _dptr(d_n_arrived, torch.int32, "d_n_arrived"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_order_by_arrival_sharded")
    return st


def psync_clip_workspace_bytes(W: int, P: int, grad_dtype: int) -> int:
    return lib().psync_clip_workspace_bytes(W, P, grad_dtype)


def psync_clip_scales(table: "GradTable", clip: float, d_scales: torch.Tensor, d_work: torch.Tensor, stream=None,
                      check: bool = True) -> int:
    """Global-norm clip factors of the W buffers (include/psync.h: psync_clip_scales)."""
    if d_scales.numel() < table.W:
        raise ValueError("d_scales needs W elements")
    st = lib().psync_clip_scales(_dptr(table.d_ptrs, torch.int64, "d_grads"), table.W, table.buffers[0].numel(),
                                 table.grad_dtype, clip, _dptr(d_scales, torch.float32, "d_scales"),
                                 _dptr(d_work, None, "d_work"), d_work.numel() * d_work.element_size(),
                                 _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_clip_scales")
    return st


PSYNC_CLIP_STATIC_SCRATCH_BYTES = 2 << 20


def psync_clip_scales_static(table: "GradTable", clip: float, d_scales: torch.Tensor, stream=None, check: bool = True) -> int:
    """psync_clip_scales without a workspace argument, for callers that cannot allocate device memory (code running
    under a framework that owns the whole device through its caching allocator, or that must avoid cudaMalloc's
    device-wide synchronisation mid-step).  The partial sums go to a fixed 2 MiB array inside libpsync.so, so the request
    must satisfy psync_clip_workspace_bytes(W, P, dtype) <= PSYNC_CLIP_STATIC_SCRATCH_BYTES (else PSYNC_EUNSUPPORTED) and
    calls that may overlap on the GPU (different streams) race on that array; calls on one stream are safe.  The first
    call per device looks the array's address up -- make it before any stream capture.  include/psync.h has the contract."""
    if d_scales.numel() < table.W:
        raise ValueError("d_scales needs W elements")
    st = lib().psync_clip_scales_static(_dptr(table.d_ptrs, torch.int64, "d_grads"), table.W, table.buffers[0].numel(),
                                        table.grad_dtype, clip, _dptr(d_scales, torch.float32, "d_scales"),
                                        _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_clip_scales_static")
    return st


def psync_clip_slices_workspace_bytes(W: int, shard_off, grad_dtype: int) -> int:
    off = np.ascontiguousarray(shard_off, dtype=np.int64)
    return lib().psync_clip_slices_workspace_bytes(W, off.size - 1, off.ctypes.data, grad_dtype)


def psync_clip_scales_slices(table: "GradTable", shard_off, d_shard_off: torch.Tensor, clip: float, d_scales: torch.Tensor,
                             d_work: torch.Tensor, stream=None, check: bool = True) -> int:
    """Global-norm clip factors of W x M per-(worker, server) slices, the norm over all of a worker's slices
    (include/psync.h: psync_clip_scales_slices).  `table` comes from make_slice_table."""
    off = np.ascontiguousarray(shard_off, dtype=np.int64)
    M = off.size - 1
    W = table.d_ptrs.numel() // M
    if d_scales.numel() < W or d_shard_off.numel() < M + 1:
        raise ValueError("d_scales needs W elements, d_shard_off M + 1")
    st = lib().psync_clip_scales_slices(_dptr(table.d_ptrs, torch.int64, "d_grads"), W, M, off.ctypes.data,
                                        _dptr(d_shard_off, torch.int64, "d_shard_off"), table.grad_dtype, clip,
                                        _dptr(d_scales, torch.float32, "d_scales"), _dptr(d_work, None, "d_work"),
                                        d_work.numel() * d_work.element_size(), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_clip_scales_slices")
    return st


def psync_kth_arrival_stats(d_arrival: torch.Tensor, d_sorted: torch.Tensor, d_count: torch.Tensor,
                            d_mean: torch.Tensor, d_median: torch.Tensor, d_iters: Optional[torch.Tensor] = None,
                            d_est_time: Optional[torch.Tensor] = None, stream=None, check: bool = True) -> int:
    """Section 3.1's straggler statistics (include/psync.h: psync_kth_arrival_stats)."""
    if d_arrival.dim() != 2:
        raise ValueError("d_arrival must be [T][W]")
    T, W = d_arrival.shape
    if d_sorted.numel() < T * W:
        raise ValueError("d_sorted needs T*W elements")
    for nm, a in (("d_count", d_count), ("d_mean", d_mean), ("d_median", d_median), ("d_iters", d_iters),
                  ("d_est_time", d_est_time)):
        if a is not None and a.numel() < W:
            raise ValueError(f"{nm} needs W elements")
    st = lib().psync_kth_arrival_stats(_dptr(d_arrival, torch.float32, "d_arrival"), T, W,
                                       _dptr(d_sorted, torch.float32, "d_sorted"), _dptr(d_count, torch.int32, "d_count"),
                                       _dptr(d_mean, torch.float64, "d_mean"), _dptr(d_median, torch.float64, "d_median"),
                                       _dptr(d_iters, torch.float64, "d_iters"),
                                       _dptr(d_est_time, torch.float64, "d_est_time"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_kth_arrival_stats")
    return st


def psync_interp_iterations(N_pts, iters_pts, W: int, d_iters: torch.Tensor, stream=None, check: bool = True) -> int:
    """iterations(N), N = 1..W, from measured points (include/psync.h: psync_interp_iterations)."""
    n = np.ascontiguousarray(N_pts, dtype=np.int32)
    it = np.ascontiguousarray(iters_pts, dtype=np.float64)
    if n.size != it.size:
        raise ValueError("one iteration count per N")
    if d_iters.numel() < W:
        raise ValueError("d_iters needs W elements")
    st = lib().psync_interp_iterations(n.ctypes.data, it.ctypes.data, n.size, W,
                                       _dptr(d_iters, torch.float64, "d_iters"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_interp_iterations")
    return st


def psync_lr_schedule(gamma0: float, beta: float, t0: int, K: int, s: float, d_gamma: torch.Tensor, stream=None,
                      check: bool = True) -> int:
    """gamma_0 beta^((t0+i) s), i < K (include/psync.h: psync_lr_schedule)."""
    if d_gamma.numel() < K:
        raise ValueError("d_gamma needs K elements")
    st = lib().psync_lr_schedule(gamma0, beta, t0, K, s, _dptr(d_gamma, torch.float32, "d_gamma"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_lr_schedule")
    return st


def psync_lr_schedule_counted(gamma0: float, beta: float, d_t: torch.Tensor, K: int, s: float, d_gamma: torch.Tensor,
                              d_n_add: Optional[torch.Tensor] = None, t_set: int = -1, stream=None, check: bool = True) -> int:
    """The schedule from a device iteration counter: d_t <- t_set if t_set >= 0 else d_t + max(d_n_add); then
    d_gamma[i] = gamma_0 beta^((d_t+i) s), i < K (include/psync.h: psync_lr_schedule_counted)."""
    if d_gamma.numel() < K or d_t.numel() < 1:
        raise ValueError("d_gamma needs K elements and d_t one")
    st = lib().psync_lr_schedule_counted(gamma0, beta, _dptr(d_t, torch.int64, "d_t"), t_set,
                                         _dptr(d_n_add, torch.int32, "d_n_add") if d_n_add is not None else None,
                                         d_n_add.numel() if d_n_add is not None else 0, K, s,
                                         _dptr(d_gamma, torch.float32, "d_gamma"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_lr_schedule_counted")
    return st


def psync_async_apply(step: psync_step, d_gamma: Optional[torch.Tensor] = None, stream=None, check: bool = True,
                      d_gscale: Optional[torch.Tensor] = None) -> int:
    """K iterations of Alg. 2 in one pass (include/psync.h: psync_async_apply)."""
    if d_gscale is not None and d_gscale.numel() < step.W:
        raise ValueError("d_gscale needs W elements (indexed by worker)")
    st = lib().psync_async_apply(ctypes.byref(step), _dptr(d_gamma, torch.float32, "d_gamma"),
                                 _dptr(d_gscale, torch.float32, "d_gscale"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_async_apply")
    return st


def psync_async_step_device(step: psync_step, d_arrival: torch.Tensor, d_gamma: Optional[torch.Tensor] = None, stream=None,
                            check: bool = True, d_gscale: Optional[torch.Tensor] = None) -> int:
    """Arrival order + K iterations of Alg. 2 in one C call (include/psync.h: psync_async_step_device)."""
    rows = step.M if step.per_shard else 1
    if d_arrival.numel() < rows * step.W:
        raise ValueError("d_arrival needs [rows][W] elements")
    if d_gscale is not None and d_gscale.numel() < step.W:
        raise ValueError("d_gscale needs W elements (indexed by worker)")
    st = lib().psync_async_step_device(ctypes.byref(step), _dptr(d_arrival, torch.float32, "d_arrival"),
                                       _dptr(d_gamma, torch.float32, "d_gamma"),
                                       _dptr(d_gscale, torch.float32, "d_gscale"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_async_step_device")
    return st


def psync_ema(d_ema: torch.Tensor, d_theta: torch.Tensor, alpha: float, stream=None, check: bool = True) -> int:
    """ema <- alpha ema + (1-alpha) theta."""
    if d_ema.numel() != d_theta.numel():
        raise ValueError("ema and theta must have the same number of elements")
    st = lib().psync_ema(_dptr(d_ema, torch.float32, "d_ema"), _dptr(d_theta, torch.float32, "d_theta"),
                         d_ema.numel(), alpha, _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_ema")
    return st


def psync_launch_geometry(step: psync_step) -> dict:
    g = [ctypes.c_int32() for _ in range(4)]
    st = lib().psync_launch_geometry(ctypes.byref(step), *[ctypes.addressof(x) for x in g])
    if st != PSYNC_OK:
        raise PsyncError(st, "psync_launch_geometry")
    return dict(grid=g[0].value, block=g[1].value, tile_elems=g[2].value, smem_bytes=g[3].value)


def psync_step_host_workspace_bytes(N: int, W: int, grad_dtype: int, chunk_elems: int = 0) -> int:
    return lib().psync_step_host_workspace_bytes(N, W, grad_dtype, chunk_elems)


class HostCtx:
    """Copy stream + events of the host-buffer step, created once (include/psync.h: psync_host_ctx_create)."""

    def __init__(self):
        h = ctypes.c_void_p()
        st = lib().psync_host_ctx_create(ctypes.byref(h))
        if st != PSYNC_OK:
            raise PsyncError(st, "psync_host_ctx_create")
        self.handle = h

    def close(self):
        if self.handle is not None:
            lib().psync_host_ctx_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:  # noqa: BLE001
            pass


def psync_step_host(step: psync_step, h_arrival: np.ndarray, h_grads: Sequence[torch.Tensor],
                    d_work: torch.Tensor, h_theta_out: Optional[torch.Tensor] = None,
                    h_kept: Optional[np.ndarray] = None, h_step_tag: Optional[np.ndarray] = None, t: int = 0,
                    chunk_elems: int = 0, stream=None, check: bool = True, ctx: Optional[HostCtx] = None):
    """The step with HOST gradient buffers (include/psync.h: psync_step_host).  h_grads are CPU tensors
    (pinned for full PCIe rate); theta/ema/state stay on the device.  Returns (status, t_nth)."""
    W = step.W
    if len(h_grads) != W or h_arrival.size != W or h_arrival.dtype != np.float32:
        raise ValueError("need W host gradient buffers and W fp32 arrival times")
    if step.grad_layout == PSYNC_GRADS_SLICES:      # h_grads[k][j]: worker k's slice for server j (None = missing)
        M = step.M
        flat_ptrs = []
        for row in h_grads:
            if len(row) != M:
                raise ValueError("every worker needs M host slices")
            for g in row:
                if g is not None and (g.is_cuda or not g.is_contiguous()):
                    raise ValueError("host slices must be contiguous CPU tensors")
                flat_ptrs.append(None if g is None else g.data_ptr())
        ptrs = (ctypes.c_void_p * (W * M))(*flat_ptrs)
    else:
        for g in h_grads:
            if g.is_cuda or not g.is_contiguous() or g.numel() != step.P:
                raise ValueError("h_grads must be contiguous CPU tensors of P elements")
        ptrs = (ctypes.c_void_p * W)(*[g.data_ptr() for g in h_grads])
    t_nth = ctypes.c_float(float("nan"))
    if h_theta_out is not None and (h_theta_out.is_cuda or h_theta_out.dtype != torch.float32
                                    or h_theta_out.numel() != step.P):
        raise ValueError("h_theta_out must be a CPU float32 tensor of P elements")
    if h_kept is not None and (h_kept.dtype != np.int32 or h_kept.size != step.N):
        raise ValueError("h_kept must be int32[N]")
    if h_step_tag is not None and (h_step_tag.dtype != np.int32 or h_step_tag.size != W):
        raise ValueError("h_step_tag must be int32[W]")
    st = lib().psync_step_host_ctx(None if ctx is None else ctx.handle, ctypes.byref(step), h_arrival.ctypes.data,
                               None if h_step_tag is None else h_step_tag.ctypes.data, t,
                               ctypes.cast(ptrs, ctypes.c_void_p),
                               None if h_theta_out is None else h_theta_out.data_ptr(),
                               None if h_kept is None else h_kept.ctypes.data, ctypes.addressof(t_nth),
                               _dptr(d_work, None, "d_work"), d_work.numel() * d_work.element_size(), chunk_elems,
                               _stream(stream))
    if check and st not in (PSYNC_OK, PSYNC_ETOOFEW):
        raise PsyncError(st, "psync_step_host")
    return st, t_nth.value


def psync_async_step_host(step: psync_step, h_arrival: np.ndarray, h_grads, d_work: torch.Tensor,
                          h_gamma: Optional[np.ndarray] = None, h_theta_out: Optional[torch.Tensor] = None,
                          h_order: Optional[np.ndarray] = None, chunk_elems: int = 0, stream=None, check: bool = True,
                          ctx: Optional[HostCtx] = None):
    """One batch of Alg. 2 with HOST gradient buffers (include/psync.h: psync_async_step_host).  h_grads: W CPU tensors, or
    with step.grad_layout = SLICES W lists of M CPU tensors.  Returns (status, n_arrived)."""
    W = step.W
    if len(h_grads) != W or h_arrival.size != W or h_arrival.dtype != np.float32:
        raise ValueError("need W host gradient buffers and W fp32 arrival times")
    if step.grad_layout == PSYNC_GRADS_SLICES:
        M = step.M
        flat_ptrs = []
        for row in h_grads:
            if len(row) != M:
                raise ValueError("every worker needs M host slices")
            for g in row:
                if g is not None and (g.is_cuda or not g.is_contiguous()):
                    raise ValueError("host slices must be contiguous CPU tensors")
                flat_ptrs.append(None if g is None else g.data_ptr())
        ptrs = (ctypes.c_void_p * (W * M))(*flat_ptrs)
    else:
        for g in h_grads:
            if g.is_cuda or not g.is_contiguous() or g.numel() != step.P:
                raise ValueError("h_grads must be contiguous CPU tensors of P elements")
        ptrs = (ctypes.c_void_p * W)(*[g.data_ptr() for g in h_grads])
    if h_gamma is not None and (h_gamma.dtype != np.float32 or h_gamma.size < W):
        raise ValueError("h_gamma must be float32[W]")
    if h_order is not None and (h_order.dtype != np.int32 or h_order.size < W):
        raise ValueError("h_order must be int32[W]")
    if h_theta_out is not None and (h_theta_out.is_cuda or h_theta_out.dtype != torch.float32
                                    or h_theta_out.numel() != step.P):
        raise ValueError("h_theta_out must be a CPU float32 tensor of P elements")
    n = ctypes.c_int32(-1)
    st = lib().psync_async_step_host(None if ctx is None else ctx.handle, ctypes.byref(step), h_arrival.ctypes.data,
                                     ctypes.cast(ptrs, ctypes.c_void_p), None if h_gamma is None else h_gamma.ctypes.data,
                                     None if h_theta_out is None else h_theta_out.data_ptr(),
                                     None if h_order is None else h_order.ctypes.data, ctypes.byref(n),
                                     _dptr(d_work, None, "d_work"), d_work.numel() * d_work.element_size(), chunk_elems,
                                     _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_async_step_host")
    return st, n.value


def psync_probe_read(d_src: torch.Tensor, d_sink: torch.Tensor, stream=None) -> int:
    n = d_src.numel() * d_src.element_size() // 16
    st = lib().psync_probe_read(_dptr(d_src), n, _dptr(d_sink, torch.float32), _stream(stream))
    if st != PSYNC_OK:
        raise PsyncError(st, "psync_probe_read")
    return n * 16


def psync_probe_copy(d_dst: torch.Tensor, d_src: torch.Tensor, stream=None) -> int:
    n = d_src.numel() * d_src.element_size() // 16
    st = lib().psync_probe_copy(_dptr(d_dst), _dptr(d_src), n, _stream(stream))
    if st != PSYNC_OK:
        raise PsyncError(st, "psync_probe_copy")
    return n * 32


def psync_probe_pipe(mode: int, iters: int, d_sink: torch.Tensor, stream=None) -> int:
    """Arithmetic-pipe probe (include/psync.h: psync_probe_pipe): returns the fp32 lane-operations of the launch."""
    ops = ctypes.c_int64(0)
    st = lib().psync_probe_pipe(mode, iters, _dptr(d_sink, torch.float32), ctypes.byref(ops), _stream(stream))
    if st != PSYNC_OK:
        raise PsyncError(st, "psync_probe_pipe")
    return ops.value


def psync_selftest_rsqrt(d_mismatch: torch.Tensor, n: int, first_bits: int = 0, d_x: Optional[torch.Tensor] = None,
                         d_y: Optional[torch.Tensor] = None, stream=None) -> int:
    """Device rsqrt_rn against __frsqrt_rn on d_x[i] or on the bit patterns first_bits + i (include/psync.h)."""
    st = lib().psync_selftest_rsqrt(_dptr(d_x, torch.float32, "d_x"), first_bits, n, _dptr(d_y, torch.float32, "d_y"),
                                    _dptr(d_mismatch, torch.int64, "d_mismatch"), _stream(stream))
    if st != PSYNC_OK:
        raise PsyncError(st, "psync_selftest_rsqrt")
    return st


def psync_staleness(d_read_iter: torch.Tensor, d_order: torch.Tensor, d_t: torch.Tensor, d_staleness: torch.Tensor,
                    d_stats: torch.Tensor, d_status: torch.Tensor, K: int = 0, d_n_arrived: Optional[torch.Tensor] = None,
                    lag: int = 0, stream=None, check: bool = True) -> int:
    """Staleness of the gradients Alg. 2 applies (include/psync.h: psync_staleness)."""
    W = d_read_iter.numel()
    if d_staleness.numel() < W or d_stats.numel() < 6 or d_order.numel() < (W if d_n_arrived is not None else K):
        raise ValueError("need d_staleness [W], d_stats [6], d_order [K]")
    st = lib().psync_staleness(_dptr(d_read_iter, torch.int64, "d_read_iter"), W, _dptr(d_order, torch.int32, "d_order"),
                               _dptr(d_n_arrived, torch.int32, "d_n_arrived"), K, _dptr(d_t, torch.int64, "d_t"), lag,
                               _dptr(d_staleness, torch.int64, "d_staleness"), _dptr(d_stats, torch.float64, "d_stats"),
                               _dptr(d_status, torch.int32, "d_status"), _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_staleness")
    return st


def psync_staleness_sharded(d_read_iter: torch.Tensor, d_order: torch.Tensor, d_t: torch.Tensor, d_staleness: torch.Tensor,
                            d_stats: torch.Tensor, d_status: torch.Tensor, K: int = 0,
                            d_n_arrived: Optional[torch.Tensor] = None, lag: int = 0, stream=None, check: bool = True) -> int:
    """Table 1's bookkeeping per parameter server (include/psync.h: psync_staleness_sharded): d_read_iter [M][W]."""
    if d_read_iter.dim() != 2:
        raise ValueError("d_read_iter must be [M][W]")
    M, W = d_read_iter.shape
    if (d_order.numel() < M * W or d_staleness.numel() < M * W or d_stats.numel() < 6 * M or d_t.numel() < M or
            d_status.numel() < M or (d_n_arrived is not None and d_n_arrived.numel() < M)):
        raise ValueError("need d_order [M][W], d_staleness [M][W], d_stats [M][6], d_t [M], d_status [M], d_n_arrived [M]")
    st = lib().psync_staleness_sharded(_dptr(d_read_iter, torch.int64, "d_read_iter"), W, M,
                                       _dptr(d_order, torch.int32, "d_order"),
                                       _dptr(d_n_arrived, torch.int32, "d_n_arrived"), K, _dptr(d_t, torch.int64, "d_t"),
                                       lag, _dptr(d_staleness, torch.int64, "d_staleness"),
                                       _dptr(d_stats, torch.float64, "d_stats"), _dptr(d_status, torch.int32, "d_status"),
                                       _stream(stream))
    if check and st != PSYNC_OK:
        raise PsyncError(st, "psync_staleness_sharded")
    return st
