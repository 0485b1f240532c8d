"""ctypes shim over the CPU oracle (oracle/psync_oracle.cpp) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports the product package (paper_1702_05800_b200) and the
product never imports it.  All arrays are numpy, host memory; bf16 gradients are uint16 bit
patterns.  The arithmetic lives in the C++ file; this module only marshals arguments.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "psync_oracle.cpp"
_LIB = _HERE / "libpsync_oracle.so"
_MIRROR_SRC = _HERE / "psync_mirror_f32.cpp"       # the fp32 diagnostic: a separate library, not the graded oracle
_MIRROR_LIB = _HERE / "libpsync_mirror_f32.so"

OK, EINVAL, ETOOFEW = 0, -1, -2
F32, BF16 = 0, 1
SGD, MOMENTUM, RMSPROP_MOM = 0, 1, 2
EMA_POST, EMA_PRE, EMA_OFF = 0, 1, 2

_lib = None
_mirror_lib = None
_mirror_on = False


def _compile(src: Path, out: Path, force: bool, extra=()) -> Path:
    if force or not out.exists() or out.stat().st_mtime < src.stat().st_mtime:
        tmp = out.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wextra", *extra,
               "-o", str(tmp), str(src)]
        subprocess.run(cmd, check=True)
        os.replace(tmp, out)
    return out


def build(force: bool = False) -> Path:
    """Compile the oracle with g++ (-O2, no fast-math, no FMA contraction, OpenMP) and, beside it, the fp32
    diagnostic mirror (its own source, its own library)."""
    _compile(_SRC, _LIB, force, ("-fopenmp",))
    _compile(_MIRROR_SRC, _MIRROR_LIB, force)
    return _LIB


def build_sanitized(out_dir) -> Path:
    """The graded oracle built with -fsanitize=address,undefined into `out_dir`; used by
    tests/test_oracle_sanitizers.py, which runs the oracle's own pin tests against it in a subprocess."""
    out = Path(out_dir) / "libpsync_oracle_asan.so"
    cmd = ["g++", "-std=c++17", "-O1", "-g", "-fno-omit-frame-pointer", "-ffp-contract=off", "-fopenmp", "-fPIC",
           "-shared", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-Wall", "-Wextra",
           "-o", str(out), str(_SRC)]
    subprocess.run(cmd, check=True)
    return out


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        override = os.environ.get("PSYNC_ORACLE_LIB")     # the sanitizer job points this at its instrumented build
        if not override:
            build()
        L = ctypes.CDLL(override or str(_LIB))
        i32, i64, f32, vp = ctypes.c_int32, ctypes.c_int64, ctypes.c_float, ctypes.c_void_p
        L.oracle_select_first_n.argtypes = [vp, vp, i32, i32, i32, vp, vp]
        L.oracle_select_first_n.restype = ctypes.c_int
        L.oracle_aggregate_update.argtypes = [i64, i32, vp, i32, i32, vp, ctypes.c_int, vp, vp, vp, vp, vp,
                                              ctypes.c_int, ctypes.c_int, f32, f32, f32, f32, f32]
        L.oracle_aggregate_update.restype = ctypes.c_int
        L.oracle_select_first_n_sharded.argtypes = [vp, vp, i32, i32, i32, i32, vp, vp, vp]
        L.oracle_select_first_n_sharded.restype = ctypes.c_int
        L.oracle_select_timeout.argtypes = [vp, vp, i32, i32, f32, i32, vp, vp]
        L.oracle_select_timeout.restype = ctypes.c_int
        L.oracle_aggregate_update_rows.argtypes = [i64, i32, vp, i32, i32, vp, ctypes.c_int, ctypes.c_int, vp, i32,
                                                   vp, vp, vp, vp, vp, vp, ctypes.c_int, ctypes.c_int,
                                                   f32, f32, f32, f32, f32]
        L.oracle_aggregate_update_rows.restype = ctypes.c_int
        L.oracle_aggregate_update_slices.argtypes = L.oracle_aggregate_update_rows.argtypes
        L.oracle_aggregate_update_slices.restype = ctypes.c_int
        L.oracle_async_apply_rows.argtypes = [i64, i32, vp, i32, i32, vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, i32,
                                              vp, vp, vp, vp, vp, vp, vp, vp, ctypes.c_int, ctypes.c_int,
                                              f32, f32, f32, f32, f32]
        L.oracle_async_apply_rows.restype = ctypes.c_int
        L.oracle_clip_scales_slices.argtypes = [vp, i32, i32, vp, ctypes.c_int, f32, vp]
        L.oracle_clip_scales_slices.restype = ctypes.c_int
        L.oracle_staleness.argtypes = [vp, i32, vp, i32, i64, i32, vp, vp, vp]
        L.oracle_staleness.restype = ctypes.c_int
        L.oracle_order_by_arrival.argtypes = [vp, i32, vp, vp]
        L.oracle_order_by_arrival.restype = ctypes.c_int
        L.oracle_async_apply.argtypes = [i64, i32, vp, i32, i32, vp, ctypes.c_int, vp, vp, vp, vp, vp, vp, vp,
                                         ctypes.c_int, ctypes.c_int, f32, f32, f32, f32, f32]
        L.oracle_kth_arrival_stats.argtypes = [vp, i32, i32, vp, vp, vp, vp, vp, vp]
        L.oracle_kth_arrival_stats.restype = ctypes.c_int
        L.oracle_interp_iterations.argtypes = [vp, vp, i32, i32, vp]
        L.oracle_interp_iterations.restype = ctypes.c_int
        L.oracle_lr_schedule.argtypes = [f32, f32, i64, i32, ctypes.c_double, vp]
        L.oracle_lr_schedule.restype = ctypes.c_int
        L.oracle_clip_scales.argtypes = [vp, i32, i64, ctypes.c_int, f32, vp]
        L.oracle_clip_scales.restype = ctypes.c_int
        L.oracle_async_apply.restype = ctypes.c_int
        L.oracle_accumulate.argtypes = [vp, vp, ctypes.c_int, i64]
        L.oracle_accumulate.restype = ctypes.c_int
        L.oracle_apply_sum.argtypes = [i64, i32, vp, i32, vp, vp, vp, vp, vp, ctypes.c_int, ctypes.c_int,
                                       f32, f32, f32, f32, f32]
        L.oracle_apply_sum.restype = ctypes.c_int
        L.oracle_ema.argtypes = [vp, vp, i64, f32]
        L.oracle_ema.restype = ctypes.c_int
        L.oracle_num_threads.restype = ctypes.c_int
        L.oracle_set_num_threads.argtypes = [ctypes.c_int]
        _lib = L
    return _lib


def mirror_lib() -> ctypes.CDLL:
    """The fp32 diagnostic mirror (oracle/psync_mirror_f32.cpp): its own library, loaded only on request."""
    global _mirror_lib
    if _mirror_lib is None:
        _compile(_MIRROR_SRC, _MIRROR_LIB, False)
        L = ctypes.CDLL(str(_MIRROR_LIB))
        i32, i64, f32, vp, ci = ctypes.c_int32, ctypes.c_int64, ctypes.c_float, ctypes.c_void_p, ctypes.c_int
        L.mirror_rsqrt_rn.argtypes = [f32]
        L.mirror_rsqrt_rn.restype = f32
        L.mirror_aggregate_update_rows.argtypes = [i64, i32, vp, i32, i32, vp, ci, ci, ci, vp, i32, vp, vp, vp, vp, vp,
                                                   vp, ci, ci, f32, f32, f32, f32, f32]
        L.mirror_accumulate.argtypes = [vp, vp, ci, i64]
        L.mirror_apply_sum.argtypes = [i64, i32, vp, i32, vp, vp, vp, vp, vp, ci, ci, f32, f32, f32, f32, f32]
        L.mirror_ema.argtypes = [vp, vp, i64, f32]
        L.mirror_async_apply.argtypes = [i64, i32, vp, i32, i32, vp, ci, vp, vp, vp, vp, vp, vp, vp, ci, ci,
                                         f32, f32, f32, f32, f32]
        for fn in (L.mirror_aggregate_update_rows, L.mirror_accumulate, L.mirror_apply_sum, L.mirror_ema,
                   L.mirror_async_apply):
            fn.restype = ci
        _mirror_lib = L
    return _mirror_lib


def _ptr(a):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


def _chk(a, dtype, name, n=None):
    if a is None:
        return
    if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags.c_contiguous):
        raise TypeError(f"{name}: need a C-contiguous numpy array of {np.dtype(dtype)}")
    if n is not None and a.size != n:
        raise ValueError(f"{name}: need {n} elements, got {a.size}")


def select_first_n(arrival, N, b, tags=None, t=0):
    """-> (status, kept[int32 N] or None, t_nth or None).  PAPER.md:L130, L148-158."""
    W = N + b
    _chk(arrival, np.float32, "arrival", W)
    _chk(tags, np.int32, "tags", W)
    kept = np.full(max(N, 0), -1, dtype=np.int32)
    t_nth = np.full(1, np.nan, dtype=np.float32)
    st = lib().oracle_select_first_n(_ptr(arrival), _ptr(tags), t, N, b, _ptr(kept), _ptr(t_nth))
    if st != OK:
        return st, None, None
    return st, kept, float(t_nth[0])


def _grad_dtype(grads):
    dt = grads[0].dtype
    if dt == np.float32:
        return F32
    if dt == np.uint16:
        return BF16
    raise TypeError("gradients must be float32 or uint16 (bf16 bit patterns)")


def aggregate_update(shard_off, N, grads, kept, theta, ema=None, state0=None, state1=None, opt=SGD,
                     ema_mode=EMA_POST, gamma_t=0.0, alpha=0.0, mu=0.0, rho=0.0, eps=0.0):
    """One step of Alg. 4 l.8-9 in place on theta / state / ema.  PAPER.md:L160-162."""
    P = theta.size
    shard_off = np.ascontiguousarray(shard_off, dtype=np.int64)
    M = shard_off.size - 1
    W = len(grads)
    gd = _grad_dtype(grads)
    for k, g in enumerate(grads):
        _chk(g, grads[0].dtype, f"grads[{k}]", P)
    _chk(kept, np.int32, "kept", N)
    for nm, a in (("theta", theta), ("ema", ema), ("state0", state0), ("state1", state1)):
        _chk(a, np.float32, nm, P)
    ptrs = (ctypes.c_void_p * W)(*[g.ctypes.data for g in grads])
    if _mirror_on:
        return mirror_lib().mirror_aggregate_update_rows(P, M, _ptr(shard_off), N, W, ctypes.cast(ptrs, ctypes.c_void_p),
                                                         gd, 0, 0, _ptr(kept), N, None, None, _ptr(theta), _ptr(ema),
                                                         _ptr(state0), _ptr(state1), opt, ema_mode, gamma_t, alpha, mu,
                                                         rho, eps)
    return lib().oracle_aggregate_update(P, M, _ptr(shard_off), N, W, ctypes.cast(ptrs, ctypes.c_void_p),
                                         gd, _ptr(kept), _ptr(theta), _ptr(ema), _ptr(state0), _ptr(state1),
                                         opt, ema_mode, gamma_t, alpha, mu, rho, eps)


def select_first_n_sharded(arrival, N, b, tags=None, t=0):
    """Alg. 4 per parameter server j: arrival[M][W] -> (status[M], kept[M][N], t_nth[M]).
    Rows of failed servers keep their fill values (kept -1, t_nth NaN)."""
    W = N + b
    if not (isinstance(arrival, np.ndarray) and arrival.ndim == 2 and arrival.shape[1] == W):
        raise ValueError("arrival must be [M][N+b]")
    M = arrival.shape[0]
    _chk(arrival, np.float32, "arrival", M * W)
    _chk(tags, np.int32, "tags", M * W)
    kept = np.full((M, N), -1, dtype=np.int32)
    t_nth = np.full(M, np.nan, dtype=np.float32)
    status = np.full(M, EINVAL, dtype=np.int32)
    rc = lib().oracle_select_first_n_sharded(_ptr(arrival), _ptr(tags), t, N, b, M, _ptr(kept), _ptr(t_nth),
                                             _ptr(status))
    if rc != OK:
        raise ValueError("oracle_select_first_n_sharded: invalid arguments")
    return status, kept, t_nth


def select_timeout(arrival, timeout, min_keep=1, tags=None, t=0):
    """Time-out rule (R19) -> (status, kept[int32 n_kept] or None)."""
    W = arrival.size
    _chk(arrival, np.float32, "arrival", W)
    _chk(tags, np.int32, "tags", W)
    kept = np.full(W, -1, dtype=np.int32)
    n = np.zeros(1, dtype=np.int32)
    st = lib().oracle_select_timeout(_ptr(arrival), _ptr(tags), t, W, timeout, min_keep, _ptr(kept), _ptr(n))
    if st != OK:
        return st, None
    return st, kept[:int(n[0])].copy()


def aggregate_update_rows(shard_off, N, grads, kept, theta, ema=None, state0=None, state1=None, per_shard=True,
                          n_kept=None, status=None, opt=SGD, ema_mode=EMA_POST, gamma_t=0.0, alpha=0.0, mu=0.0,
                          rho=0.0, eps=0.0):
    """Alg. 4 l.8-9 with one kept row per server (per_shard) and/or a per-row count n_kept (time-out rule).
    kept is int32 [rows][stride]; status int32 [rows] or None; rows = M if per_shard else 1."""
    P = theta.size
    shard_off = np.ascontiguousarray(shard_off, dtype=np.int64)
    M = shard_off.size - 1
    W = len(grads)
    gd = _grad_dtype(grads)
    for k, g in enumerate(grads):
        _chk(g, grads[0].dtype, f"grads[{k}]", P)
    rows = M if per_shard else 1
    if not (isinstance(kept, np.ndarray) and kept.ndim == 2 and kept.shape[0] == rows):
        raise ValueError("kept must be int32 [rows][stride]")
    _chk(kept, np.int32, "kept")
    _chk(n_kept, np.int32, "n_kept", rows)
    _chk(status, np.int32, "status", rows)
    for nm, a in (("theta", theta), ("ema", ema), ("state0", state0), ("state1", state1)):
        _chk(a, np.float32, nm, P)
    ptrs = (ctypes.c_void_p * W)(*[g.ctypes.data for g in grads])
    if _mirror_on:
        return mirror_lib().mirror_aggregate_update_rows(P, M, _ptr(shard_off), N, W, ctypes.cast(ptrs, ctypes.c_void_p),
                                                         gd, 0, 1 if per_shard else 0, _ptr(kept), kept.shape[1],
                                                         _ptr(n_kept), _ptr(status), _ptr(theta), _ptr(ema),
                                                         _ptr(state0), _ptr(state1), opt, ema_mode, gamma_t, alpha, mu,
                                                         rho, eps)
    return lib().oracle_aggregate_update_rows(P, M, _ptr(shard_off), N, W, ctypes.cast(ptrs, ctypes.c_void_p), gd,
                                              1 if per_shard else 0, _ptr(kept), kept.shape[1], _ptr(n_kept),
                                              _ptr(status), _ptr(theta), _ptr(ema), _ptr(state0), _ptr(state1),
                                              opt, ema_mode, gamma_t, alpha, mu, rho, eps)


def aggregate_update_slices(shard_off, N, slices, kept, theta, ema=None, state0=None, state1=None, per_shard=False,
                            n_kept=None, status=None, opt=SGD, ema_mode=EMA_POST, gamma_t=0.0, alpha=0.0, mu=0.0,
                            rho=0.0, eps=0.0):
    """Alg. 4 l.8-9 on what each server RECEIVES: slices[k][j] is worker k's G_k[j], a
    separate array of len_j elements (None where server j does not keep worker k).  kept is int32 [rows][stride]
    (a 1-D kept[N] is one row); n_kept / status int32 [rows] or None; rows = M if per_shard else 1."""
    P = theta.size
    shard_off = np.ascontiguousarray(shard_off, dtype=np.int64)
    M = shard_off.size - 1
    W = len(slices)
    first = next(a for row in slices for a in row if a is not None)
    gd = _grad_dtype([first])
    for k, row in enumerate(slices):
        if len(row) != M:
            raise ValueError(f"slices[{k}] needs M = {M} entries")
        for j, a in enumerate(row):
            _chk(a, first.dtype, f"slices[{k}][{j}]", int(shard_off[j + 1] - shard_off[j]))
    kept = np.ascontiguousarray(kept, dtype=np.int32)
    if kept.ndim == 1:
        kept = kept[None, :]
    rows = M if per_shard else 1
    if kept.shape[0] != rows:
        raise ValueError("kept must be int32 [rows][stride]")
    _chk(n_kept, np.int32, "n_kept", rows)
    _chk(status, np.int32, "status", rows)
    for nm, a in (("theta", theta), ("ema", ema), ("state0", state0), ("state1", state1)):
        _chk(a, np.float32, nm, P)
    flat = [None if a is None else a.ctypes.data for row in slices for a in row]
    ptrs = (ctypes.c_void_p * (W * M))(*flat)
    if _mirror_on:
        return mirror_lib().mirror_aggregate_update_rows(P, M, _ptr(shard_off), N, W, ctypes.cast(ptrs, ctypes.c_void_p),
                                                         gd, 1, 1 if per_shard else 0, _ptr(kept), kept.shape[1],
                                                         _ptr(n_kept), _ptr(status), _ptr(theta), _ptr(ema),
                                                         _ptr(state0), _ptr(state1), opt, ema_mode, gamma_t, alpha, mu,
                                                         rho, eps)
    return lib().oracle_aggregate_update_slices(P, M, _ptr(shard_off), N, W, ctypes.cast(ptrs, ctypes.c_void_p), gd,
                                                1 if per_shard else 0, _ptr(kept), kept.shape[1], _ptr(n_kept),
                                                _ptr(status), _ptr(theta), _ptr(ema), _ptr(state0), _ptr(state1),
                                                opt, ema_mode, gamma_t, alpha, mu, rho, eps)


def order_by_arrival(arrival):
    """Alg. 2's arrival order: worker indices by ascending (time, index), finite times only."""
    W = arrival.size
    _chk(arrival, np.float32, "arrival", W)
    order = np.full(W, -1, dtype=np.int32)
    n = np.zeros(1, dtype=np.int32)
    st = lib().oracle_order_by_arrival(_ptr(arrival), W, _ptr(order), _ptr(n))
    if st != OK:
        raise ValueError("oracle_order_by_arrival: invalid arguments")
    return order[:int(n[0])].copy()


def staleness(read_iter, order, t0, lag=0):
    """Staleness of the gradients Alg. 2 applies (Table 1) -> (status, staleness int64 [K],
    read_iter_out int64 [W], stats float64 [6] = min, mean, median, max, std, count)."""
    W, K = read_iter.size, order.size
    _chk(read_iter, np.int64, "read_iter", W)
    _chk(order, np.int32, "order", K)
    st = np.zeros(K, np.int64)
    nxt = np.zeros(W, np.int64)
    stats = np.zeros(6, np.float64)
    rc = lib().oracle_staleness(_ptr(read_iter), W, _ptr(order), K, t0, lag, _ptr(st), _ptr(nxt), _ptr(stats))
    if rc != OK:
        return rc, None, None, None
    return rc, st, nxt, stats


def kth_arrival_stats(arrival, iters=None):
    """Section 3.1's procedure on arrival[T][W] -> dict(sorted, count, mean, median[, est_time])."""
    if not (isinstance(arrival, np.ndarray) and arrival.ndim == 2):
        raise ValueError("arrival must be [T][W]")
    T, W = arrival.shape
    _chk(arrival, np.float32, "arrival", T * W)
    _chk(iters, np.float64, "iters", W)
    out = dict(sorted=np.zeros((T, W), np.float32), count=np.zeros(W, np.int32), mean=np.zeros(W, np.float64),
               median=np.zeros(W, np.float64))
    est = None if iters is None else np.zeros(W, np.float64)
    rc = lib().oracle_kth_arrival_stats(_ptr(arrival), T, W, _ptr(out["sorted"]), _ptr(out["count"]), _ptr(out["mean"]),
                                        _ptr(out["median"]), _ptr(iters), _ptr(est))
    if rc != OK:
        raise ValueError("oracle_kth_arrival_stats: invalid arguments")
    if est is not None:
        out["est_time"] = est
    return out


def interp_iterations(N_pts, iters_pts, W):
    """Fig. 5's measured points linearly interpolated to every N = 1..W -> float64 [W]."""
    N_pts = np.ascontiguousarray(N_pts, dtype=np.int32)
    iters_pts = np.ascontiguousarray(iters_pts, dtype=np.float64)
    if N_pts.size != iters_pts.size:
        raise ValueError("one iteration count per N")
    out = np.zeros(max(W, 0), dtype=np.float64)
    if lib().oracle_interp_iterations(_ptr(N_pts), _ptr(iters_pts), N_pts.size, W, _ptr(out)) != OK:
        raise ValueError("oracle_interp_iterations: invalid arguments")
    return out


def lr_schedule(gamma0, beta, t0, K, s):
    """gamma_0 beta^(t s) for t = t0 .. t0+K-1 -> float32 [K]."""
    out = np.zeros(K, dtype=np.float32)
    if lib().oracle_lr_schedule(gamma0, beta, t0, K, s, _ptr(out)) != OK:
        raise ValueError("oracle_lr_schedule: invalid arguments")
    return out


def clip_scales(grads, clip):
    """Global-norm clip factor clip / max(||G_k||, clip) of every worker's buffer -> float32 [W]."""
    W = len(grads)
    gd = _grad_dtype(grads)
    for k, g in enumerate(grads):
        _chk(g, grads[0].dtype, f"grads[{k}]", grads[0].size)
    ptrs = (ctypes.c_void_p * W)(*[g.ctypes.data for g in grads])
    out = np.zeros(W, dtype=np.float32)
    if lib().oracle_clip_scales(ctypes.cast(ptrs, ctypes.c_void_p), W, grads[0].size, gd, clip, _ptr(out)) != OK:
        raise ValueError("oracle_clip_scales: invalid arguments")
    return out


def clip_scales_slices(shard_off, slices, clip):
    """The same factors for gradients that lie as W x M per-(worker, server) slices: the norm is over all of a worker's
    slices ("across all layers") -> float32 [W]."""
    shard_off = np.ascontiguousarray(shard_off, dtype=np.int64)
    M, W = shard_off.size - 1, len(slices)
    first = next(a for row in slices for a in row if a is not None)
    gd = _grad_dtype([first])
    for k, row in enumerate(slices):
        if len(row) != M:
            raise ValueError("every worker needs M slices")
        for j, a in enumerate(row):
            _chk(a, first.dtype, f"slices[{k}][{j}]", int(shard_off[j + 1] - shard_off[j]))
    ptrs = (ctypes.c_void_p * (W * M))(*[None if a is None else a.ctypes.data for row in slices for a in row])
    out = np.zeros(W, dtype=np.float32)
    if lib().oracle_clip_scales_slices(ctypes.cast(ptrs, ctypes.c_void_p), W, M, _ptr(shard_off), gd, clip,
                                       _ptr(out)) != OK:
        raise ValueError("oracle_clip_scales_slices: invalid arguments")
    return out


def async_apply(shard_off, grads, order, theta, ema=None, state0=None, state1=None, gammas=None, gscales=None, opt=SGD,
                ema_mode=EMA_PRE, gamma_t=0.0, alpha=0.0, mu=0.0, rho=0.0, eps=0.0):
    """len(order) iterations of Alg. 2, one gradient each, in place."""
    P = theta.size
    shard_off = np.ascontiguousarray(shard_off, dtype=np.int64)
    M = shard_off.size - 1
    W = len(grads)
    gd = _grad_dtype(grads)
    for k, g in enumerate(grads):
        _chk(g, grads[0].dtype, f"grads[{k}]", P)
    _chk(order, np.int32, "order")
    _chk(gammas, np.float32, "gammas", order.size)
    _chk(gscales, np.float32, "gscales", order.size)
    for nm, a in (("theta", theta), ("ema", ema), ("state0", state0), ("state1", state1)):
        _chk(a, np.float32, nm, P)
    ptrs = (ctypes.c_void_p * W)(*[g.ctypes.data for g in grads])
    fn = mirror_lib().mirror_async_apply if _mirror_on else lib().oracle_async_apply
    return fn(P, M, _ptr(shard_off), order.size, W, ctypes.cast(ptrs, ctypes.c_void_p), gd,
              _ptr(order), _ptr(gammas), _ptr(gscales), _ptr(theta), _ptr(ema), _ptr(state0), _ptr(state1),
              opt, ema_mode, gamma_t, alpha, mu, rho, eps)


def async_apply_rows(shard_off, grads, order, theta, ema=None, state0=None, state1=None, slices=False, per_shard=True,
                     n_arrived=None, status=None, gammas=None, gscales=None, opt=SGD, ema_mode=EMA_PRE, gamma_t=0.0,
                     alpha=0.0, mu=0.0, rho=0.0, eps=0.0):
    """Alg. 2 per parameter server j: order is int32 [rows][stride] (rows = M if per_shard else 1),
    n_arrived int32 [rows] or None (= stride), gscales float32 [W] indexed by WORKER.  grads: W flat arrays, or with
    slices=True a list of W lists of M arrays (None where not needed)."""
    P = theta.size
    shard_off = np.ascontiguousarray(shard_off, dtype=np.int64)
    M = shard_off.size - 1
    W = len(grads)
    if slices:
        first = next(a for row in grads for a in row if a is not None)
        gd = _grad_dtype([first])
        for k, row in enumerate(grads):
            for j, a in enumerate(row):
                _chk(a, first.dtype, f"grads[{k}][{j}]", int(shard_off[j + 1] - shard_off[j]))
        flat = [None if a is None else a.ctypes.data for row in grads for a in row]
        ptrs = (ctypes.c_void_p * (W * M))(*flat)
    else:
        gd = _grad_dtype(grads)
        for k, g in enumerate(grads):
            _chk(g, grads[0].dtype, f"grads[{k}]", P)
        ptrs = (ctypes.c_void_p * W)(*[g.ctypes.data for g in grads])
    order = np.ascontiguousarray(order, dtype=np.int32)
    if order.ndim == 1:
        order = order[None, :]
    rows = M if per_shard else 1
    if order.shape[0] != rows:
        raise ValueError("order must be int32 [rows][stride]")
    _chk(n_arrived, np.int32, "n_arrived", rows)
    _chk(status, np.int32, "status", rows)
    _chk(gammas, np.float32, "gammas")
    _chk(gscales, np.float32, "gscales", W)
    for nm, a in (("theta", theta), ("ema", ema), ("state0", state0), ("state1", state1)):
        _chk(a, np.float32, nm, P)
    if _mirror_on:
        raise NotImplementedError("the fp32 mirror has no per-server Alg. 2; compare rows one server at a time")
    return lib().oracle_async_apply_rows(P, M, _ptr(shard_off), order.shape[1], W, ctypes.cast(ptrs, ctypes.c_void_p), gd,
                                         1 if slices else 0, 1 if per_shard else 0, _ptr(order), order.shape[1],
                                         _ptr(n_arrived), _ptr(status), _ptr(gammas), _ptr(gscales), _ptr(theta),
                                         _ptr(ema), _ptr(state0), _ptr(state1), opt, ema_mode, gamma_t, alpha, mu, rho,
                                         eps)


def accumulate(S, grad):
    """S[i] += grad[i] in double (one kept worker); call in ascending kept order."""
    _chk(S, np.float64, "S")
    gd = _grad_dtype([grad])
    _chk(grad, grad.dtype, "grad", S.size)
    fn = mirror_lib().mirror_accumulate if _mirror_on else lib().oracle_accumulate
    return fn(_ptr(S), _ptr(grad), gd, S.size)


def apply_sum(shard_off, N, S, theta, ema=None, state0=None, state1=None, opt=SGD, ema_mode=EMA_POST,
              gamma_t=0.0, alpha=0.0, mu=0.0, rho=0.0, eps=0.0):
    """Alg. 4 l.8-9 given the per-element sums S of the kept gradients."""
    P = theta.size
    shard_off = np.ascontiguousarray(shard_off, dtype=np.int64)
    M = shard_off.size - 1
    _chk(S, np.float64, "S", P)
    for nm, a in (("theta", theta), ("ema", ema), ("state0", state0), ("state1", state1)):
        _chk(a, np.float32, nm, P)
    fn = mirror_lib().mirror_apply_sum if _mirror_on else lib().oracle_apply_sum
    return fn(P, M, _ptr(shard_off), N, _ptr(S), _ptr(theta), _ptr(ema), _ptr(state0), _ptr(state1), opt, ema_mode,
              gamma_t, alpha, mu, rho, eps)


def ema_update(ema, theta, alpha):
    """ema <- alpha ema + (1-alpha) theta in place.  PAPER.md:L40."""
    _chk(ema, np.float32, "ema")
    _chk(theta, np.float32, "theta", ema.size)
    fn = mirror_lib().mirror_ema if _mirror_on else lib().oracle_ema
    return fn(_ptr(ema), _ptr(theta), ema.size, alpha)


class fp32_mirror:
    """Context manager: inside it aggregate_update / aggregate_update_rows / async_apply / accumulate / apply_sum /
    ema_update are served by the SEPARATE fp32 diagnostic library (oracle/psync_mirror_f32.cpp), which restates the
    operation list DESIGN.md readings R9/R10 give for the GPU (fp32 adds in the listed order, the five stated FMAs, a
    correctly rounded reciprocal square root) -- a GPU result must match it BIT FOR BIT.  It is a regression check of the
    kernels against their documented arithmetic, not parity evidence: the double-arithmetic oracle
    (oracle/psync_oracle.cpp, which contains none of this) stays the graded truth.  Selection, schedules, statistics
    are always the graded oracle's."""

    def __enter__(self):
        global _mirror_on
        self.prev = _mirror_on
        _mirror_on = True
        return self

    def __exit__(self, *exc):
        global _mirror_on
        _mirror_on = self.prev
        return False


def num_threads() -> int:
    return lib().oracle_num_threads()


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(n)
