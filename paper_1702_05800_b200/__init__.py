"""psync: the parameter-server step of synchronous SGD with backup workers (arXiv 1702.05800,
Algorithm 4) as hand-written CUDA for sm_100a behind a C ABI (include/psync.h).

`binding` mirrors the C entry points (argument marshalling only), `server` bundles the device
buffers of one parameter server, `synth` draws the seeded synthetic workloads, `build` compiles
libpsync.so in-tree.  Nothing in this package imports oracle/.
"""
from . import binding, synth  # noqa: F401
from .binding import (  # noqa: F401
    HostCtx, PSYNC_BF16, PSYNC_ECUDA, PSYNC_EINVAL, PSYNC_EMA_OFF, PSYNC_EMA_POST, PSYNC_EMA_PRE, PSYNC_ETOOFEW,
    PSYNC_EUNSUPPORTED, PSYNC_F32, PSYNC_GRADS_FLAT, PSYNC_GRADS_SLICES, PSYNC_MOMENTUM, PSYNC_OK,
    PSYNC_RMSPROP_MOM, PSYNC_SGD, PsyncError, make_grad_table, make_slice_table, make_step,
    psync_aggregate_update, psync_async_apply, psync_async_step_device, psync_async_step_host, psync_clip_scales, psync_clip_scales_slices, psync_clip_scales_static,
    PSYNC_CLIP_STATIC_SCRATCH_BYTES,
    psync_clip_slices_workspace_bytes, psync_clip_workspace_bytes, psync_ema, psync_interp_iterations,
    psync_kth_arrival_stats, psync_launch_geometry, psync_lr_schedule, psync_lr_schedule_counted, psync_order_by_arrival,
    psync_order_by_arrival_sharded, psync_select_first_n, psync_select_first_n_sharded, psync_select_timeout,
    psync_shard_worklist, psync_staleness, psync_staleness_sharded, psync_step_device, psync_step_host,
    psync_step_host_workspace_bytes)
from .server import AsyncServerStep, ParameterServerStep  # noqa: F401
