"""CPU-only checks of the C-ABI boundary: libpsync.so loads without a GPU, exports every symbol that
include/psync.h declares, the ctypes mirror of psync_step matches the C layout, and host-detectable
argument errors return PSYNC_EINVAL without touching a device."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "psync.h")


@pytest.fixture(scope="module")
def B():
    from paper_1702_05800_b200 import build
    build.build()                       # nvcc cross-compiles without a GPU
    from paper_1702_05800_b200 import binding
    return binding


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"PSYNC_API\s+[\w\s\*]+?\b(psync_\w+)\s*\(", text)))


def test_every_declared_symbol_is_exported(B):
    names = declared_functions()
    assert set(names) == set(B.EXPORTS) and len(names) >= 8
    L = B.lib()
    for n in names:
        assert hasattr(L, n), f"{n} declared in psync.h but not exported by libpsync.so"
    out = subprocess.run(["nm", "-D", "--defined-only", str(B.LIB_PATH)], capture_output=True, text=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if ln.strip()}
    assert set(names) <= exported
    assert all(e.startswith("psync_") for e in exported), "only the psync_* C symbols may be visible"


def test_version_and_status_strings(B):
    assert B.psync_version() >= 110
    assert "ETOOFEW" in B.status_string(B.PSYNC_ETOOFEW) and "EINVAL" in B.status_string(B.PSYNC_EINVAL)


def test_ctypes_struct_matches_c_layout(B, tmp_path):
    fields = [f[0] for f in B.psync_step._fields_]
    prog = ['#include <stdio.h>', '#include <stddef.h>', f'#include "{HEADER}"', 'int main(void){',
            'printf("%zu\\n", sizeof(psync_step));']
    prog += [f'printf("%zu\\n", offsetof(psync_step, {f}));' for f in fields]
    prog += ['printf("%d %d %d %d\\n", PSYNC_OK, PSYNC_EINVAL, PSYNC_ETOOFEW, PSYNC_ECUDA);',
             'printf("%d\\n", PSYNC_MAX_WORKERS); return 0;}']
    src = tmp_path / "layout.c"
    src.write_text("\n".join(prog))
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", str(src), "-o", str(exe)], check=True)   # header is plain C
    out = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split("\n")
    assert int(out[0]) == ctypes.sizeof(B.psync_step)
    for f, line in zip(fields, out[1:]):
        assert int(line) == getattr(B.psync_step, f).offset, f
    assert out[1 + len(fields)].split() == ["0", "-1", "-2", "-4"]
    assert int(out[2 + len(fields)]) == B.PSYNC_MAX_WORKERS


def test_einval_without_a_device(B):
    L = B.lib()
    assert L.psync_select_first_n(None, None, 0, 1, 0, None, None, None, None) == B.PSYNC_EINVAL
    assert L.psync_select_first_n(8, None, 0, 0, 0, 8, None, 8, None) == B.PSYNC_EINVAL
    assert L.psync_select_first_n(8, None, 0, 1024, 1, 8, None, 8, None) == B.PSYNC_EINVAL
    assert L.psync_aggregate_update(None, None) == B.PSYNC_EINVAL
    assert L.psync_ema(None, None, 4, 0.5, None) == B.PSYNC_EINVAL
    assert L.psync_ema(16, 32, -1, 0.5, None) == B.PSYNC_EINVAL
    off = np.array([0, 5, 10], dtype=np.int64)
    s = B.psync_step()
    s.P, s.M, s.h_shard_off, s.N, s.W = 10, 2, off.ctypes.data, 2, 3
    s.d_grads, s.d_kept, s.d_theta, s.d_ema = 64, 128, 256, 512
    bad_off = np.array([0, 7, 9], dtype=np.int64)
    for mutate in (lambda: setattr(s, "N", 0), lambda: setattr(s, "W", 1), lambda: setattr(s, "W", 1025),
                   lambda: setattr(s, "grad_dtype", 2), lambda: setattr(s, "opt", 7), lambda: setattr(s, "ema_mode", 3),
                   lambda: setattr(s, "d_theta", None), lambda: setattr(s, "d_ema", None),
                   lambda: setattr(s, "h_shard_off", bad_off.ctypes.data), lambda: setattr(s, "M", 0),
                   lambda: setattr(s, "opt", 1)):      # momentum without state0
        saved = bytes(s)
        mutate()
        assert L.psync_aggregate_update(ctypes.byref(s), None) == B.PSYNC_EINVAL
        ctypes.memmove(ctypes.byref(s), saved, len(saved))
    for mutate in (lambda: setattr(s, "per_shard", 2), lambda: setattr(s, "per_shard", 1),   # per_shard without d_shard_off
                   lambda: setattr(s, "kept_stride", -1), lambda: setattr(s, "kept_stride", 1),  # stride < N, fixed count
                   lambda: setattr(s, "kept_stride", 1025)):
        saved = bytes(s)
        mutate()
        assert L.psync_aggregate_update(ctypes.byref(s), None) == B.PSYNC_EINVAL
        ctypes.memmove(ctypes.byref(s), saved, len(saved))
    s.per_shard, s.d_shard_off, s.variant = 1, 1024, 2
    assert L.psync_aggregate_update(ctypes.byref(s), None) == B.PSYNC_EUNSUPPORTED
    s.per_shard, s.d_shard_off, s.variant = 0, None, 0
    assert L.psync_select_first_n_sharded(None, None, 0, 1, 0, 1, None, None, None, None) == B.PSYNC_EINVAL
    assert L.psync_select_first_n_sharded(8, None, 0, 1, 0, 0, 8, None, 8, None) == B.PSYNC_EINVAL
    assert L.psync_select_first_n_sharded(8, None, 0, 1000, 25, 2, 8, None, 8, None) == B.PSYNC_EINVAL
    assert L.psync_select_timeout(None, None, 0, 4, 1, 1.0, 1, None, None, None, None) == B.PSYNC_EINVAL
    assert L.psync_select_timeout(8, None, 0, 0, 1, 1.0, 1, 8, 8, 8, None) == B.PSYNC_EINVAL
    assert L.psync_select_timeout(8, None, 0, 1025, 1, 1.0, 1, 8, 8, 8, None) == B.PSYNC_EINVAL
    assert L.psync_select_timeout(8, None, 0, 4, 0, 1.0, 1, 8, 8, 8, None) == B.PSYNC_EINVAL
    assert L.psync_select_timeout(8, None, 0, 4, 1, 1.0, 0, 8, 8, 8, None) == B.PSYNC_EINVAL
    assert L.psync_select_timeout(8, None, 0, 4, 1, float("nan"), 1, 8, 8, 8, None) == B.PSYNC_EINVAL
    assert B.psync_step_host_workspace_bytes(0, 3, 0, 0) == 0
    assert B.psync_step_host_workspace_bytes(2, 3, 0, 100) == 0
    n = B.psync_step_host_workspace_bytes(100, 106, 0, 1 << 20)
    assert n >= 2 * 100 * 4 * (1 << 20)


def test_launch_geometry_without_a_device(B):
    off = np.array([0, 25_165_824], dtype=np.int64)
    s = B.psync_step()
    s.P, s.M, s.h_shard_off, s.N, s.W = 25_165_824, 1, off.ctypes.data, 100, 106
    s.d_theta, s.d_ema, s.d_state0, s.d_state1, s.opt = 256, 512, 1024, 2048, B.PSYNC_RMSPROP_MOM
    g = B.psync_launch_geometry(s)
    assert g["block"] in (128, 256, 512) and g["grid"] >= 148 and g["tile_elems"] >= 512
    assert g["grid"] == -(-25_165_824 // g["tile_elems"])            # one tile per CTA, always
    s.grid_ctas = 37                                                 # accepted and ignored
    assert B.psync_launch_geometry(s)["grid"] == g["grid"]


def test_binding_refuses_cpu_tensors(B):
    import torch
    a = torch.zeros(4)
    with pytest.raises(ValueError):
        B.psync_ema(a, a.clone(), 0.5)
    with pytest.raises(ValueError):
        B.psync_select_first_n(a, 2, 2, torch.zeros(2, dtype=torch.int32), torch.zeros(1, dtype=torch.int32))


def test_product_never_imports_the_oracle():
    """The product package must not import, link or execute anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1702_05800_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "psync_oracle" not in text and "liboracle" not in text, f
    code = "import sys; import paper_1702_05800_b200; assert 'oracle' not in sys.modules"
    subprocess.run([sys.executable, "-c", code], check=True, cwd=ROOT)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            assert "paper_1702_05800_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "(paper_1702_05800_b200/csrc)", "").replace("product package (paper_1702_05800_b200)", "")
