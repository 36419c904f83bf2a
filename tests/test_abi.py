"""CPU-only checks of the C-ABI boundary: the library builds for sm_100a, loads without a GPU
and exports every symbol include/tpx3.h declares; host-side argument validation works; the
product package never imports the oracle."""
import ctypes
import os
import re
import subprocess

import pytest

import paper_2603_04942_b200 as m

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "tpx3.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tpx3_[a-z_]+)\s*\(", src)))


def test_header_symbols_match_binding_list():
    assert declared_functions() == sorted(m.exported_symbols)


def test_library_builds_loads_and_exports_every_symbol():
    lib = m.load_library()
    for name in declared_functions():
        assert hasattr(lib, name), name
    out = subprocess.check_output(["nm", "-D", "--defined-only", m._build.LIB]).decode()
    for name in declared_functions():
        assert re.search(r"\bT %s\b" % name, out), name


def test_library_is_sm100a():
    out = subprocess.check_output(["cuobjdump", "-lelf", m._build.LIB]).decode()
    assert "sm_100a" in out


def test_plan_validation_host_only():
    lib = m.load_library()
    h = ctypes.c_void_p()
    ws = ctypes.c_size_t()

    def mk(**kw):
        d = dict(struct_size=ctypes.sizeof(m._CConfig), sensor_w=256, sensor_h=256, toa_window_ticks=320,
                 shot_period_ticks=640000, max_hits=1 << 20, device=0, flags=0, max_shot_hits=0, reserved=0)
        d.update(kw)
        return m._CConfig(**d)

    assert lib.tpx3_plan(None, ctypes.byref(h), ctypes.byref(ws)) == m.ERR_INVALID_ARG
    for bad in (dict(struct_size=4), dict(sensor_w=0), dict(sensor_h=257), dict(max_hits=0),
                dict(max_hits=(1 << 28) + 1), dict(toa_window_ticks=1 << 31), dict(device=-1), dict(reserved=1)):
        c = mk(**bad)
        assert lib.tpx3_plan(ctypes.byref(c), ctypes.byref(h), ctypes.byref(ws)) == m.ERR_INVALID_ARG, bad
    c = mk()
    assert lib.tpx3_plan(ctypes.byref(c), ctypes.byref(h), ctypes.byref(ws)) == m.OK
    assert ws.value > 46 * (1 << 20)  # general-path buffers are sized from max_hits
    assert lib.tpx3_launch_count(h) == 0
    assert lib.tpx3_free(h) == m.OK
    assert lib.tpx3_free(None) == m.ERR_INVALID_ARG
    c = mk(max_hits=1 << 28)
    assert lib.tpx3_plan(ctypes.byref(c), ctypes.byref(h), ctypes.byref(ws)) == m.OK
    assert ws.value < 20 * (1 << 30)  # fits easily beside 14 GB of resident input on a 180 GB part
    lib.tpx3_free(h)


def test_strerror():
    assert m.strerror(0) == "ok"
    assert "max_clusters" in m.strerror(m.ERR_CAPACITY)
    assert m.strerror(-99) == "unknown error"


def test_host_io_bytes_monotone():
    lib = m.load_library()
    a = lib.tpx3_host_io_bytes(1000, 100)
    b = lib.tpx3_host_io_bytes(2000, 100)
    assert b > a >= 14 * 1000 + 8 * 1000 + 52 * 100


def test_no_cpu_fallback_without_gpu():
    import torch

    if torch.cuda.is_available():
        pytest.skip("needs a box without a GPU")
    with pytest.raises(RuntimeError):
        m.plan(m.Config())


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2603_04942_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", s, flags=re.M), f
                assert "tpx3_oracle" not in s and "oracle/" not in s, f


def test_shard_shots_partition():
    for n_shots in (0, 1, 7, 100000):
        for ws in (1, 2, 3, 8):
            r = [m.shard_shots(n_shots, ws, k) for k in range(ws)]
            assert r[0][0] == 0 and r[-1][1] == n_shots
            assert all(r[k][1] == r[k + 1][0] for k in range(ws - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1


def test_timewalk_table_host_helper_matches_the_oracle():
    """tpx3_timewalk_table is host-only (Eq. 1): both sides evaluate it in fp64 and round to the
    nearest tick, so the tables must be identical."""
    import numpy as np
    from oracle import preprocess as pp

    for a, b, c, d, n in [(1000.0, 10.0, -2.0, 1.0, 64), (800.0, 4.0, 0.0, 1.0, 1024), (500.0, 3.0, 1.0, 1.2, 1024),
                          (0.0, 1.0, 2.5, 1.0, 8), (123.456, 0.0, -7.25, 0.9, 300), (50.0, -2.0, 0.0, 1.0, 16)]:
        assert np.array_equal(m.timewalk_table(a, b, c, d, n), pp.timewalk_table(a, b, c, d, n)), (a, b, c, d)
    assert m.timewalk_table(1.0, 1.0, 1.0, 1.0, 0).shape == (0,)


def test_stream_and_pipeline_buffer_sizes_host_only():
    """Pure host arithmetic of the two size queries: the stream buffer holds two carry banks, the emit arrays
    (14 bytes per event plus perm and label) and the block counters; the host-I/O buffer grows by the two
    per-push tables and a stream buffer exactly when the call is large enough to be pipelined (2^23 events)."""
    lib = m.load_library()
    chunk, carry = 1 << 20, 1 << 16
    b = lib.tpx3_stream_bytes(chunk, carry)
    floor = 2 * 14 * carry + (14 + 8) * (chunk + carry)
    assert floor <= b <= floor + (1 << 20)
    assert lib.tpx3_stream_bytes(2 * chunk, carry) > b and lib.tpx3_stream_bytes(chunk, 2 * carry) > b
    n_small, n_big, cap = (1 << 23) - 1, 1 << 23, 1 << 20
    small, big = lib.tpx3_host_io_bytes(n_small, cap), lib.tpx3_host_io_bytes(n_big, cap)
    per_push = (1 << 22) + (1 << 20)
    extra = 2 * 64 * per_push + lib.tpx3_stream_bytes(1 << 22, 1 << 20)
    assert extra <= big - small <= extra + (1 << 16)
    assert m.load_library().tpx3_host_route(None) == m.ERR_INVALID_ARG
