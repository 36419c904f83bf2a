"""ORACLE — TEST INFRASTRUCTURE ONLY.

Plain CPU definition of the hot path (per-shot BFS connected components + ToT-weighted centroid,
see tpx3_oracle.cpp for the passage-by-passage citations). Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package. It never imports the product package (paper_2603_04942_b200) and the product never
imports it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

from . import bruteforce  # noqa: F401

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpx3_oracle.cpp")
_LIB = os.path.join(_HERE, "libtpx3_oracle.so")

# -O2, no -ffast-math: the fp32 divide must be IEEE round-to-nearest (reading R12).
CXXFLAGS = ["-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["g++", *CXXFLAGS, _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.tpx3_oracle_run.restype = ctypes.c_int
        lib.tpx3_oracle_run.argtypes = [ctypes.c_uint64] + [ctypes.c_void_p] * 4 + [
            ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int] + [ctypes.c_void_p] * 14
        lib.tpx3_oracle_localmax.restype = ctypes.c_int
        lib.tpx3_oracle_localmax.argtypes = [ctypes.c_uint64] + [ctypes.c_void_p] * 4 + [
            ctypes.c_uint64] * 4 + [ctypes.c_int] + [ctypes.c_void_p] * 14
        _lib = lib
    return _lib


def run(x, y, toa, tot, W: int, P: int, threads: int = 1, clusters: bool = True) -> dict:
    """Cluster + centroid on host arrays. Returns perm, label (sorted-position indexed),
    n_clusters and the per-cluster arrays (prefix c_), clusters in ascending label order."""
    lib = _load()
    x = np.ascontiguousarray(x, dtype=np.uint16)
    y = np.ascontiguousarray(y, dtype=np.uint16)
    toa = np.ascontiguousarray(toa, dtype=np.uint64)
    tot = np.ascontiguousarray(tot, dtype=np.uint16)
    n = x.shape[0]
    assert y.shape[0] == n and toa.shape[0] == n and tot.shape[0] == n
    perm = np.empty(n, dtype=np.uint32)
    label = np.empty(n, dtype=np.uint32)
    nc = ctypes.c_uint64(0)
    out = {"perm": perm, "label": label}
    if clusters:
        carr = {
            "c_label": np.empty(n, dtype=np.uint32), "c_size": np.empty(n, dtype=np.uint32),
            "c_shot": np.empty(n, dtype=np.uint32), "c_sum_tot": np.empty(n, dtype=np.int64),
            "c_sum_tot_x": np.empty(n, dtype=np.int64), "c_sum_tot_y": np.empty(n, dtype=np.int64),
            "c_toa_peak": np.empty(n, dtype=np.uint64), "c_cx": np.empty(n, dtype=np.float32),
            "c_cy": np.empty(n, dtype=np.float32),
            "c_sum_tot_tof": np.empty(n, dtype=np.int64), "c_ctof": np.empty(n, dtype=np.float32),
        }
        cptr = [a.ctypes.data for a in carr.values()]
    else:
        carr, cptr = {}, [None] * 11
    rc = lib.tpx3_oracle_run(n, x.ctypes.data, y.ctypes.data, toa.ctypes.data, tot.ctypes.data,
                             int(W), int(P), int(threads), perm.ctypes.data, label.ctypes.data,
                             ctypes.addressof(nc), *cptr)
    if rc != 0:
        raise RuntimeError("tpx3_oracle_run failed: %d" % rc)
    out["n_clusters"] = int(nc.value)
    for k, a in carr.items():
        out[k] = a[: out["n_clusters"]].copy()
    return out


def run_localmax(x, y, toa, tot, wx: int, wy: int, wt: int, P: int, threads: int = 0) -> dict:
    """Paper-literal mode (Eq. 3-9): hits = local ToT maxima of the box neighbourhood
    (wx, wy, wt, same shot), centroid over the box about each maximum. Returns perm, lmax
    (lmax[k] = k for a hit, 0xFFFFFFFF otherwise), n_clusters and the per-hit arrays (prefix c_)."""
    lib = _load()
    x = np.ascontiguousarray(x, dtype=np.uint16)
    y = np.ascontiguousarray(y, dtype=np.uint16)
    toa = np.ascontiguousarray(toa, dtype=np.uint64)
    tot = np.ascontiguousarray(tot, dtype=np.uint16)
    n = x.shape[0]
    perm = np.empty(n, dtype=np.uint32)
    lmax = np.empty(n, dtype=np.uint32)
    nc = ctypes.c_uint64(0)
    carr = {
        "c_label": np.empty(n, dtype=np.uint32), "c_size": np.empty(n, dtype=np.uint32),
        "c_shot": np.empty(n, dtype=np.uint32), "c_sum_tot": np.empty(n, dtype=np.int64),
        "c_sum_tot_x": np.empty(n, dtype=np.int64), "c_sum_tot_y": np.empty(n, dtype=np.int64),
        "c_toa_peak": np.empty(n, dtype=np.uint64), "c_cx": np.empty(n, dtype=np.float32),
        "c_cy": np.empty(n, dtype=np.float32),
        "c_sum_tot_tof": np.empty(n, dtype=np.int64), "c_ctof": np.empty(n, dtype=np.float32),
    }
    rc = lib.tpx3_oracle_localmax(n, x.ctypes.data, y.ctypes.data, toa.ctypes.data, tot.ctypes.data,
                                  int(wx), int(wy), int(wt), int(P), int(threads), perm.ctypes.data,
                                  lmax.ctypes.data, ctypes.addressof(nc), *[a.ctypes.data for a in carr.values()])
    if rc != 0:
        raise RuntimeError("tpx3_oracle_localmax failed: %d" % rc)
    out = {"perm": perm, "lmax": lmax, "n_clusters": int(nc.value)}
    for k, a in carr.items():
        out[k] = a[: out["n_clusters"]].copy()
    return out
