"""Seeded synthetic TimePix3 workloads (BASELINE.json configs 0-4).

Shared by the oracle tests, the GPU parity tests and bench.py. This module holds none of the
method's arithmetic: it only draws pixel events. The C++ backend (``tpx3_gen.cpp``) is built
in-tree with g++ on first use.

Stand-in statement: the paper's real workloads (argon ATI electrons at 1 kHz, PAPER.md:38,
179, 195) are "available on request" only; these seeded synthetic inputs take
their shapes and stand in for them.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpx3_gen.cpp")
_LIB = os.path.join(_HERE, "libtpx3_gen.so")

SHOT_PERIOD_TICKS = 640000  # 1 kHz at 1.5625 ns ticks
TOA_WINDOW_TICKS = 320  # 500 ns
SENSOR = 256
BASE_SEED = 4942000

CONFIG_NAMES = {
    0: "cfg0_tiny_electron_vmi",
    1: "cfg1_electron_vmi_1khz",
    2: "cfg2_ion_vmi_tof",
    3: "cfg3_covariance_high_count",
    4: "cfg4_streaming",
    5: "cfg5_well_separated",
}


def build(force: bool = False) -> str:
    """Compile the generator backend (g++ -O2 -fopenmp). Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", _SRC, "-o", tmp]
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.tpx3gen_default_shots.restype = ctypes.c_int64
        lib.tpx3gen_default_shots.argtypes = [ctypes.c_int]
        lib.tpx3gen_particles_per_shot.restype = ctypes.c_int32
        lib.tpx3gen_particles_per_shot.argtypes = [ctypes.c_int]
        lib.tpx3gen_count.restype = ctypes.c_int64
        lib.tpx3gen_count.argtypes = [
            ctypes.c_int, ctypes.c_uint64, ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int,
        ]
        lib.tpx3gen_fill.restype = None
        lib.tpx3gen_fill.argtypes = [
            ctypes.c_int, ctypes.c_uint64, ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
        ]
        _lib = lib
    return _lib


@dataclass
class Workload:
    cfg_id: int
    seed: int
    shot_begin: int
    shots: int
    x: np.ndarray  # uint16[n]
    y: np.ndarray  # uint16[n]
    toa: np.ndarray  # uint64[n]
    tot: np.ndarray  # uint16[n]
    shot_offsets: np.ndarray  # int64[shots+1], hit range of each generated shot (delivery order)
    truth: dict = field(default_factory=dict)
    shot_period_ticks: int = SHOT_PERIOD_TICKS
    toa_window_ticks: int = TOA_WINDOW_TICKS
    sensor_w: int = SENSOR
    sensor_h: int = SENSOR

    @property
    def n(self) -> int:
        return int(self.x.shape[0])

    @property
    def name(self) -> str:
        return CONFIG_NAMES[self.cfg_id]

    def slice_shots(self, s0: int, s1: int) -> "Workload":
        """Sub-workload holding generated shots [s0, s1) (indices relative to shot_begin)."""
        a, b = int(self.shot_offsets[s0]), int(self.shot_offsets[s1])
        return Workload(
            self.cfg_id, self.seed, self.shot_begin + s0, s1 - s0,
            self.x[a:b], self.y[a:b], self.toa[a:b], self.tot[a:b],
            self.shot_offsets[s0:s1 + 1] - a, {},
            self.shot_period_ticks, self.toa_window_ticks, self.sensor_w, self.sensor_h,
        )

    def chunks(self, max_hits: int):
        """Shot-aligned chunk boundaries [(shot0, shot1)], each holding <= max_hits hits
        (config 4: chunks of 2^20 / 2^24 / 2^26 / 2^28 cut at shot boundaries)."""
        out = []
        s0 = 0
        off = self.shot_offsets
        while s0 < self.shots:
            lim = off[s0] + max_hits
            s1 = int(np.searchsorted(off, lim, side="right")) - 1
            if s1 <= s0:
                raise ValueError("a single shot exceeds max_hits")
            s1 = min(s1, self.shots)
            out.append((s0, s1))
            s0 = s1
        return out


def default_shots(cfg_id: int) -> int:
    return int(_load().tpx3gen_default_shots(cfg_id))


def particles_per_shot(cfg_id: int) -> int:
    return int(_load().tpx3gen_particles_per_shot(cfg_id))


_KMAX = {0: 12, 1: 20, 2: 30, 3: 16, 4: 30, 5: 12}


def max_shot_hits(cfg_id: int) -> int:
    """Upper bound on the pixel hits one shot of a config can hold (particles x largest footprint,
    + 5 % noise hits in config 3): a fact of the recipe, used as the library's tile-size hint."""
    h = particles_per_shot(cfg_id) * _KMAX[cfg_id]
    return h + h // 20 if cfg_id == 3 else h


def generate(cfg_id: int, shots: int | None = None, seed: int | None = None, shot_begin: int = 0,
             truth: bool = False, threads: int = 0, max_hits: int | None = None) -> Workload:
    """Generate ``shots`` shots of config ``cfg_id`` starting at shot ``shot_begin``.

    ``max_hits`` (optional) trims to the largest whole-shot prefix holding <= max_hits hits.
    """
    lib = _load()
    if shots is None:
        shots = default_shots(cfg_id)
    if seed is None:
        seed = BASE_SEED + cfg_id
    s0, s1 = shot_begin, shot_begin + shots
    counts = np.zeros(shots, dtype=np.int64)
    lib.tpx3gen_count(cfg_id, seed, s0, s1, counts.ctypes.data, threads)
    offsets = np.zeros(shots + 1, dtype=np.int64)
    np.cumsum(counts, out=offsets[1:])
    if max_hits is not None and offsets[-1] > max_hits:
        shots = int(np.searchsorted(offsets, max_hits, side="right")) - 1
        s1 = s0 + shots
        offsets = offsets[: shots + 1].copy()
    total = int(offsets[-1])
    x = np.empty(total, dtype=np.uint16)
    y = np.empty(total, dtype=np.uint16)
    toa = np.empty(total, dtype=np.uint64)
    tot = np.empty(total, dtype=np.uint16)
    tr = {}
    null = ctypes.c_void_p(0)
    if truth:
        npart = shots * particles_per_shot(cfg_id)
        tr = {
            "cx": np.empty(npart, dtype=np.float64),
            "cy": np.empty(npart, dtype=np.float64),
            "k": np.empty(npart, dtype=np.int32),
            "t0": np.empty(npart, dtype=np.int64),
            "shot": np.repeat(np.arange(s0, s1, dtype=np.int64), particles_per_shot(cfg_id)),
        }
        targs = [tr["cx"].ctypes.data, tr["cy"].ctypes.data, tr["k"].ctypes.data, tr["t0"].ctypes.data]
    else:
        targs = [null, null, null, null]
    lib.tpx3gen_fill(cfg_id, seed, s0, s1, offsets.ctypes.data, x.ctypes.data, y.ctypes.data,
                     toa.ctypes.data, tot.ctypes.data, *targs, threads)
    return Workload(cfg_id, seed, shot_begin, shots, x, y, toa, tot, offsets, tr)


def array_hash(a: np.ndarray) -> str:
    """64-bit FNV-1a style digest of an array's bytes (printed in reports so runs are comparable)."""
    import hashlib

    return hashlib.blake2b(np.ascontiguousarray(a).view(np.uint8), digest_size=8).hexdigest()
