"""paper_2603_04942_b200 — thin Python binding of libtpx3 (include/tpx3.h).

The binding only marshals arguments: PyTorch supplies device memory and the CUDA stream; every
step of the hot path (sort, link, label compression, reduction, centroid) runs in the CUDA
kernels of csrc/. There is no CPU fallback: if the library cannot be built or loaded, or the
tensors are not CUDA tensors, the calls raise.

Function names follow the C ABI: plan / cluster / centroid / cluster_centroid / process_host /
status / free (tpx3_* in the header).
"""
from __future__ import annotations

import ctypes
from dataclasses import dataclass

from . import _build

__all__ = [
    "Tpx3Error", "Config", "Clusters", "Plan", "Stream", "plan", "load_library", "exported_symbols",
    "FLAG_VALIDATE_INPUT", "FLAG_FORCE_GENERAL", "strerror", "shard_shots", "unwrap_toa_static",
]

FLAG_VALIDATE_INPUT = 1 << 0
FLAG_FORCE_GENERAL = 1 << 1

OK, ERR_INVALID_ARG, ERR_CAPACITY, ERR_OUT_OF_RANGE, ERR_CUDA, ERR_NOT_CONTIGUOUS, ERR_TOO_LARGE = 0, -1, -2, -3, -4, -5, -6
STATIC_UNWRAP_MAX = 1 << 26   # tpx3.h: TPX3_STATIC_UNWRAP_MAX

# Every symbol include/tpx3.h declares (tests check the built library exports all of them).
exported_symbols = (
    "tpx3_plan", "tpx3_cluster", "tpx3_centroid", "tpx3_cluster_centroid", "tpx3_localmax_centroid",
    "tpx3_unwrap_toa", "tpx3_unwrap_toa_static", "tpx3_timewalk_table", "tpx3_preprocess", "tpx3_preprocess_cluster_centroid", "tpx3_host_io_bytes",
    "tpx3_stream_bytes", "tpx3_stream_open", "tpx3_stream_push", "tpx3_stream_close",
    "tpx3_process_host", "tpx3_host_route", "tpx3_status", "tpx3_launch_count", "tpx3_profile_enable", "tpx3_profile_read",
    "tpx3_free", "tpx3_strerror",
)
STAGES = ("fused", "sort", "link", "centroid")


class Tpx3Error(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__("%s failed: %s (%d)" % (where, strerror(code), code))


class _CConfig(ctypes.Structure):
    _fields_ = [
        ("struct_size", ctypes.c_uint32), ("sensor_w", ctypes.c_uint16), ("sensor_h", ctypes.c_uint16),
        ("toa_window_ticks", ctypes.c_uint32), ("shot_period_ticks", ctypes.c_uint64),
        ("max_hits", ctypes.c_uint64), ("device", ctypes.c_int32), ("flags", ctypes.c_uint32),
        ("max_shot_hits", ctypes.c_uint32), ("reserved", ctypes.c_uint32),
    ]


class _CClusters(ctypes.Structure):
    _fields_ = [(k, ctypes.c_void_p) for k in
                ("label", "size", "shot", "sum_tot", "sum_tot_x", "sum_tot_y", "toa_peak", "cx", "cy", "sum_tot_tof",
                 "ctof")]


class _CStreamInfo(ctypes.Structure):
    _fields_ = [(k, ctypes.c_uint64) for k in ("n_emitted", "n_carry", "n_late", "late_total", "label_base",
                                               "shots_emitted")]


class _CStatus(ctypes.Structure):
    _fields_ = [("error", ctypes.c_uint32), ("path", ctypes.c_uint32), ("n_clusters", ctypes.c_uint32),
                ("sort_passes", ctypes.c_uint32), ("n", ctypes.c_uint64)]


class _CProfile(ctypes.Structure):
    _fields_ = [("ms", ctypes.c_double * 4), ("launches", ctypes.c_uint64 * 4), ("calls", ctypes.c_uint64)]


_lib = None


def load_library(build: bool = True) -> ctypes.CDLL:
    """Load (building first if stale) libtpx3.so and declare the prototypes. Raises on failure."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build() if build else _build.LIB
    lib = ctypes.CDLL(path)
    vp, u64, u32p = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p
    lib.tpx3_plan.restype = ctypes.c_int
    lib.tpx3_plan.argtypes = [ctypes.POINTER(_CConfig), ctypes.POINTER(vp), ctypes.POINTER(ctypes.c_size_t)]
    lib.tpx3_cluster.restype = ctypes.c_int
    lib.tpx3_cluster.argtypes = [vp, vp, vp, u64, vp, vp, vp, vp, vp, vp, u32p]
    lib.tpx3_centroid.restype = ctypes.c_int
    lib.tpx3_centroid.argtypes = [vp, vp, vp, u64, vp, vp, vp, vp, vp, vp, u64, ctypes.POINTER(_CClusters), u32p]
    lib.tpx3_cluster_centroid.restype = ctypes.c_int
    lib.tpx3_cluster_centroid.argtypes = [vp, vp, vp, u64, vp, vp, vp, vp, vp, vp, u64,
                                          ctypes.POINTER(_CClusters), u32p]
    lib.tpx3_localmax_centroid.restype = ctypes.c_int
    lib.tpx3_localmax_centroid.argtypes = [vp, vp, vp, u64, vp, vp, vp, vp, ctypes.c_uint32, ctypes.c_uint32,
                                           ctypes.c_uint32, vp, vp, u64, ctypes.POINTER(_CClusters), u32p]
    lib.tpx3_unwrap_toa.restype = ctypes.c_int
    lib.tpx3_unwrap_toa.argtypes = [vp, vp, vp, u64, vp, u64, u64, ctypes.c_int64, ctypes.c_int, u64, vp, vp]
    lib.tpx3_unwrap_toa_static.restype = ctypes.c_int
    lib.tpx3_unwrap_toa_static.argtypes = [ctypes.c_int, vp, u64, vp, u64, u64, ctypes.c_int64, ctypes.c_int, u64, vp, vp]
    lib.tpx3_timewalk_table.restype = ctypes.c_int
    lib.tpx3_timewalk_table.argtypes = [ctypes.c_double] * 4 + [ctypes.c_uint32, vp]
    lib.tpx3_preprocess_cluster_centroid.restype = ctypes.c_int
    lib.tpx3_preprocess_cluster_centroid.argtypes = [vp, vp, vp, u64, vp, vp, vp, vp, u64, vp, u64, vp, ctypes.c_uint32,
                                                     u64, vp, vp, u64, ctypes.POINTER(_CClusters), u32p, u32p]
    lib.tpx3_preprocess.restype = ctypes.c_int
    lib.tpx3_preprocess.argtypes = [vp, vp, vp, u64, vp, vp, vp, vp, u64, vp, u64, vp, ctypes.c_uint32, u64,
                                    vp, vp, vp, vp, vp, vp]
    lib.tpx3_stream_bytes.restype = ctypes.c_size_t
    lib.tpx3_stream_bytes.argtypes = [u64, u64]
    lib.tpx3_stream_open.restype = ctypes.c_int
    lib.tpx3_stream_open.argtypes = [vp, vp, u64, u64, u64, vp, ctypes.POINTER(vp)]
    lib.tpx3_stream_push.restype = ctypes.c_int
    lib.tpx3_stream_push.argtypes = [vp, vp, vp, u64, vp, vp, vp, vp, ctypes.c_int, u64,
                                     ctypes.POINTER(_CClusters), vp, ctypes.POINTER(_CStreamInfo)]
    lib.tpx3_stream_close.restype = ctypes.c_int
    lib.tpx3_stream_close.argtypes = [vp]
    lib.tpx3_host_io_bytes.restype = ctypes.c_size_t
    lib.tpx3_host_io_bytes.argtypes = [u64, u64]
    lib.tpx3_process_host.restype = ctypes.c_int
    lib.tpx3_process_host.argtypes = [vp, vp, vp, vp, u64, vp, vp, vp, vp, vp, vp, u64,
                                      ctypes.POINTER(_CClusters), vp]
    lib.tpx3_host_route.restype = ctypes.c_int
    lib.tpx3_host_route.argtypes = [vp]
    lib.tpx3_status.restype = ctypes.c_int
    lib.tpx3_status.argtypes = [vp, vp, vp, ctypes.POINTER(_CStatus)]
    lib.tpx3_launch_count.restype = ctypes.c_uint64
    lib.tpx3_launch_count.argtypes = [vp]
    lib.tpx3_profile_enable.restype = ctypes.c_int
    lib.tpx3_profile_enable.argtypes = [vp, ctypes.c_int]
    lib.tpx3_profile_read.restype = ctypes.c_int
    lib.tpx3_profile_read.argtypes = [vp, ctypes.POINTER(_CProfile)]
    lib.tpx3_free.restype = ctypes.c_int
    lib.tpx3_free.argtypes = [vp]
    lib.tpx3_strerror.restype = ctypes.c_char_p
    lib.tpx3_strerror.argtypes = [ctypes.c_int]
    _lib = lib
    return lib


def timewalk_table(a: float, b: float, c: float, d: float, length: int):
    """Eq. 1 as an int32 numpy table in ticks (tpx3_timewalk_table, host only)."""
    import numpy as np

    out = np.empty(int(length), dtype=np.int32)
    rc = load_library().tpx3_timewalk_table(float(a), float(b), float(c), float(d), int(length), out.ctypes.data)
    if rc != OK:
        raise Tpx3Error(rc, "tpx3_timewalk_table")
    return out


def unwrap_toa_static(raw, modulus: int, jump: int, out, wraps_out, wraps_in: int = 0, prev_raw=None, stream=None):
    """tpx3_unwrap_toa_static: ToA unwrapping without a plan or workspace and without any device allocation (the
    scratch is a fixed array inside the library; n <= STATIC_UNWRAP_MAX). The caller passes every tensor, outputs
    included; calls that overlap on the GPU race on the shared scratch. Argument marshalling only."""
    import torch

    n = int(raw.numel())
    _check_dev(raw, torch.uint64, n, "raw")
    _check_dev(out, torch.uint64, n, "out")
    _check_dev(wraps_out, torch.int64, 1, "wraps_out")
    dev = raw.device
    rc = load_library().tpx3_unwrap_toa_static(dev.index if dev.index is not None else torch.cuda.current_device(),
                                               _stream_ptr(stream, dev), n, raw.data_ptr(), int(modulus), int(jump),
                                               int(wraps_in), 0 if prev_raw is None else 1,
                                               0 if prev_raw is None else int(prev_raw), out.data_ptr(),
                                               wraps_out.data_ptr())
    if rc != OK:
        raise Tpx3Error(rc, "tpx3_unwrap_toa_static")
    return out, wraps_out


def strerror(code: int) -> str:
    return load_library().tpx3_strerror(int(code)).decode()


@dataclass
class Config:
    sensor_w: int = 256
    sensor_h: int = 256
    toa_window_ticks: int = 320
    shot_period_ticks: int = 640000
    max_hits: int = 1 << 20
    device: int = 0
    flags: int = 0
    max_shot_hits: int = 0  # hint: most events in one shot; picks the fused path's window (0 = no hint: 2048, 4096, 8192 are tried on the device, tpx3.h)


_CLUSTER_FIELDS = (
    ("label", "uint32"), ("size", "uint32"), ("shot", "uint32"), ("sum_tot", "int64"), ("sum_tot_x", "int64"),
    ("sum_tot_y", "int64"), ("toa_peak", "uint64"), ("cx", "float32"), ("cy", "float32"),
    ("sum_tot_tof", "int64"), ("ctof", "float32"),
)


class Clusters:
    """Per-hit output arrays (structure of arrays) of capacity ``max_clusters``.
    device tensors (torch) or pinned host tensors, depending on who allocated them."""

    def __init__(self, max_clusters: int, device, pin: bool = False):
        import torch

        self.max_clusters = int(max_clusters)
        cap = max(self.max_clusters, 1)
        for name, dt in _CLUSTER_FIELDS:
            t = torch.empty(cap, dtype=getattr(torch, dt), device=device, pin_memory=pin)
            setattr(self, name, t)

    def _c(self) -> _CClusters:
        c = _CClusters()
        for name, _ in _CLUSTER_FIELDS:
            setattr(c, name, getattr(self, name).data_ptr())
        return c

    def numpy(self, n: int) -> dict:
        """First n entries of every array as numpy (keys prefixed c_, like the oracle's)."""
        return {"c_" + name: getattr(self, name)[:n].cpu().numpy() for name, _ in _CLUSTER_FIELDS}


def _stream_ptr(stream, device=None) -> int:
    import torch

    if stream is None:
        stream = torch.cuda.current_stream(device)   # of the plan's device, not of the current one
    return int(stream.cuda_stream)


def _check_host(t, dtype, n, name):
    import torch

    if not isinstance(t, torch.Tensor) or t.is_cuda:
        raise TypeError("%s must be a host (CPU) tensor" % name)
    if t.dtype != dtype or not t.is_contiguous() or t.numel() < n:
        raise TypeError("%s must be a contiguous %s host tensor with at least %d elements" % (name, dtype, n))


def _check_dev(t, dtype, n, name):
    import torch

    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("%s must be a CUDA tensor (there is no CPU path)" % name)
    if t.dtype != dtype or not t.is_contiguous() or t.numel() < n:
        raise TypeError("%s must be a contiguous %s tensor with at least %d elements" % (name, dtype, n))


class Plan:
    """tpx3_plan + a torch-allocated workspace on the plan's device."""

    def __init__(self, cfg: Config):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2603_04942_b200 needs a CUDA device; there is no CPU fallback")
        self.lib = load_library()
        self.cfg = cfg
        c = _CConfig(ctypes.sizeof(_CConfig), cfg.sensor_w, cfg.sensor_h, cfg.toa_window_ticks,
                     cfg.shot_period_ticks, cfg.max_hits, cfg.device, cfg.flags, cfg.max_shot_hits, 0)
        h = ctypes.c_void_p()
        ws = ctypes.c_size_t()
        rc = self.lib.tpx3_plan(ctypes.byref(c), ctypes.byref(h), ctypes.byref(ws))
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_plan")
        self.handle = h
        self.workspace_bytes = int(ws.value)
        self.device = torch.device("cuda", cfg.device)
        self.workspace = torch.empty(self.workspace_bytes, dtype=torch.uint8, device=self.device)
        self._io = None

    # -- S0-S3 ---------------------------------------------------------------------------------
    def cluster(self, x, y, toa, tot, perm=None, label=None, n_clusters=None, stream=None):
        import torch

        n = int(x.numel())
        self._check_inputs(x, y, toa, tot, n)
        perm = torch.empty(max(n, 1), dtype=torch.uint32, device=self.device) if perm is None else perm
        label = torch.empty(max(n, 1), dtype=torch.uint32, device=self.device) if label is None else label
        n_clusters = torch.empty(1, dtype=torch.uint32, device=self.device) if n_clusters is None else n_clusters
        rc = self.lib.tpx3_cluster(self.handle, self.workspace.data_ptr(), _stream_ptr(stream, self.device), n, x.data_ptr(),
                                   y.data_ptr(), toa.data_ptr(), tot.data_ptr(), perm.data_ptr(), label.data_ptr(),
                                   n_clusters.data_ptr())
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_cluster")
        return perm, label, n_clusters

    # -- preprocessing: trigger assignment, ToF cut, timewalk, rebase (PAPER.md IV.B-C) ------------
    def preprocess(self, x, y, toa, tot, trig, cut: int, table=None, shot_base: int = 0, stream=None):
        """Returns (x', y', toa', tot', index, n_out) — device tensors of capacity n and a device count."""
        import torch

        n = int(x.numel())
        self._check_inputs(x, y, toa, tot, n)
        _check_dev(trig, torch.uint64, 0, "trig")
        if table is not None:
            _check_dev(table, torch.int32, 0, "table")
        mk = lambda dt: torch.empty(max(n, 1), dtype=dt, device=self.device)  # noqa: E731
        xo, yo, to, oo, io = mk(torch.uint16), mk(torch.uint16), mk(torch.uint64), mk(torch.uint16), mk(torch.uint32)
        n_out = torch.empty(1, dtype=torch.uint32, device=self.device)
        rc = self.lib.tpx3_preprocess(self.handle, self.workspace.data_ptr(), _stream_ptr(stream, self.device), n, x.data_ptr(),
                                      y.data_ptr(), toa.data_ptr(), tot.data_ptr(), int(trig.numel()),
                                      trig.data_ptr(), int(cut), 0 if table is None else table.data_ptr(),
                                      0 if table is None else int(table.numel()), int(shot_base), xo.data_ptr(),
                                      yo.data_ptr(), to.data_ptr(), oo.data_ptr(), io.data_ptr(), n_out.data_ptr())
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_preprocess")
        return xo, yo, to, oo, io, n_out

    # -- preprocessing fused into the clustering call (tpx3.h) ---------------------------------------
    def preprocess_cluster_centroid(self, x, y, toa, tot, trig, cut: int, table, shot_base: int, clusters: "Clusters",
                                    perm=None, label=None, n_clusters=None, n_kept=None, stream=None):
        """Returns (perm, label, n_clusters, n_kept): perm[k] = input position of the surviving event at sorted
        position k; label over the surviving events. A stream the tile kernel cannot take shows as
        ERR_NOT_CONTIGUOUS in status()."""
        import torch

        n = int(x.numel())
        self._check_inputs(x, y, toa, tot, n)
        _check_dev(trig, torch.uint64, 0, "trig")
        if table is not None:
            _check_dev(table, torch.int32, 0, "table")
        mk = lambda k: torch.empty(k, dtype=torch.uint32, device=self.device)  # noqa: E731
        perm = mk(max(n, 1)) if perm is None else perm
        label = mk(max(n, 1)) if label is None else label
        n_clusters = mk(1) if n_clusters is None else n_clusters
        n_kept = mk(1) if n_kept is None else n_kept
        c = clusters._c()
        rc = self.lib.tpx3_preprocess_cluster_centroid(
            self.handle, self.workspace.data_ptr(), _stream_ptr(stream, self.device), n, x.data_ptr(), y.data_ptr(),
            toa.data_ptr(), tot.data_ptr(), int(trig.numel()), trig.data_ptr(), int(cut),
            0 if table is None else table.data_ptr(), 0 if table is None else int(table.numel()), int(shot_base),
            perm.data_ptr(), label.data_ptr(), clusters.max_clusters, ctypes.byref(c), n_clusters.data_ptr(),
            n_kept.data_ptr())
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_preprocess_cluster_centroid")
        return perm, label, n_clusters, n_kept

    # -- ToA counter unwrapping (PAPER.md IV.A) ----------------------------------------------------
    def unwrap_toa(self, raw, modulus: int, jump: int, wraps_in: int = 0, prev_raw=None, out=None, wraps_out=None,
                   stream=None):
        import torch

        n = int(raw.numel())
        _check_dev(raw, torch.uint64, n, "raw")
        out = torch.empty(max(n, 1), dtype=torch.uint64, device=self.device) if out is None else out
        wraps_out = torch.empty(1, dtype=torch.int64, device=self.device) if wraps_out is None else wraps_out
        rc = self.lib.tpx3_unwrap_toa(self.handle, self.workspace.data_ptr(), _stream_ptr(stream, self.device), n, raw.data_ptr(),
                                      int(modulus), int(jump), int(wraps_in), 0 if prev_raw is None else 1,
                                      0 if prev_raw is None else int(prev_raw), out.data_ptr(), wraps_out.data_ptr())
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_unwrap_toa")
        return out, wraps_out

    # -- paper-literal mode (local ToT maxima + box centroid, Eq. 3-9) ----------------
    def localmax_centroid(self, x, y, toa, tot, wx: int, wy: int, wt: int, clusters: "Clusters", perm=None,
                          lmax=None, n_hits=None, stream=None):
        import torch

        n = int(x.numel())
        self._check_inputs(x, y, toa, tot, n)
        perm = torch.empty(max(n, 1), dtype=torch.uint32, device=self.device) if perm is None else perm
        lmax = torch.empty(max(n, 1), dtype=torch.uint32, device=self.device) if lmax is None else lmax
        n_hits = torch.empty(1, dtype=torch.uint32, device=self.device) if n_hits is None else n_hits
        c = clusters._c()
        rc = self.lib.tpx3_localmax_centroid(self.handle, self.workspace.data_ptr(), _stream_ptr(stream, self.device), n,
                                             x.data_ptr(), y.data_ptr(), toa.data_ptr(), tot.data_ptr(), int(wx),
                                             int(wy), int(wt), perm.data_ptr(), lmax.data_ptr(),
                                             clusters.max_clusters, ctypes.byref(c), n_hits.data_ptr())
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_localmax_centroid")
        return perm, lmax, n_hits

    # -- S4-S5 ---------------------------------------------------------------------------------
    def centroid(self, x, y, toa, tot, perm, label, clusters: Clusters, n_clusters=None, stream=None):
        import torch

        n = int(x.numel())
        self._check_inputs(x, y, toa, tot, n)
        _check_dev(perm, torch.uint32, n, "perm")
        _check_dev(label, torch.uint32, n, "label")
        n_clusters = torch.empty(1, dtype=torch.uint32, device=self.device) if n_clusters is None else n_clusters
        c = clusters._c()
        rc = self.lib.tpx3_centroid(self.handle, self.workspace.data_ptr(), _stream_ptr(stream, self.device), n, x.data_ptr(),
                                    y.data_ptr(), toa.data_ptr(), tot.data_ptr(), perm.data_ptr(), label.data_ptr(),
                                    clusters.max_clusters, ctypes.byref(c), n_clusters.data_ptr())
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_centroid")
        return n_clusters

    # -- S0-S5 fused ---------------------------------------------------------------------------
    def cluster_centroid(self, x, y, toa, tot, clusters: Clusters, perm=None, label=None, n_clusters=None,
                         stream=None):
        import torch

        n = int(x.numel())
        self._check_inputs(x, y, toa, tot, n)
        perm = torch.empty(max(n, 1), dtype=torch.uint32, device=self.device) if perm is None else perm
        label = torch.empty(max(n, 1), dtype=torch.uint32, device=self.device) if label is None else label
        n_clusters = torch.empty(1, dtype=torch.uint32, device=self.device) if n_clusters is None else n_clusters
        c = clusters._c()
        rc = self.lib.tpx3_cluster_centroid(self.handle, self.workspace.data_ptr(), _stream_ptr(stream, self.device), n,
                                            x.data_ptr(), y.data_ptr(), toa.data_ptr(), tot.data_ptr(),
                                            perm.data_ptr(), label.data_ptr(), clusters.max_clusters,
                                            ctypes.byref(c), n_clusters.data_ptr())
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_cluster_centroid")
        return perm, label, n_clusters

    # -- chunked stream, cuts not shot-aligned -----------------------------
    def stream_open(self, max_chunk: int, max_carry: int, disorder_ticks: int = 0, stream=None) -> "Stream":
        return Stream(self, max_chunk, max_carry, disorder_ticks, stream)

    # -- end to end with host buffers ------------------------------------------------------------
    def process_host(self, x, y, toa, tot, clusters_host: Clusters, perm=None, label=None, stream=None) -> int:
        """x, y, toa, tot: host tensors (pinned for full copy speed). perm / label: host uint32
        tensors or None. Copies in, runs the fused call, copies out, synchronises. Returns the hit count."""
        import torch

        n = int(x.numel())
        for t, dt, name in ((x, torch.uint16, "x"), (y, torch.uint16, "y"), (toa, torch.uint64, "toa"), (tot, torch.uint16, "tot")):
            _check_host(t, dt, n, name)
        for t, name in ((perm, "perm"), (label, "label")):
            if t is not None:
                _check_host(t, torch.uint32, n, name)
        for name, dt in _CLUSTER_FIELDS:
            _check_host(getattr(clusters_host, name), getattr(torch, dt), min(clusters_host.max_clusters, 1), name)
        need = int(self.lib.tpx3_host_io_bytes(n, clusters_host.max_clusters))
        if self._io is None or self._io.numel() < need:
            self._io = torch.empty(need, dtype=torch.uint8, device=self.device)
        nc = ctypes.c_uint32(0)
        c = clusters_host._c()
        rc = self.lib.tpx3_process_host(
            self.handle, self.workspace.data_ptr(), self._io.data_ptr(), _stream_ptr(stream, self.device), n, x.data_ptr(),
            y.data_ptr(), toa.data_ptr(), tot.data_ptr(), perm.data_ptr() if perm is not None else None,
            label.data_ptr() if label is not None else None, clusters_host.max_clusters, ctypes.byref(c),
            ctypes.addressof(nc))
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_process_host")
        return int(nc.value)

    def status(self, stream=None) -> dict:
        s = _CStatus()
        rc = self.lib.tpx3_status(self.handle, self.workspace.data_ptr(), _stream_ptr(stream, self.device), ctypes.byref(s))
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_status")
        return {"error": -int(s.error), "path": int(s.path), "n_clusters": int(s.n_clusters),
                "sort_passes": int(s.sort_passes), "n": int(s.n)}

    def host_route(self) -> int:
        return int(self.lib.tpx3_host_route(self.handle))

    def launch_count(self) -> int:
        return int(self.lib.tpx3_launch_count(self.handle))

    def profile_enable(self, enable: bool = True):
        rc = self.lib.tpx3_profile_enable(self.handle, int(bool(enable)))
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_profile_enable")

    def profile_read(self) -> dict:
        """Summed per-stage device time (ms) and kernel launches since the last read."""
        pr = _CProfile()
        rc = self.lib.tpx3_profile_read(self.handle, ctypes.byref(pr))
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_profile_read")
        return {"calls": int(pr.calls), "ms": {k: float(pr.ms[i]) for i, k in enumerate(STAGES)},
                "launches": {k: int(pr.launches[i]) for i, k in enumerate(STAGES)}}

    def free(self):
        if self.handle:
            self.lib.tpx3_free(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass

    def _check_inputs(self, x, y, toa, tot, n):
        import torch

        _check_dev(x, torch.uint16, n, "x")
        _check_dev(y, torch.uint16, n, "y")
        _check_dev(toa, torch.uint64, n, "toa")
        _check_dev(tot, torch.uint16, n, "tot")
        if n > self.cfg.max_hits:
            raise Tpx3Error(ERR_INVALID_ARG, "n > max_hits")


class Stream:
    """tpx3_stream_open / _push / _close: argument marshalling only."""

    def __init__(self, pl: "Plan", max_chunk: int, max_carry: int, disorder_ticks: int, stream=None):
        import torch

        self.plan = pl
        self.buf = torch.empty(int(pl.lib.tpx3_stream_bytes(max_chunk, max_carry)), dtype=torch.uint8,
                               device=pl.device)
        h = ctypes.c_void_p()
        rc = pl.lib.tpx3_stream_open(pl.handle, self.buf.data_ptr(), max_chunk, max_carry, disorder_ticks,
                                     _stream_ptr(stream, pl.device), ctypes.byref(h))
        if rc != OK:
            raise Tpx3Error(rc, "tpx3_stream_open")
        self.handle = h

    def push(self, x, y, toa, tot, clusters: "Clusters", final: bool = False, n_hits=None, stream=None,
             want_info: bool = True):
        """Returns (n_hits device tensor, info dict). With want_info the call synchronises the stream once to read
        the per-push counts; without it nothing waits (info is None; a carry overflow shows in Plan.status())."""
        import torch

        pl = self.plan
        n = int(x.numel())
        pl._check_inputs(x, y, toa, tot, n)
        n_hits = torch.empty(1, dtype=torch.uint32, device=pl.device) if n_hits is None else n_hits
        c = clusters._c()
        info = _CStreamInfo()
        rc = pl.lib.tpx3_stream_push(self.handle, pl.workspace.data_ptr(), _stream_ptr(stream, pl.device), n, x.data_ptr(),
                                     y.data_ptr(), toa.data_ptr(), tot.data_ptr(), 1 if final else 0,
                                     clusters.max_clusters, ctypes.byref(c), n_hits.data_ptr(),
                                     ctypes.byref(info) if want_info else None)
        d = {k: int(getattr(info, k)) for k, _ in _CStreamInfo._fields_} if want_info else None
        if rc != OK:
            e = Tpx3Error(rc, "tpx3_stream_push")
            e.info = d
            raise e
        return n_hits, d

    def close(self):
        if self.handle:
            self.plan.lib.tpx3_stream_close(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def plan(cfg: Config) -> Plan:
    return Plan(cfg)


def shard_shots(n_shots: int, world_size: int, rank: int) -> tuple[int, int]:
    """Contiguous shot range [s0, s1) of `rank`: shots are independent units (no link crosses a
    shot boundary), so multi-GPU runs shard whole shots with no data-path collective."""
    base, rem = divmod(int(n_shots), int(world_size))
    s0 = rank * base + min(rank, rem)
    return s0, s0 + base + (1 if rank < rem else 0)
