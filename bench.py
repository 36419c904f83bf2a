#!/usr/bin/env python
"""bench.py — throughput of the TimePix3 cluster + centroid hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg1]

One "step" = one pass of the whole hot path (S0-S5: shot/key, stable sort, neighbour link, label
compression, segmented reduction, centroid — tpx3_cluster_centroid) over the whole synthetic
workload. Default workload: the largest streaming configuration of BASELINE.json, one shot-aligned
2^28-hit chunk of configs[4] (ion VMI with time of flight, delivery order locally shuffled, so the
in-tile sort runs; 3.76 GB of input: far larger than the 126 MB L2, so no explicit L2 flush is
needed between steps) — the configuration north_star's roofline target is stated on. The same line
carries the smaller chunk sizes of configs[4] (2^20 / 2^24 / 2^26 hits, `chunk_sweep`); the other
configs are `--workload cfg0..cfg3`. Metric: pixel hits/s clustered + centroided, device-timed.

Multi-GPU (torchrun, one rank per GPU): shots are independent units, so every rank processes its
own contiguous range of `shots` shots (rank r: shots [r*S, (r+1)*S)) with no data-path
collective; "scaling": "weak". torch.distributed is used for the barrier and the max-over-ranks
timing only.

Rank 0 prints ONE JSON line. `--impl reference` times the CPU oracle (oracle/) on a bounded
sample of the same workload on the host cores; it is a deliberately plain program,
a reported baseline and not the optimisation target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "pixel hits/sec clustered+centroided (device-timed, 1 B200); % of HBM peak"
UNIT = "pixel hits/s"
WORKLOADS = {  # name -> (generator config id, default shots)   [BASELINE.json configs]
    "cfg0": (0, 1000), "cfg1": (1, 100000), "cfg2": (2, 200000), "cfg3": (3, 50000),
    "cfg4_1M": (4, None), "cfg4_16M": (4, None), "cfg4_64M": (4, None), "cfg4_256M": (4, None),
}
CFG4_CHUNK = {"cfg4_1M": 1 << 20, "cfg4_16M": 1 << 24, "cfg4_64M": 1 << 26, "cfg4_256M": 1 << 28}
FALLBACK_HBM_GBS = 6650.0  # B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def make_workload(name: str, shots: int | None, rank: int):
    """Seeded synthetic input of the named BASELINE.json config (recipe: DESIGN.md 'Input recipe')."""
    import gen

    cfg_id, dflt = WORKLOADS[name]
    if cfg_id == 4:
        chunk = CFG4_CHUNK[name]
        # one shot-aligned chunk of config 4 (about 900 hits/shot): generate a little more than
        # needed and trim to the largest whole-shot prefix <= chunk hits
        s = shots if shots is not None else int(chunk / 850) + 64
        return gen.generate(4, shots=s, shot_begin=rank * s, max_hits=chunk)
    s = shots if shots is not None else dflt
    return gen.generate(cfg_id, shots=s, shot_begin=rank * s)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self, t0: float, t1: float) -> dict:
        sm, smax, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        rows = [r for t, r in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for _, r in self.rows[-3:]]
        for r in rows:
            f = [c.strip() for c in r.split(",")]
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
            except Exception:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def host_threads() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def time_oracle(w, shots: int, threads: int = 0):
    """Oracle (sort + per-shot BFS + sums + centroid) on the first `shots` shots; returns (seconds, hits, clusters)."""
    import oracle

    s = w.slice_shots(0, min(shots, w.shots))
    t0 = time.perf_counter()
    o = oracle.run(s.x, s.y, s.toa, s.tot, w.toa_window_ticks, w.shot_period_ticks, threads=threads)
    return time.perf_counter() - t0, s.n, o["n_clusters"]


def sized_oracle_sample(w, target_s: float):
    """Pick a whole-shot prefix of the workload that takes about target_s seconds of oracle time."""
    probe = max(1, min(w.shots, 2000))
    dt, hits, _ = time_oracle(w, probe)
    rate = hits / max(dt, 1e-6)
    per_shot = max(w.n / max(w.shots, 1), 1.0)
    shots = int(max(1, min(w.shots, rate * target_s / per_shot)))
    return shots


def cpu_baseline(w, target_s: float = 12.0) -> dict:
    shots = sized_oracle_sample(w, target_s)
    dt, hits, ncl = time_oracle(w, shots)
    return {"value": hits / dt, "unit": UNIT, "cores": host_threads(), "kind": "oracle",
            "sample": "first %d shots of %s (%d pixel hits, %d particle hits), %.2f s, OpenMP over shots; "
                      "sort is single-threaded" % (shots, w.name, hits, ncl, dt),
            "particle_hits_per_s": ncl / dt}


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    cfg_id, dflt = WORKLOADS[args.workload]
    # the oracle only ever sees a bounded sample: do not generate more shots than it can use
    cap = args.shots if args.shots is not None else (min(dflt, 20000) if dflt else 20000)
    w = make_workload(args.workload, cap, 0)
    per_step = max(0.5, min(5.0, 120.0 / max(args.steps + args.warmup, 1)))
    shots = sized_oracle_sample(w, per_step)
    for _ in range(args.warmup):
        time_oracle(w, shots)
    t_total, hits, ncl = 0.0, 0, 0
    for _ in range(args.steps):
        dt, hits, ncl = time_oracle(w, shots)
        t_total += dt
    ms = 1e3 * t_total / max(args.steps, 1)
    val = hits / (ms * 1e-3)
    sample = "first %d shots of %s per step (%d pixel hits, %d particle hits)" % (shots, w.name, hits, ncl)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": w.name, "shots": w.shots, "pixel_hits": w.n, "sample": sample,
                   "what": "CPU oracle (oracle/tpx3_oracle.cpp) on host cores; no GPU work"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": host_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# Algorithmic bytes: what the method must move once, per pixel hit and
# per particle hit. Inputs 14 B/hit (x, y, tot u16 + toa u64), outputs perm + label 8 B/hit,
# cluster row 64 B (label, size, shot u32; four i64 sums; toa_peak u64; cx, cy, ctof f32).
BYTES_PER_HIT_IN = 14
BYTES_PER_HIT_OUT = 8
BYTES_PER_CLUSTER = 64
STAGE_BYTES = {  # per stage of the general path: single-touch floor of that stage
    "fused": lambda n, c: (BYTES_PER_HIT_IN + BYTES_PER_HIT_OUT) * n + BYTES_PER_CLUSTER * c,
    "sort": lambda n, c: (8 + 4) * n,                      # read toa, write perm
    "link": lambda n, c: (4 + 6 + 8 + 4) * n,              # perm, x/y/tot gather, toa, label
    "centroid": lambda n, c: (4 + 4 + 6) * n + BYTES_PER_CLUSTER * c,
}


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2603_04942_b200 as m

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    m.load_library()  # fails loudly if libtpx3.so cannot be built / loaded

    w = make_workload(args.workload, args.shots, rank)
    n = w.n
    cfg = m.Config(max_hits=max(n, 1), toa_window_ticks=w.toa_window_ticks, shot_period_ticks=w.shot_period_ticks,
                   device=local, flags=(m.FLAG_FORCE_GENERAL if args.force_general else 0),
                   max_shot_hits=(args.max_shot_hits if args.max_shot_hits is not None
                                  else __import__("gen").max_shot_hits(w.cfg_id)))
    pl = m.plan(cfg)
    stream = torch.cuda.Stream(device=local)
    max_clusters = max(n // 2, 1024)  # hits have >= 3 pixels in every config; capacity errors are reported
    host = [torch.from_numpy(a).pin_memory() for a in (w.x, w.y, w.toa, w.tot)]
    dev = [t.to("cuda", non_blocking=True) for t in host]
    cl = m.Clusters(max_clusters, pl.device)
    perm = torch.empty(max(n, 1), dtype=torch.uint32, device=pl.device)
    label = torch.empty(max(n, 1), dtype=torch.uint32, device=pl.device)
    nc = torch.zeros(1, dtype=torch.uint32, device=pl.device)
    torch.cuda.synchronize()

    lm = args.mode == "localmax"
    wx, wy, wt = args.window

    split = args.mode == "split"

    def step():
        if lm:   # paper-literal mode: local ToT maxima + box centroid
            pl.localmax_centroid(*dev, wx, wy, wt, cl, perm=perm, lmax=label, n_hits=nc, stream=stream)
        elif split:   # the two calls BASELINE.json north_star names: tpx3_cluster (S0-S3), then tpx3_centroid (S4-S5)
            pl.cluster(*dev, perm=perm, label=label, n_clusters=nc, stream=stream)
            pl.centroid(*dev, perm, label, cl, n_clusters=nc, stream=stream)
        else:
            pl.cluster_centroid(*dev, cl, perm=perm, label=label, n_clusters=nc, stream=stream)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        step()
    barrier()
    st = pl.status(stream)
    if st["error"]:
        raise RuntimeError("device status error %d (%s)" % (st["error"], m.strerror(st["error"])))
    ncl = st["n_clusters"]

    # ---- timed region: K steps, device-timed with CUDA events on the launching stream ----------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    pl.profile_enable(True)
    pl.profile_read()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = pl.launch_count()
    barrier()
    t_wall0 = time.time()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    barrier()
    t_wall1 = time.time()
    launches = pl.launch_count() - l0
    ms_total = ev0.elapsed_time(ev1)
    prof = pl.profile_read()
    pl.profile_enable(False)
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
        tot = torch.tensor([n, ncl], dtype=torch.int64, device="cuda")
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
        n_all, ncl_all = int(tot[0].item()), int(tot[1].item())
    else:
        n_all, ncl_all = n, ncl
    ms_step = ms_total / max(args.steps, 1)
    value = n_all / (ms_step * 1e-3)

    # ---- the smaller chunk sizes of configs[4] (BASELINE.json: "Report hits/s and HBM GB/s per chunk size"):
    #      shot-aligned prefixes of the same stream, same plan, device-timed after the headline region ------
    sweep = None
    if w.cfg_id == 4 and not lm and world == 1 and not args.no_sweep:
        sweep = {}
        peak_gbs, _ = measured_peak()
        for cname, chunk in (("2^20", 1 << 20), ("2^24", 1 << 24), ("2^26", 1 << 26)):
            if chunk >= n:
                continue
            s1 = int(np.searchsorted(w.shot_offsets, chunk, side="right")) - 1
            mc = int(w.shot_offsets[s1])
            if mc == 0:
                continue
            views = [d[:mc] for d in dev]

            def cstep():
                pl.cluster_centroid(*views, cl, perm=perm, label=label, n_clusters=nc, stream=stream)

            for _ in range(3):
                cstep()
            torch.cuda.synchronize()
            c_ncl = int(nc.cpu().numpy()[0])
            reps = max(5, min(200, int((1 << 28) // mc)))
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                cstep()
            e1.record(stream)
            torch.cuda.synchronize()
            c_ms = e0.elapsed_time(e1) / reps
            c_bytes = STAGE_BYTES["fused"](mc, c_ncl)
            sweep[cname] = {"pixel_hits": mc, "particle_hits": c_ncl, "shots": s1, "ms_per_step": c_ms, "steps": reps,
                            "pixel_hits_per_s": mc / (c_ms * 1e-3), "algorithmic_gbs": c_bytes / (c_ms * 1e-3) / 1e9,
                            "frac_of_hbm_peak": c_bytes / (c_ms * 1e-3) / 1e9 / peak_gbs,
                            "l2": "fits the 126 MB L2: launch-latency bound, DRAM not exercised" if 22 * mc < 126e6
                                  else "larger than L2"}
        step()   # leave the full-size result in the output buffers
        torch.cuda.synchronize()

    # ---- end to end through the C ABI with HOST buffers (tpx3_process_host) --------------------
    clh = m.Clusters(ncl + 4096, "cpu", pin=True)   # host table for the hits the workload has (count known from the warm-up)

    def e2e_step():
        if not lm:
            return pl.process_host(*host, clh, stream=stream)  # synchronises the stream itself
        # no host-buffer entry point for this mode: pinned H2D copies, the call, D2H of the count and the table
        with torch.cuda.stream(stream):
            for d, h in zip(dev, host):
                d.copy_(h, non_blocking=True)
            step()
            k = int(nc.cpu().numpy()[0])
            for name, _ in m._CLUSTER_FIELDS:
                getattr(clh, name)[:k].copy_(getattr(cl, name)[:k], non_blocking=True)
        stream.synchronize()
        return k

    e2e_s = e2e_full_s = route_e2e = None
    if not args.no_e2e:
        for _ in range(2):
            e2e_step()
        barrier()
        e2e_steps = max(1, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            ncl_e2e = e2e_step()
        torch.cuda.synchronize()
        e2e_s = (time.perf_counter() - t0) / e2e_steps
        if world > 1:
            t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e2e_s = float(t.item())
        assert ncl_e2e == ncl, (ncl_e2e, ncl)
        route_e2e = pl.host_route()
        # the same call asking for perm and label as well (8 B/hit more on the way back; runs in one piece)
        e2e_full_s = None
        if not lm and world == 1:
            hperm = torch.empty(max(n, 1), dtype=torch.uint32).pin_memory()
            hlabel = torch.empty(max(n, 1), dtype=torch.uint32).pin_memory()
            pl.process_host(*host, clh, hperm, hlabel, stream=stream)
            t0 = time.perf_counter()
            for _ in range(2):
                pl.process_host(*host, clh, hperm, hlabel, stream=stream)
            torch.cuda.synchronize()
            e2e_full_s = (time.perf_counter() - t0) / 2
            del hperm, hlabel
    if rank == 0:
        sampler.stop()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant stage (CUDA-event time per stage, recorded on `stream`) ------
    peak, peak_src = measured_peak()
    stage_ms = {k: v / max(args.steps, 1) for k, v in prof["ms"].items()}   # per step (a step may be two calls)
    dom = max(stage_ms, key=lambda k: stage_ms[k])
    dom_bytes = STAGE_BYTES[dom](n, ncl)
    dom_gbs = dom_bytes / (stage_ms[dom] * 1e-3) / 1e9 if stage_ms[dom] > 0 else 0.0
    whole_bytes = STAGE_BYTES["fused"](n, ncl)
    roofline = {
        "bound": "hbm", "kernel": {"fused": "fused stage: k_fused_shot_tiles (95 %) + k_fused_compact", "sort": "general path: radix sort stage",
                                   "link": "general path: gather + hash link + compress stage",
                                   "centroid": "centroid stage"}[dom],
        "achieved": dom_gbs, "peak": peak, "unit": "GB/s", "frac": dom_gbs / peak, "traffic": None,
        "peak_source": peak_src, "algorithmic_bytes_per_launch": dom_bytes,
        "frac_of_nominal_8TBs": dom_gbs / 8000.0,    # BASELINE.json north_star quotes the nominal peak too
        "stage_ms": stage_ms, "stage_launches": {k: v / max(args.steps, 1) for k, v in prof["launches"].items()},
        "whole_path": {"algorithmic_bytes_per_step": whole_bytes,
                       "achieved": whole_bytes / (ms_step * 1e-3) / 1e9 * (n_all / max(n, 1)) / max(world, 1),
                       "frac": whole_bytes / (ms_step * 1e-3) / 1e9 / peak},
    }
    traffic_file = os.path.join(ROOT, "profiles", "traffic.json")  # ncu --set full dram bytes, per launch
    try:
        with open(traffic_file) as f:
            tr = json.load(f)
        key = "%s:%s:%d" % (w.name, dom, n)                   # a capture is of one workload size
        if key not in tr:
            key = "%s:%s" % (w.name, dom)
        if key in tr and tr[key].get("pixel_hits", n) == n:
            roofline["traffic"] = tr[key]["dram_bytes_per_launch"]
            roofline["traffic_source"] = tr[key].get("source")
            if stage_ms[dom] > 0:
                # achieved DRAM GB/s = ncu bytes (committed capture) / device time of this run's stage
                roofline["dram_gbs_from_traffic"] = tr[key]["dram_bytes_per_launch"] / (stage_ms[dom] * 1e-3) / 1e9
            wi = tr[key].get("warp_instructions_per_launch")
            if wi and stage_ms[dom] > 0:
                # what actually bounds the kernel: warp instructions issued per second against
                # 148 SMs x 4 schedulers x the SM clock; instruction count from the same ncu capture
                ipeak = 148 * 4 * 1965e6
                roofline["issue"] = {"achieved": wi / (stage_ms[dom] * 1e-3), "peak": ipeak, "unit": "warp instructions/s",
                                     "frac": wi / (stage_ms[dom] * 1e-3) / ipeak,
                                     "note": "peak = 148 SMs x 4 issue slots x 1965 MHz (B200_PROFILING.md unit counts)"}
    except Exception:
        pass

    cpu = None
    if world == 1 and not args.no_cpu_baseline and not lm:
        cpu = cpu_baseline(w, args.cpu_seconds)

    h2d = BYTES_PER_HIT_IN * n
    d2h = 4 + BYTES_PER_CLUSTER * ncl
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64", "data": "synthetic",
        "config": {
            "workload": w.name, "mode": ("paper-literal local maxima, box (wx, wy, wt) = (%d, %d, %d)" % (wx, wy, wt))
            if lm else ("connected components, tpx3_cluster then tpx3_centroid (two calls)" if split else "connected components (north_star)"), "shots_per_gpu": w.shots, "pixel_hits_per_gpu": n, "particle_hits_per_gpu": ncl,
            "pixel_hits_total": n_all, "particle_hits_total": ncl_all, "toa_window_ticks": w.toa_window_ticks,
            "shot_period_ticks": w.shot_period_ticks, "path": {1: "fused", 2: "general", 3: "localmax"}.get(st["path"], st["path"]),
            "sort_passes": st["sort_passes"], "max_shot_hits": cfg.max_shot_hits, "parallelism": "shots sharded over %d gpu(s), no collective" % world,
            "l2": "inputs (%.0f MB) larger than the 126 MB L2; no flush between steps" % (14 * n / 1e6)
                  if 14 * n > 2 * 126e6 else "inputs fit L2 (%.0f MB): DRAM traffic is not exercised" % (14 * n / 1e6),
            "input_hash": {"toa": __import__("gen").array_hash(w.toa), "x": __import__("gen").array_hash(w.x)},
        },
        "particle_hits_per_s": ncl_all / (ms_step * 1e-3),
        "e2e": None if e2e_s is None else {"value": n_all / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_s * 1e3, "route": {0: "one piece", 1: "pipelined in 2^22-event chunks", 2: "pipelined attempt redone in one piece"}.get(route_e2e) if not lm else None,
                "with_perm_label": None if e2e_full_s is None else {"value": n_all / e2e_full_s, "ms_per_step": e2e_full_s * 1e3,
                                                                   "d2h_bytes_per_step": d2h + 8 * n, "route": "one piece"}, "api": "tpx3_process_host (pinned host buffers; cluster table copied "
                "back, perm/label left on the device)" if not lm else "pinned H2D copies + tpx3_localmax_centroid + "
                "D2H of the count and the hit table"},
        "gpu_launches": launches,
        "roofline": roofline,
        "clocks": sampler.summary(t_wall0, time.time()),
        "context": "paper: ~25x faster than acquisition at 1 kHz, ~10 particles/shot, PyTorch on a Titan RTX "
                   "(PAPER.md:179) ~ 2.5e5 particle hits/s; other hardware, context only",
    }
    if cpu is not None:
        line["cpu_baseline"] = cpu
    if sweep is not None:
        line["chunk_sweep"] = sweep
    print(json.dumps(line), flush=True)
    pl.free()
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_stream(args):
    """--mode stream: one step = the whole workload pushed through tpx3_stream_push in chunks of --chunk events
    cut anywhere (last clause). Single GPU; a secondary bench line (no cpu_baseline)."""
    import numpy as np
    import torch

    import paper_2603_04942_b200 as m

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(0)
    m.load_library()
    w = make_workload(args.workload, args.shots, 0)
    n, chunk, carry = w.n, args.chunk, args.max_carry
    t = w.toa.astype(np.int64)
    D = int(np.max(np.maximum.accumulate(t) - t)) if n else 0
    cfg = m.Config(max_hits=chunk + carry, toa_window_ticks=w.toa_window_ticks, shot_period_ticks=w.shot_period_ticks,
                   max_shot_hits=(args.max_shot_hits if args.max_shot_hits is not None
                                  else __import__("gen").max_shot_hits(w.cfg_id)))
    pl = m.plan(cfg)
    stream = torch.cuda.Stream(device=0)
    dev = [torch.from_numpy(a).cuda() for a in (w.x, w.y, w.toa, w.tot)]
    cl = m.Clusters(max((chunk + carry) // 2, 1024), pl.device)
    nc = torch.zeros(1, dtype=torch.uint32, device=pl.device)
    cuts = list(range(0, n, chunk)) + [n]
    torch.cuda.synchronize()

    def step(count=False):
        s = pl.stream_open(chunk, carry, D, stream=stream)
        hits = emitted = late = max_carry_seen = 0
        for a, b in zip(cuts[:-1], cuts[1:]):
            # timed steps: nothing waits on the host (no per-push counts); the counting step reads them
            _, info = s.push(*(d[a:b] for d in dev), cl, final=(b == n), n_hits=nc, stream=stream, want_info=count)
            if count:
                emitted += info["n_emitted"]
                late += info["n_late"]
                max_carry_seen = max(max_carry_seen, info["n_carry"])
                stream.synchronize()
                hits += int(nc.cpu().numpy()[0])
        s.close()
        return hits, emitted, late, max_carry_seen

    for _ in range(max(args.warmup, 1)):
        ncl, emitted, late, carried = step(count=True)
    assert emitted == n and late == 0, (emitted, n, late)
    st = pl.status(stream)
    if st["error"]:
        raise RuntimeError("device status error %d" % st["error"])
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.3)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    l0 = pl.launch_count()
    t_wall0 = time.time()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    torch.cuda.synchronize()
    launches = pl.launch_count() - l0
    ms_step = ev0.elapsed_time(ev1) / max(args.steps, 1)
    sampler.stop()
    peak, peak_src = measured_peak()
    # the stream layer reads ToA twice (sample + mark: 8 B, scatter: 8 B) and moves every event once (6 + 14 B)
    bytes_step = STAGE_BYTES["fused"](n, ncl) + 36 * n
    line = {
        "metric": METRIC, "value": n / (ms_step * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64", "data": "synthetic",
        "config": {"workload": w.name, "mode": "chunked stream, cuts not shot-aligned (tpx3_stream_push)",
                   "chunk_events": chunk, "pushes_per_step": len(cuts) - 1, "max_carry": carry,
                   "largest_carry_seen": carried, "disorder_ticks": D, "pixel_hits_per_gpu": n,
                   "particle_hits_per_gpu": ncl, "max_shot_hits": cfg.max_shot_hits,
                   "path": {1: "fused", 2: "general"}.get(st["path"], st["path"])},
        "particle_hits_per_s": ncl / (ms_step * 1e-3),
        "gpu_launches": launches,
        "roofline": {"bound": "hbm", "kernel": "whole push: stream split (3 kernels) + fused stage", "achieved":
                     bytes_step / (ms_step * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": bytes_step / (ms_step * 1e-3) / 1e9 / peak, "traffic": None, "peak_source": peak_src,
                     "algorithmic_bytes_per_step": bytes_step},
        "clocks": sampler.summary(t_wall0, time.time()),
    }
    print(json.dumps(line), flush=True)
    pl.free()
    return 0


def run_sweep1g(args):
    """--mode sweep1g: BASELINE.json configs[4] to the letter: 10^9 pixel hits of the streaming config (whole shots, four
    parts of up to 2^28 hits generated one after the other and kept resident: 14 GB), processed in shot-aligned chunks of
    2^20, 2^24, 2^26 and 2^28 hits, one tpx3_cluster_centroid call per chunk; per chunk size the time of ONE pass over all
    10^9 hits, device-timed. Single GPU; a secondary bench line (the default line times one 2^28 chunk)."""
    import torch

    import gen
    import paper_2603_04942_b200 as m

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(0)
    m.load_library()
    big = 1 << 28
    target = 10 ** 9
    parts, total, shot_begin = [], 0, 0
    while total < target:
        w = gen.generate(4, shots=int(big / 850) + 64, shot_begin=shot_begin, max_hits=min(big, target - total + 2000))
        shot_begin += w.shots
        total += w.n
        parts.append(([torch.from_numpy(a).cuda() for a in (w.x, w.y, w.toa, w.tot)], w.shot_offsets.copy(),
                      {sz: w.chunks(sz) for sz in (1 << 20, 1 << 24, 1 << 26, big)}, w.n))
        del w
    pl = m.plan(m.Config(max_hits=big, toa_window_ticks=gen.TOA_WINDOW_TICKS, shot_period_ticks=gen.SHOT_PERIOD_TICKS,
                         max_shot_hits=gen.max_shot_hits(4)))
    stream = torch.cuda.Stream(device=0)
    cl = m.Clusters(big // 8, pl.device)
    perm = torch.empty(big, dtype=torch.uint32, device=pl.device)
    label = torch.empty(big, dtype=torch.uint32, device=pl.device)
    nc = torch.zeros(1, dtype=torch.uint32, device=pl.device)

    def one_pass(size, count=False):
        hits = calls = 0
        for dev, off, chunks, _ in parts:
            for s0, s1 in chunks[size]:
                a, b = int(off[s0]), int(off[s1])
                pl.cluster_centroid(*(d[a:b] for d in dev), cl, perm=perm, label=label, n_clusters=nc, stream=stream)
                calls += 1
                if count:
                    stream.synchronize()
                    st = pl.status(stream)
                    if st["error"] or st["path"] != 1:
                        raise RuntimeError("chunk [%d, %d): %r" % (a, b, st))
                    hits += st["n_clusters"]
        return hits, calls

    peak, peak_src = measured_peak()
    sampler = ClockSampler(0)
    sampler.start()
    t_wall0 = time.time()
    sweep, ncl = {}, None
    for name, size in (("2^28", big), ("2^26", 1 << 26), ("2^24", 1 << 24), ("2^20", 1 << 20)):
        hits, calls = one_pass(size, count=True)             # warm-up pass; also counts the hits and checks every call
        if ncl is None:
            ncl = hits
        assert hits == ncl, (name, hits, ncl)                 # the rows do not depend on the chunk size
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = max(args.steps, 1) if size >= (1 << 24) else 1
        e0.record(stream)
        for _ in range(reps):
            one_pass(size)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        nbytes = STAGE_BYTES["fused"](total, ncl)
        sweep[name] = {"calls_per_pass": calls, "ms_per_pass": ms, "pixel_hits_per_s": total / (ms * 1e-3),
                       "particle_hits_per_s": ncl / (ms * 1e-3), "algorithmic_gbs": nbytes / (ms * 1e-3) / 1e9,
                       "frac_of_hbm_peak": nbytes / (ms * 1e-3) / 1e9 / peak}
    sampler.stop()
    head = sweep["2^28"]
    line = {
        "metric": METRIC, "value": head["pixel_hits_per_s"], "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": 1, "ms_per_step": head["ms_per_pass"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64", "data": "synthetic",
        "config": {"workload": "cfg4_streaming, 10^9 pixel hits in %d resident parts" % len(parts), "mode": "sweep1g",
                   "pixel_hits_total": total, "particle_hits_total": ncl, "max_shot_hits": gen.max_shot_hits(4),
                   "what": "one step = one pass over all hits, one tpx3_cluster_centroid call per shot-aligned chunk"},
        "chunk_sweep": sweep,
        "roofline": {"bound": "hbm", "kernel": "fused stage, whole pass in 2^28-hit chunks", "achieved": head["algorithmic_gbs"],
                     "peak": peak, "unit": "GB/s", "frac": head["frac_of_hbm_peak"], "traffic": None, "peak_source": peak_src},
        "clocks": sampler.summary(t_wall0, time.time()),
    }
    print(json.dumps(line), flush=True)
    pl.free()
    return 0


def run_aux(args):
    """--mode unwrap | preprocess: the two preprocessing calls of SURVEY.md 8f NEXT #4 / #3 on the workload's
    events (device-resident, device-timed), against the HBM roofline of their algorithmic bytes."""
    import numpy as np
    import torch

    import paper_2603_04942_b200 as m

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(0)
    m.load_library()
    w = make_workload(args.workload, args.shots, 0)
    n, P = w.n, w.shot_period_ticks
    pl = m.plan(m.Config(max_hits=max(n, 1), toa_window_ticks=w.toa_window_ticks, shot_period_ticks=P,
                         max_shot_hits=__import__("gen").max_shot_hits(w.cfg_id)))
    stream = torch.cuda.Stream(device=0)
    two_calls = None
    if args.mode == "unwrap":
        # the workload's ToA folded into a counter of 2^34 ticks (several wraps over the run)
        modulus, jump = 1 << 34, 1 << 33
        raw = torch.from_numpy((w.toa % np.uint64(modulus)).astype(np.uint64)).cuda()
        out = torch.empty_like(raw)
        wr = torch.empty(1, dtype=torch.int64, device="cuda")
        step = lambda: pl.unwrap_toa(raw, modulus, jump, out=out, wraps_out=wr, stream=stream)  # noqa: E731
        bytes_step = 16 * n
        what = {"call": "tpx3_unwrap_toa", "modulus": modulus, "jump": jump}
    else:
        # irregular triggers, timewalk added to every pixel, every 10th event turned into a dark count past the cut
        shot = (w.toa // np.uint64(P)).astype(np.int64)
        s0 = int(shot.min())
        nshot = int(shot.max()) - s0 + 1
        trig = (np.arange(nshot, dtype=np.int64) + s0) * P + 1000 * (np.arange(nshot) % 7)
        table = m.timewalk_table(2000.0, 2.0, 3.0, 1.2, 1024)
        cut = 64000
        toa = trig[shot - s0] + (w.toa.astype(np.int64) - shot * P) + table[np.minimum(w.tot, 1023)]
        dark = np.arange(n) % 10 == 0
        toa[dark] = trig[shot[dark] - s0] + cut + 1 + (np.arange(n)[dark] % 1000)
        dev = [torch.from_numpy(a).cuda() for a in (w.x, w.y, toa.astype(np.uint64), w.tot)]
        dtrig = torch.from_numpy(trig.astype(np.uint64)).cuda()
        dtab = torch.from_numpy(table).cuda()
        res = {}

        def step():
            res["out"] = pl.preprocess(*dev, dtrig, cut, dtab, shot_base=s0, stream=stream)

        step()
        torch.cuda.synchronize()
        kept = int(res["out"][5].cpu().numpy()[0])
        bytes_step = 14 * n + 18 * kept + 4 * kept
        what = {"call": "tpx3_preprocess", "triggers": nshot, "cut_ticks": cut, "kept": kept, "dropped": n - kept}
        if args.mode == "prefused":
            # SURVEY 8f NEXT #3 as worded: the preprocessing inside the clustering call, against the two calls back to back
            cl = m.Clusters(max(n // 2, 1024), pl.device)
            perm = torch.empty(max(n, 1), dtype=torch.uint32, device=pl.device)
            label = torch.empty(max(n, 1), dtype=torch.uint32, device=pl.device)
            nc = torch.zeros(1, dtype=torch.uint32, device=pl.device)
            nk = torch.zeros(1, dtype=torch.uint32, device=pl.device)

            def two():
                xo, yo, to, oo, io, no = pl.preprocess(*dev, dtrig, cut, dtab, shot_base=s0, stream=stream)
                pl.cluster_centroid(xo[:kept], yo[:kept], to[:kept], oo[:kept], cl, perm=perm, label=label, n_clusters=nc,
                                    stream=stream)

            def step():
                pl.preprocess_cluster_centroid(*dev, dtrig, cut, dtab, s0, cl, perm=perm, label=label, n_clusters=nc,
                                               n_kept=nk, stream=stream)

            for _ in range(max(args.warmup, 1)):
                two()
            torch.cuda.synchronize()
            ncl_two = int(nc.cpu().numpy()[0])
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(args.steps):
                two()
            e1.record(stream)
            torch.cuda.synchronize()
            two_calls = e0.elapsed_time(e1) / max(args.steps, 1)
            step()
            torch.cuda.synchronize()
            st = pl.status(stream)
            if st["error"] or int(nc.cpu().numpy()[0]) != ncl_two or int(nk.cpu().numpy()[0]) != kept:
                raise RuntimeError("fused preprocessing call disagrees with the two calls: %r" % (st,))
            ncl = ncl_two
            bytes_step = 8 * n + 14 * n + 8 * kept + 64 * ncl     # pre-pass ToA + the tile kernel's single touch
            what = {"call": "tpx3_preprocess_cluster_centroid", "triggers": nshot, "cut_ticks": cut, "kept": kept,
                    "dropped": n - kept, "particle_hits": ncl}
    for _ in range(max(args.warmup, 1)):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.3)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = pl.launch_count()
    t_wall0 = time.time()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    torch.cuda.synchronize()
    launches = pl.launch_count() - l0
    ms_step = ev0.elapsed_time(ev1) / max(args.steps, 1)
    sampler.stop()
    peak, peak_src = measured_peak()
    what.update({"workload": w.name, "mode": args.mode, "pixel_hits_per_gpu": n})
    if two_calls is not None:
        what.update({"two_calls_ms_per_step": two_calls, "speedup_over_two_calls": two_calls / ms_step})
    line = {
        "metric": METRIC, "value": n / (ms_step * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64", "data": "synthetic", "config": what, "gpu_launches": launches,
        "roofline": {"bound": "hbm", "kernel": what["call"] + (" (3 kernels)" if two_calls is None else " (pre-pass + tile kernel)"), "achieved": bytes_step / (ms_step * 1e-3) / 1e9,
                     "peak": peak, "unit": "GB/s", "frac": bytes_step / (ms_step * 1e-3) / 1e9 / peak, "traffic": None,
                     "peak_source": peak_src, "algorithmic_bytes_per_step": bytes_step},
        "clocks": sampler.summary(t_wall0, time.time()),
    }
    print(json.dumps(line), flush=True)
    pl.free()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--workload", choices=sorted(WORKLOADS), default="cfg4_256M")
    ap.add_argument("--shots", type=int, default=None, help="override the number of shots (testing only)")
    ap.add_argument("--force-general", action="store_true", help="never take the fused shot-tile path")
    ap.add_argument("--max-shot-hits", type=int, default=None,
                    help="tile-size hint for the plan (default: the workload recipe's bound on hits per shot)")
    ap.add_argument("--chunk", type=int, default=1 << 22, help="--mode stream: events per push")
    ap.add_argument("--max-carry", type=int, default=1 << 20, help="--mode stream: carry capacity in events")
    ap.add_argument("--mode", choices=("components", "split", "localmax", "stream", "unwrap", "preprocess", "prefused", "sweep1g"), default="components",
                    help="components: the hot path (default). localmax: the paper-literal mode, SURVEY 8f NEXT #2")
    ap.add_argument("--window", type=int, nargs=3, default=(2, 2, 320), metavar=("WX", "WY", "WT"),
                    help="box half-widths of --mode localmax (pixels, pixels, ticks)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="development only: skip the end-to-end (host buffer) leg")
    ap.add_argument("--no-sweep", action="store_true", help="cfg4 workloads: skip the smaller chunk sizes")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print("note: timing rules ask for >= 3 warm-up steps", file=sys.stderr)
    if args.impl == "reference":
        return run_reference(args)
    if args.mode == "sweep1g":
        return run_sweep1g(args)
    if args.mode in ("unwrap", "preprocess", "prefused"):
        return run_aux(args)
    return run_stream(args) if args.mode == "stream" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
