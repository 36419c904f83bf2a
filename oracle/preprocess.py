"""ORACLE — TEST INFRASTRUCTURE ONLY (see oracle/tpx3_oracle.cpp header).

Plain, sequential CPU definitions of the paper's preprocessing steps (section IV), written in the
paper's order with Python integers (no overflow games). They share no code with the CUDA path.

  unwrap_toa   section IV.A, PAPER.md:58-62   ToA counter unwrapping
  StreamModel  SURVEY.md 8f NEXT #3, last clause: chunk cuts that are not shot-aligned (R24)
"""
from __future__ import annotations

import numpy as np


def unwrap_toa(raw, modulus: int, jump: int, wraps_in: int = 0, prev_raw=None):
    """"Each time the ToA of the next pixel or TDC is more than 20 seconds less than the previous
    one, the global counter of time wrappings is incremented by one and the appropriate integer multiple of
    fundamental time units is added to all subsequent data in the stream." PAPER.md:62 (the out-of-order edge
    case): "both large negative and large positive jumps are tracked in the ToA and the appropriate time
    unwrapping adjustment is applied in each case" — a jump UP by more than the threshold is an event from
    before the wrap reported after it, and takes the counter back down by one (reading R22).

    raw: counter values in [0, modulus); modulus: the counter period (2^42 units for pixels, 2^44 for TDCs,
    PAPER.md:58) in the caller's tick; jump: the "20 seconds" threshold in ticks, strict (">").
    wraps_in / prev_raw carry the state across calls (chunks). Returns (unwrapped uint64[n], wraps_out)."""
    raw_l = [int(v) for v in np.asarray(raw)]
    out = np.empty(len(raw_l), dtype=np.uint64)
    wraps = int(wraps_in)
    prev = None if prev_raw is None else int(prev_raw)
    for i, v in enumerate(raw_l):
        if prev is not None:
            if prev - v > jump:       # large negative shift: the counter wrapped
                wraps += 1
            elif v - prev > jump:     # large positive shift: a pre-wrap event reported late (or the way back)
                wraps -= 1
        out[i] = (v + wraps * modulus) % (1 << 64)
        prev = v
    return out, wraps


def timewalk_table(a: float, b: float, c: float, d: float, length: int) -> np.ndarray:
    """Eq. 1: dToF(ToT; a, b, c, d) = a / (ToT + b)^d + c, evaluated in fp64 for ToT = 0 ..
    length-1 and rounded to the nearest integer tick (half away from zero) — the calibration product that
    is "applied to every pixel in the data stream". a, c in ticks; ToT, b in ToT units."""
    out = np.empty(length, dtype=np.int32)
    for tot in range(length):
        base = float(tot) + float(b)
        v = float(a) / (base ** float(d)) + float(c) if base > 0.0 else float(c)
        out[tot] = int(np.floor(abs(v) + 0.5)) * (1 if v >= 0 else -1)
    return out


def preprocess(x, y, toa, tot, trig, cut: int, table, P_out: int, shot_base: int = 0):
    """Section IV.B-C in the paper's order, event by event:
      shot    s = the most recent laser trigger: the largest s with trig[s] <= toa;
              events before the first trigger have none and are dropped
      cut     ToF = toa - trig[s]; the event is written "only ... if its ToF does not exceed 100 us"
              (PAPER.md:68): keep iff ToF <= cut
      walk    ToF' = ToF - dToF(ToT) with the calibrated table (Eq. 1, :74-76; ToT beyond the table uses its
              last entry), clamped to [0, P_out - 1] (reading R23)
      rebase  toa' = (shot_base + s) * P_out + ToF', so that downstream `shot = toa' div P_out` is the
              trigger index (reading R6 made exact)
    Kept events stay in stream order. Returns x', y', toa', tot' and the kept input indices."""
    trig_l = [int(t) for t in np.asarray(trig)]
    table = np.asarray(table, dtype=np.int64)
    xs, ys, ts, os_, idx = [], [], [], [], []
    for i, t in enumerate(int(v) for v in np.asarray(toa)):
        lo, hi = 0, len(trig_l)          # bisect_right
        while lo < hi:
            mid = (lo + hi) // 2
            if trig_l[mid] <= t:
                lo = mid + 1
            else:
                hi = mid
        s = lo - 1
        if s < 0:
            continue
        tof = t - trig_l[s]
        if tof > cut:
            continue
        tt = int(tot[i])
        corr = int(table[min(tt, len(table) - 1)]) if len(table) else 0
        tofc = min(max(tof - corr, 0), P_out - 1)
        xs.append(int(x[i])); ys.append(int(y[i])); os_.append(tt); idx.append(i)
        ts.append((shot_base + s) * P_out + tofc)
    return (np.array(xs, dtype=np.uint16), np.array(ys, dtype=np.uint16), np.array(ts, dtype=np.uint64),
            np.array(os_, dtype=np.uint16), np.array(idx, dtype=np.int64))


class StreamModel:
    """Chunked processing of an endless stream whose chunk cuts fall anywhere (SURVEY.md 8f NEXT #3:
    "chunk cuts that are not shot-aligned"). The definition it must reproduce is the batch one: the hits of
    the whole stream, because "each pixel [is] associated with the most recent laser trigger"
    and no hit crosses a shot (reading R6) — so a chunk may be cut anywhere as long as every shot is
    clustered in ONE piece. Reading R24, step by step for one push of a chunk (plain lists, stream order):

      1. t_max = the largest ToA of everything seen so far, this chunk included. The stream promises a
         bounded disorder D: no later event has ToA < (largest ToA so far) - D (pixels report
         out of order, dimmer ones first). (Any lower bound of t_max keeps step 2 safe: it only emits a
         shot later. What a push emits is therefore not part of the definition; the rows of all pushes are.)
      2. s_cut = max(s_emitted, (t_max - D) div P): every shot below s_cut is complete. final: s_cut = inf.
      3. working set = carried events ++ chunk, in that order (the carried ones came first in the stream):
           shot <  s_emitted  -> late (its shot went out already): dropped and counted
           shot <  s_cut      -> emitted now: one batch call on exactly these events, in stream order
           otherwise          -> carried to the next push, in stream order
      4. s_emitted = s_cut.
    Returns per push the emitted events; the caller clusters them with the batch oracle. With no late event
    the emitted sets, concatenated, are the stream re-cut at shot boundaries, so their hits in order are the
    batch hits of the whole stream and `label_base` (events emitted before) makes the labels global."""

    def __init__(self, P: int, D: int):
        assert P > 0
        self.P, self.D = int(P), int(D)
        self.t_max = 0
        self.s_emitted = 0
        self.label_base = 0
        self.carry = []          # (x, y, toa, tot) tuples in stream order
        self.late_total = 0

    def push(self, x, y, toa, tot, final: bool = False):
        chunk = [(int(a), int(b), int(c), int(d)) for a, b, c, d in zip(x, y, toa, tot)]
        for ev in chunk:
            self.t_max = max(self.t_max, ev[2])
        if final:
            s_cut = None
        else:
            s_cut = max(self.s_emitted, (self.t_max - self.D) // self.P if self.t_max >= self.D else 0)
        emit, keep, late = [], [], 0
        for ev in self.carry + chunk:
            s = ev[2] // self.P
            if s < self.s_emitted:
                late += 1
            elif s_cut is None or s < s_cut:
                emit.append(ev)
            else:
                keep.append(ev)
        self.carry = keep
        if s_cut is not None:
            self.s_emitted = s_cut
        self.late_total += late
        base = self.label_base
        self.label_base += len(emit)
        cols = list(zip(*emit)) if emit else [[], [], [], []]
        return {"x": np.array(cols[0], dtype=np.uint16), "y": np.array(cols[1], dtype=np.uint16),
                "toa": np.array(cols[2], dtype=np.uint64), "tot": np.array(cols[3], dtype=np.uint16),
                "n_late": late, "n_carry": len(keep), "label_base": base}
