"""ORACLE — TEST INFRASTRUCTURE ONLY (see oracle/tpx3_oracle.cpp header).

Plain, sequential CPU definitions of the paper's preprocessing steps (section IV), written in the
paper's order with Python integers (no overflow games). They share no code with the CUDA path.

  unwrap_toa   section IV.A, PAPER.md:58-62   ToA counter unwrapping
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
