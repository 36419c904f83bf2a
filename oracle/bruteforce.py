"""ORACLE — TEST INFRASTRUCTURE ONLY (see oracle/tpx3_oracle.cpp header).

Dense, paper-literal array formulation for TINY inputs (n <= a few hundred), written directly
from the equations so that it can be checked against the paper by eye. It pins the C++ oracle
(BFS) and replays the paper's worked example. Shares no code with the CUDA path nor with
tpx3_oracle.cpp.

  distance_matrix      Eq. 3   D_ij = X_j - X_i
  adjacency_1d         Eq. 4   A_ij = [|D_ij| <= w]   (inclusive)
  adjacency            Eq. 5   A = A^X (.) A^Y (.) A^ToF  (+ same-shot mask)
  masked_tot           Eq. 6   M_ij = ToT_j * A_ij
  local_maxima         Eq. 7   rows of M - M^T whose maximum is 0
  box_centroid         Eq. 9   sum_j X_j A_ij ToT_j / sum_j ToT_j A_ij
  components           transitive closure of A (north_star's "hit"), min-label fixed point
  cluster_bruteforce   the whole north_star path by brute force
"""
from __future__ import annotations

import numpy as np


def distance_matrix(v) -> np.ndarray:
    """Eq. 3: the repeated matrix {{X_i}} minus its transpose, D_ij = X_j - X_i."""
    v = np.asarray(v, dtype=np.int64)
    rep = np.tile(v[None, :], (v.shape[0], 1))
    return rep - rep.T


def adjacency_1d(v, w: int) -> np.ndarray:
    """Eq. 4: A_ij = 1 where |D_ij| <= w (inclusive)."""
    return (np.abs(distance_matrix(v)) <= w).astype(np.int64)


def adjacency(x, y, t, wx: int, wy: int, wt: int, shot=None) -> np.ndarray:
    """Eq. 5: Hadamard product of the three 1-D adjacency matrices; optionally AND same shot.
    The diagonal is 1 as in the paper (A_ii = 1, Eq. 4)."""
    a = adjacency_1d(x, wx) * adjacency_1d(y, wy) * adjacency_1d(t, wt)
    if shot is not None:
        s = np.asarray(shot, dtype=np.int64)
        a = a * (s[None, :] == s[:, None]).astype(np.int64)
    return a


def masked_tot(tot, a) -> np.ndarray:
    """Eq. 6: (ToT_ij) (.) (A_ij) with ToT_ij the repeated ToT array, i.e. M_ij = ToT_j A_ij."""
    tot = np.asarray(tot)
    return np.tile(tot[None, :], (tot.shape[0], 1)) * a


def local_maxima(tot, a, lift: str = "paper") -> np.ndarray:
    """Eq. 7 + tie rule: indices i whose row of M - M^T has maximum 0.

    lift="paper": add 0.001*i to ToT (floating point, as printed).
    lift="lex":   integer lexicographic (tot, i): ToT*n + i (same intent, exact for any n).
    lift="none":  no tie-breaking.
    """
    tot = np.asarray(tot)
    n = tot.shape[0]
    if lift == "paper":
        t = tot.astype(np.float64) + 0.001 * np.arange(n)
    elif lift == "lex":
        t = tot.astype(np.int64) * n + np.arange(n)
    else:
        t = tot.astype(np.int64)
    m = masked_tot(t, a)
    anti = m - m.T
    return np.nonzero(anti.max(axis=1) == 0)[0]


def box_centroid(v, tot, a) -> np.ndarray:
    """Eq. 9: centroid about every pixel i over its neighbourhood row A_i. (float64)"""
    v = np.asarray(v, dtype=np.float64)
    tot = np.asarray(tot, dtype=np.float64)
    return (a * (v * tot)[None, :]).sum(axis=1) / (a * tot[None, :]).sum(axis=1)


def components(a) -> np.ndarray:
    """Connected components of the relation A (i != j): label = min index, by repeated
    neighbour-minimum until nothing changes."""
    n = a.shape[0]
    lab = np.arange(n, dtype=np.int64)
    nb = a.astype(bool) | np.eye(n, dtype=bool)
    while True:
        new = np.array([lab[nb[i]].min() for i in range(n)], dtype=np.int64) if n else lab
        if np.array_equal(new, lab):
            return lab
        lab = new


def cluster_bruteforce(x, y, toa, tot, W: int, P: int) -> dict:
    """The north_star path on a tiny input by brute force (all pairs, fixed-point closure,
    Python-loop sums). Same output contract as the C++ oracle."""
    x = np.asarray(x, dtype=np.int64)
    y = np.asarray(y, dtype=np.int64)
    tot = np.asarray(tot, dtype=np.int64)
    toa_l = [int(t) for t in np.asarray(toa)]  # python ints: no uint64 overflow games
    n = len(toa_l)
    shot = [t // P if P else 0 for t in toa_l]
    perm = sorted(range(n), key=lambda i: (shot[i], toa_l[i]))  # sorted() is stable
    xs, ys, ts = x[perm], y[perm], tot[perm]
    tl = [toa_l[i] for i in perm]
    sl = [shot[i] for i in perm]
    a = np.zeros((n, n), dtype=np.int64)
    for i in range(n):
        for j in range(n):
            if i != j and sl[i] == sl[j] and abs(int(xs[i]) - int(xs[j])) <= 1 \
                    and abs(int(ys[i]) - int(ys[j])) <= 1 and abs(tl[i] - tl[j]) <= W:
                a[i, j] = 1
    lab = components(a)
    roots = [k for k in range(n) if lab[k] == k]
    out = {
        "perm": np.array(perm, dtype=np.uint32), "label": lab.astype(np.uint32), "n_clusters": len(roots),
        "c_label": [], "c_size": [], "c_shot": [], "c_sum_tot": [], "c_sum_tot_x": [], "c_sum_tot_y": [],
        "c_toa_peak": [], "c_cx": [], "c_cy": [], "c_sum_tot_tof": [], "c_ctof": [],
    }
    for r in roots:
        mem = [k for k in range(n) if lab[k] == r]
        st = sum(int(ts[k]) for k in mem)
        sx = sum(int(ts[k]) * int(xs[k]) for k in mem)
        sy = sum(int(ts[k]) * int(ys[k]) for k in mem)
        peak = max(mem, key=lambda k: (int(ts[k]), k))
        sf = sum(int(ts[k]) * (tl[k] - sl[k] * P) for k in mem)  # ToF = ToA - shot*P
        out["c_label"].append(r)
        out["c_size"].append(len(mem))
        out["c_shot"].append(sl[r])
        out["c_sum_tot"].append(st)
        out["c_sum_tot_x"].append(sx)
        out["c_sum_tot_y"].append(sy)
        out["c_toa_peak"].append(tl[peak])
        out["c_cx"].append(np.float32(sx) / np.float32(st))
        out["c_cy"].append(np.float32(sy) / np.float32(st))
        out["c_sum_tot_tof"].append(sf)
        out["c_ctof"].append(np.float32(sf) / np.float32(st))
    for k in ("c_label", "c_size", "c_shot"):
        out[k] = np.array(out[k], dtype=np.uint32)
    for k in ("c_sum_tot", "c_sum_tot_x", "c_sum_tot_y", "c_sum_tot_tof"):
        out[k] = np.array(out[k], dtype=np.int64)
    out["c_toa_peak"] = np.array(out["c_toa_peak"], dtype=np.uint64)
    out["c_cx"] = np.array(out["c_cx"], dtype=np.float32)
    out["c_cy"] = np.array(out["c_cy"], dtype=np.float32)
    out["c_ctof"] = np.array(out["c_ctof"], dtype=np.float32)
    return out
