"""Pins for the oracle (CPU only). The oracle is checked against things other than itself:
values the paper prints (tests/golden/paper_worked_example.txt), a dense brute-force
restatement of Eq. 3-5 + closure on tiny inputs, closed forms, invariants, library routines
(numpy stable argsort) and generated truth. A plausible mistake (dropped term, wrong sign or
index, strict vs inclusive threshold, transposed operand) fails at least one of these."""
import os

import numpy as np
import pytest

import gen
import oracle
from oracle import bruteforce as bf

W, P = 320, 640000


def load_golden(path):
    vec, rows = {}, {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        head, vals = line.split(":")
        head = head.split()
        vals = [int(v) for v in vals.split()]
        if len(head) == 1:
            vec[head[0]] = vals
        else:
            rows.setdefault(head[0], {})[int(head[1])] = vals
    return vec, rows


# ------------------------------------------------------------------ paper's worked example
def test_paper_worked_example(golden_dir):
    vec, rows = load_golden(os.path.join(golden_dir, "paper_worked_example.txt"))
    X, TOT, w = vec["X"], vec["TOT"], vec["W"][0]
    D = bf.distance_matrix(X)
    for r, vals in rows["DX"].items():  # Eq. 3
        assert D[r - 1].tolist() == vals
    A = bf.adjacency_1d(X, w)
    for r, vals in rows["AX"].items():  # Eq. 4
        assert A[r - 1].tolist() == vals
    M = bf.masked_tot(TOT, A)
    for r, vals in rows["M"].items():  # Eq. 6
        assert M[r - 1].tolist() == vals
    anti = M - M.T
    for r, vals in rows["ANTI"].items():  # Eq. 7
        assert anti[r - 1].tolist() == vals
    for lift in ("paper", "lex", "none"):
        lm = bf.local_maxima(TOT, A, lift=lift)
        assert (lm + 1).tolist() == vec["LOCAL_MAXIMA"]
        assert len(lm) == vec["HIT_COUNT"][0]


def test_worked_example_components_and_centroids():
    # Derived from Eq. 9 on the paper's example (not printed): components at w=5 are {1,2,5},{3,4};
    # here component == box of the local maximum, so both definitions agree.
    X = np.array([20, 21, 90, 92, 18]); TOT = np.array([50, 200, 300, 25, 100])
    z = np.zeros(5, dtype=np.int64)
    A = bf.adjacency(X, z, z, 5, 0, 0)
    assert bf.components(A).tolist() == [0, 0, 2, 2, 0]
    cent = bf.box_centroid(X, TOT, A)
    lm = bf.local_maxima(TOT, A)
    assert cent[lm[0]] == 7000 / 350 == 20.0
    assert cent[lm[1]] == pytest.approx(29300 / 325)
    # At the north_star's w = 1 the same data gives {1,2},{3},{4},{5}; run the C++ oracle.
    o = oracle.run(X, z, z, TOT, W, 0)
    assert o["perm"].tolist() == [0, 1, 2, 3, 4]  # all ToA equal: stable order = input order
    assert o["label"].tolist() == [0, 0, 2, 3, 4]
    assert o["n_clusters"] == 4
    assert o["c_sum_tot"].tolist() == [250, 300, 25, 100]
    assert o["c_sum_tot_x"].tolist() == [50 * 20 + 200 * 21, 300 * 90, 25 * 92, 100 * 18]
    assert o["c_cx"][0] == np.float32(5200) / np.float32(250)
    assert o["c_cx"][1:].tolist() == [90.0, 92.0, 18.0]


def test_tie_break_later_pixel_wins():
    # equal ToT -> the pixel later in the stream wins.
    x = np.array([10, 11, 12]); y = np.array([5, 5, 5]); toa = np.array([100, 100, 100]); tot = np.array([7, 9, 9])
    A = bf.adjacency(x, y, toa, 1, 1, W)
    assert bf.local_maxima(tot, A, "paper").tolist() == [2]
    assert bf.local_maxima(tot, A, "lex").tolist() == [2]
    assert sorted(bf.local_maxima(tot, A, "none").tolist()) == [1, 2]  # over-counting without the lift
    toa2 = np.array([100, 105, 103])  # sorted order: idx 0 (100), idx 2 (103), idx 1 (105)
    o = oracle.run(x, y, toa2, tot, W, P)
    assert o["perm"].tolist() == [0, 2, 1]
    assert o["n_clusters"] == 1 and o["c_toa_peak"].tolist() == [105]  # tot 9 at sorted pos 1 and 2 -> pos 2


# ------------------------------------------------------------------ brute force on tiny inputs
def assert_same(o, b):
    assert o["n_clusters"] == b["n_clusters"]
    for k in ("perm", "label", "c_label", "c_size", "c_shot", "c_sum_tot", "c_sum_tot_x", "c_sum_tot_y", "c_toa_peak",
              "c_sum_tot_tof"):
        assert np.array_equal(o[k], b[k]), k
    assert np.array_equal(o["c_cx"].view(np.uint32), b["c_cx"].view(np.uint32))
    assert np.array_equal(o["c_cy"].view(np.uint32), b["c_cy"].view(np.uint32))
    assert np.array_equal(o["c_ctof"].view(np.uint32), b["c_ctof"].view(np.uint32))


def tiny_random(rng, n, span_xy=6, span_t=900, shots=2):
    x = rng.integers(0, span_xy, n) + rng.integers(0, 2) * (256 - span_xy)
    y = rng.integers(0, span_xy, n) + rng.integers(0, 2) * (256 - span_xy)
    toa = rng.integers(0, shots, n) * P + rng.integers(0, span_t, n)
    tot = rng.integers(1, 6, n)
    return x, y, toa.astype(np.uint64), tot


@pytest.mark.parametrize("seed", range(40))
def test_bruteforce_random(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(2, 65))
    x, y, toa, tot = tiny_random(rng, n, span_xy=int(rng.integers(2, 9)), span_t=int(rng.integers(1, 1500)),
                                 shots=int(rng.integers(1, 4)))
    assert_same(oracle.run(x, y, toa, tot, W, P), bf.cluster_bruteforce(x, y, toa, tot, W, P))


def test_bruteforce_adversarial():
    cases = []
    # chain A-B-C with |tA - tC| > W: still one component (transitive closure)
    cases.append(([10, 11, 12], [10, 10, 10], [1000, 1000 + W, 1000 + 2 * W], [5, 6, 7]))
    # dt == W links, dt == W + 1 does not (inclusive threshold)
    cases.append(([10, 11, 20, 21], [10, 10, 10, 10], [0, W, 0, W + 1], [5, 6, 7, 8]))
    # repeated address inside the window is adjacent (dx = dy = 0 satisfies Eq. 5), outside is not
    cases.append(([7, 7, 7], [9, 9, 9], [0, 100, 100 + W + 1], [3, 3, 3]))
    # sensor corners, no wrap-around
    cases.append(([0, 255, 0, 255, 1, 254], [0, 255, 255, 0, 1, 254], [5, 5, 5, 5, 5, 5], [1, 2, 3, 4, 5, 6]))
    # hits straddling a shot boundary: tick sP-1 and sP are different shots (never linked)
    cases.append(([50, 50, 51], [60, 60, 60], [P - 1, P, P + 1], [9, 9, 9]))
    # all hits identical
    cases.append(([3] * 8, [4] * 8, [777] * 8, [2] * 8))
    # dx = 2 is not adjacent; diagonal is
    cases.append(([10, 12, 13, 14], [10, 10, 11, 12], [0, 0, 0, 0], [1, 1, 1, 1]))
    # unsorted input with equal ToA in different input order (stable sort)
    cases.append(([1, 2, 3, 4, 5], [1, 1, 1, 1, 1], [50, 40, 50, 40, 45], [1, 2, 3, 4, 5]))
    for x, y, toa, tot in cases:
        x, y, tot = np.array(x), np.array(y), np.array(tot)
        toa = np.array(toa, dtype=np.uint64)
        o = oracle.run(x, y, toa, tot, W, P)
        assert_same(o, bf.cluster_bruteforce(x, y, toa, tot, W, P))
    o = oracle.run(*[np.array(c) for c in cases[0][:2]], np.array(cases[0][2], dtype=np.uint64), np.array(cases[0][3]), W, P)
    assert o["n_clusters"] == 1
    o = oracle.run(np.array(cases[1][0]), np.array(cases[1][1]), np.array(cases[1][2], dtype=np.uint64), np.array(cases[1][3]), W, P)
    assert o["n_clusters"] == 3
    o = oracle.run(np.array(cases[4][0]), np.array(cases[4][1]), np.array(cases[4][2], dtype=np.uint64), np.array(cases[4][3]), W, P)
    assert o["label"].tolist() == [0, 1, 1] and o["c_shot"].tolist() == [0, 1]


def test_empty_and_single():
    e16, e64 = np.zeros(0, np.uint16), np.zeros(0, np.uint64)
    o = oracle.run(e16, e16, e64, e16, W, P)
    assert o["n_clusters"] == 0 and o["perm"].shape == (0,) and o["c_cx"].shape == (0,)
    o = oracle.run([17], [200], [3 * P + 12345], [321], W, P)
    assert o["n_clusters"] == 1 and o["label"].tolist() == [0]
    assert o["c_size"].tolist() == [1] and o["c_cx"].tolist() == [17.0] and o["c_cy"].tolist() == [200.0]
    assert o["c_toa_peak"].tolist() == [3 * P + 12345] and o["c_shot"].tolist() == [3]


def test_shot_period_zero_is_one_shot():
    x = np.array([5, 6]); y = np.array([5, 5]); toa = np.array([P - 1, P], dtype=np.uint64); tot = np.array([1, 1])
    assert oracle.run(x, y, toa, tot, W, P)["n_clusters"] == 2
    assert oracle.run(x, y, toa, tot, W, 0)["n_clusters"] == 1
    assert_same(oracle.run(x, y, toa, tot, W, 0), bf.cluster_bruteforce(x, y, toa, tot, W, 0))


# ------------------------------------------------------------------ closed forms
def test_two_pixel_closed_form():
    for (x1, y1, t1), (x2, y2, t2) in [((100, 50, 3), (101, 51, 9)), ((255, 0, 1023), (254, 0, 1)), ((0, 7, 13), (0, 8, 29))]:
        o = oracle.run([x1, x2], [y1, y2], [10, 20], [t1, t2], W, P)
        assert o["n_clusters"] == 1 and o["c_size"].tolist() == [2]
        assert o["c_sum_tot"].tolist() == [t1 + t2]
        assert o["c_cx"][0] == np.float32(t1 * x1 + t2 * x2) / np.float32(t1 + t2)
        assert o["c_cy"][0] == np.float32(t1 * y1 + t2 * y2) / np.float32(t1 + t2)
        assert abs(float(o["c_cx"][0]) - (t1 * x1 + t2 * x2) / (t1 + t2)) < 2e-5  # exact value within fp32 rounding
        assert o["c_toa_peak"].tolist() == [10 if t1 > t2 else 20]


def test_tof_centroid_closed_forms():
    """ToT-weighted time-of-flight centroid: "identical for X, Y and ToF", ToF = ToA - trigger
     = ToA - shot*P (R6)."""
    # Eq. 9 on a hand-computed example: one hit of three pixels in shot 7, ToF 100, 104, 110, ToT 10, 30, 20
    toa = 7 * P + np.array([100, 104, 110]); tot = np.array([10, 30, 20])
    o = oracle.run([50, 51, 50], [60, 60, 61], toa, tot, W, P)
    assert o["n_clusters"] == 1 and o["c_shot"].tolist() == [7]
    assert o["c_sum_tot_tof"].tolist() == [10 * 100 + 30 * 104 + 20 * 110] == [6320]
    assert o["c_ctof"][0] == np.float32(6320) / np.float32(60)
    assert abs(float(o["c_ctof"][0]) - 6320 / 60) < 1e-5
    # the same through the paper-literal row reduction (Eq. 9 with the ToF vector in place of X)
    A = bf.adjacency(np.array([50, 51, 50]), np.array([60, 60, 61]), toa, 1, 1, W) | np.eye(3, dtype=np.int64)
    assert bf.box_centroid(toa - 7 * P, tot, A)[1] == pytest.approx(6320 / 60)
    # single pixel: the centroid is the pixel's own ToF
    o = oracle.run([9], [9], [3 * P + 4321], [77], W, P)
    assert o["c_sum_tot_tof"].tolist() == [77 * 4321] and o["c_ctof"].tolist() == [4321.0]
    # two pixels: (t1 f1 + t2 f2) / (t1 + t2)
    o = oracle.run([9, 10], [9, 9], [P + 10, P + 30], [3, 1], W, P)
    assert o["c_ctof"].tolist() == [15.0]
    # P = 0: one shot, the trigger is tick 0, ToF = ToA
    o = oracle.run([9, 10], [9, 9], [P + 10, P + 30], [3, 1], W, 0)
    assert o["c_sum_tot_tof"].tolist() == [3 * (P + 10) + (P + 30)]


def test_tof_centroid_transforms():
    w = gen.generate(2, shots=60)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    # whole shots later: only shot and toa_peak change
    o2 = oracle.run(w.x, w.y, w.toa + np.uint64(5 * P), w.tot, W, P)
    assert np.array_equal(o["c_sum_tot_tof"], o2["c_sum_tot_tof"]) and np.array_equal(o["c_ctof"], o2["c_ctof"])
    # every event d ticks later inside its shot: sum_tot_tof grows by d * sum_tot, nothing else moves
    d = 1000
    o3 = oracle.run(w.x, w.y, w.toa + np.uint64(d), w.tot, W, P)
    assert np.array_equal(o3["label"], o["label"])
    assert np.array_equal(o3["c_sum_tot_tof"], o["c_sum_tot_tof"] + d * o["c_sum_tot"])
    # the centroid lies between the earliest and the latest member ToF of the hit; conservation
    tof = (w.toa[o["perm"]] % np.uint64(P)).astype(np.int64)
    lo = np.full(o["n_clusters"], 1 << 62); hi = np.zeros(o["n_clusters"], dtype=np.int64)
    slot = np.searchsorted(o["c_label"], o["label"])
    np.minimum.at(lo, slot, tof); np.maximum.at(hi, slot, tof)
    assert np.all(o["c_ctof"] >= lo.astype(np.float32)) and np.all(o["c_ctof"] <= hi.astype(np.float32))
    assert int(o["c_sum_tot_tof"].sum()) == int((w.tot[o["perm"]].astype(np.int64) * tof).sum())


# ------------------------------------------------------------------ invariants on the configs
WORKLOADS = [(0, 1000), (1, 300), (2, 150), (3, 40), (4, 150)]


@pytest.fixture(scope="module", params=WORKLOADS, ids=lambda p: "cfg%d" % p[0])
def wl(request):
    cfg, shots = request.param
    w = gen.generate(cfg, shots=shots)
    return w, oracle.run(w.x, w.y, w.toa, w.tot, W, P)


def test_invariants(wl):
    w, o = wl
    n = w.n
    perm, label = o["perm"].astype(np.int64), o["label"].astype(np.int64)
    k = np.arange(n)
    # perm: the unique stable sort (library pin: numpy's stable argsort; (shot, toa) order == toa order)
    assert np.array_equal(perm, np.argsort(w.toa, kind="stable"))
    assert np.all(label <= k)
    assert np.array_equal(label[label], label)
    assert o["n_clusters"] == int(np.sum(label == k))
    assert np.array_equal(o["c_label"], k[label == k])
    assert int(o["c_size"].sum()) == n
    assert int(o["c_sum_tot"].sum()) == int(w.tot.astype(np.int64).sum())
    assert int(o["c_sum_tot_x"].sum()) == int((w.tot.astype(np.int64) * w.x).sum())
    assert int(o["c_sum_tot_y"].sum()) == int((w.tot.astype(np.int64) * w.y).sum())
    # independent numpy recomputation of the per-cluster sums from the labels
    xs, ys, ts, toas = w.x[perm].astype(np.int64), w.y[perm].astype(np.int64), w.tot[perm].astype(np.int64), w.toa[perm]
    slot = np.cumsum(label == k) - 1
    c = slot[label]
    nc = o["n_clusters"]
    assert np.array_equal(np.bincount(c, minlength=nc), o["c_size"])
    assert np.array_equal(np.bincount(c, weights=ts, minlength=nc).astype(np.int64), o["c_sum_tot"])
    assert np.array_equal(np.bincount(c, weights=ts * xs, minlength=nc).astype(np.int64), o["c_sum_tot_x"])
    assert np.array_equal(np.bincount(c, weights=ts * ys, minlength=nc).astype(np.int64), o["c_sum_tot_y"])
    # centroid inside the bounding box of the members; all members in the root's shot
    xmin = np.full(nc, 1 << 30); xmax = np.full(nc, -1)
    np.minimum.at(xmin, c, xs); np.maximum.at(xmax, c, xs)
    assert np.all(o["c_cx"] >= xmin) and np.all(o["c_cx"] <= xmax)
    shot = (toas // np.uint64(P)).astype(np.int64)
    assert np.array_equal(shot[label], shot)
    assert np.array_equal(o["c_shot"], shot[label == k])
    # peak: member with max (tot, k)
    key = ts * (n + 1) + k
    best = np.zeros(nc, dtype=np.int64)
    np.maximum.at(best, c, key)
    assert np.array_equal(o["c_toa_peak"], toas[best % (n + 1)])
    # singles: centroid is the pixel itself
    single = o["c_size"] == 1
    roots = k[label == k]
    assert np.array_equal(o["c_cx"][single], xs[roots[single]].astype(np.float32))
    assert np.array_equal(o["c_toa_peak"][single], toas[roots[single]])


def test_every_link_is_valid_and_closed(wl):
    """Labels are a valid closure: every adjacent pair (brute force inside each shot) has equal
    labels, and every non-root hit has an adjacent hit with the same label (so no component is
    the union of two unrelated pieces, checked per component by BFS-free counting)."""
    w, o = wl
    perm, label = o["perm"].astype(np.int64), o["label"].astype(np.int64)
    xs, ys, toas = w.x[perm].astype(np.int64), w.y[perm].astype(np.int64), w.toa[perm].astype(np.int64)
    shot = toas // P
    bounds = np.flatnonzero(np.diff(shot)) + 1
    starts = np.concatenate([[0], bounds]); ends = np.concatenate([bounds, [len(shot)]])
    checked = 0
    for a, b in list(zip(starts, ends))[:25]:
        X, Y, T, L = xs[a:b], ys[a:b], toas[a:b], label[a:b]
        A = (np.abs(X[:, None] - X[None, :]) <= 1) & (np.abs(Y[:, None] - Y[None, :]) <= 1) & (np.abs(T[:, None] - T[None, :]) <= W)
        np.fill_diagonal(A, False)
        i, j = np.nonzero(A)
        assert np.array_equal(L[i], L[j])
        assert np.array_equal(bf.components(A.astype(np.int64)) + a, L)
        checked += 1
    assert checked > 0


def test_transform_invariants():
    w = gen.generate(2, shots=60)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    # translation in x by a adds a * sum_tot to sum_tot_x
    a = 3
    o2 = oracle.run(w.x + a, w.y, w.toa, w.tot, W, P)
    assert np.array_equal(o2["label"], o["label"])
    assert np.array_equal(o2["c_sum_tot_x"], o["c_sum_tot_x"] + a * o["c_sum_tot"])
    # adding m*P to every ToA changes only shot and toa_peak
    m = 7
    o3 = oracle.run(w.x, w.y, w.toa + np.uint64(m * P), w.tot, W, P)
    for k in ("perm", "label", "c_size", "c_sum_tot", "c_sum_tot_x", "c_sum_tot_y", "c_cx", "c_cy"):
        assert np.array_equal(o3[k], o[k]), k
    assert np.array_equal(o3["c_shot"], o["c_shot"] + m)
    assert np.array_equal(o3["c_toa_peak"], o["c_toa_peak"] + np.uint64(m * P))
    # swapping x and y swaps the sums (catches a transposed operand)
    o4 = oracle.run(w.y, w.x, w.toa, w.tot, W, P)
    assert np.array_equal(o4["c_sum_tot_x"], o["c_sum_tot_y"]) and np.array_equal(o4["c_cy"], o["c_cx"])
    # growing W never increases the cluster count; W = 0 still links equal-ToA neighbours
    counts = [oracle.run(w.x, w.y, w.toa, w.tot, ww, P)["n_clusters"] for ww in (0, 5, 30, 320, 5000)]
    assert all(c1 >= c2 for c1, c2 in zip(counts, counts[1:]))
    assert counts[0] > counts[3]


def test_permutation_invariance_distinct_toa():
    # With distinct ToA the cluster SET does not depend on the input order.
    rng = np.random.default_rng(5)
    w = gen.generate(0, shots=30)
    toa = w.toa * np.uint64(4000) + np.arange(w.n, dtype=np.uint64) % np.uint64(4000)  # make ToA distinct, keep order
    Pd, Wd = P * 4000, W * 4000
    assert len(np.unique(toa)) == w.n
    o = oracle.run(w.x, w.y, toa, w.tot, Wd, Pd)
    p = rng.permutation(w.n)
    o2 = oracle.run(w.x[p], w.y[p], toa[p], w.tot[p], Wd, Pd)
    assert np.array_equal(p[o2["perm"]], o["perm"])
    for k in ("label", "c_size", "c_sum_tot", "c_sum_tot_x", "c_sum_tot_y", "c_toa_peak", "c_cx", "c_cy"):
        assert np.array_equal(o2[k], o[k]), k


def test_local_maxima_vs_components():
    # #local maxima at w = 1 >= n_clusters with at least one per component (links the paper's
    # definition of a hit, Eq. 6-7, with the north_star's connected component).
    w = gen.generate(2, shots=3)
    for s in range(3):
        ws = w.slice_shots(s, s + 1)
        o = oracle.run(ws.x, ws.y, ws.toa, ws.tot, W, P)
        perm = o["perm"].astype(np.int64)
        A = bf.adjacency(ws.x[perm], ws.y[perm], ws.toa[perm].astype(np.int64), 1, 1, W)
        lm = bf.local_maxima(ws.tot[perm], A, "lex")
        assert len(lm) >= o["n_clusters"]
        assert set(o["label"][lm].tolist()) == set(o["c_label"].tolist())


# ------------------------------------------------------------------ generated truth
def test_well_separated_truth():
    w = gen.generate(5, shots=400, truth=True)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    assert o["n_clusters"] == len(w.truth["cx"]) == 4000  # exact particle count
    assert np.array_equal(np.sort(o["c_size"]), np.sort(w.truth["k"]))
    # match clusters to particles per shot by nearest centre
    err = []
    cs = o["c_shot"].astype(np.int64)
    for s in range(0, 400, 7):
        m = cs == s
        t = w.truth["shot"] == s
        cx, cy = o["c_cx"][m].astype(np.float64), o["c_cy"][m].astype(np.float64)
        d = np.hypot(cx[:, None] - w.truth["cx"][t][None, :], cy[:, None] - w.truth["cy"][t][None, :])
        assert sorted(d.argmin(axis=1).tolist()) == list(range(10))  # one-to-one
        err.extend(d.min(axis=1).tolist())
    err = np.array(err)
    assert err.mean() < 0.3 and err.max() < 1.0  # truncated, noisy footprint: tolerance, not equality


# ------------------------------------------------------------------ paper-literal mode (NEXT #2)
LM_KEYS = ("c_label", "c_size", "c_shot", "c_sum_tot", "c_sum_tot_x", "c_sum_tot_y", "c_toa_peak", "c_sum_tot_tof")


def test_localmax_paper_worked_example(golden_dir):
    """X, ToT of Eq. 2 / :134 at |D| <= 5 -> "local maxima are pixel 2 and pixel 3"."""
    g = {}
    for line in open(os.path.join(golden_dir, "paper_worked_example.txt")):
        if line.startswith("#") or ":" not in line:
            continue
        k, v = line.split(":")
        g[k.strip()] = [int(t) for t in v.split()]
    X, TOT, w = np.array(g["X"]), np.array(g["TOT"]), g["W"][0]
    z = np.zeros(len(X), dtype=np.int64)
    o = oracle.run_localmax(X, z, z, TOT, w, 0, 0, 0)
    assert (o["c_label"] + 1).tolist() == [2, 3] and o["n_clusters"] == 2        # the paper's answer (:148)
    assert o["lmax"].tolist() == [0xFFFFFFFF, 1, 2, 0xFFFFFFFF, 0xFFFFFFFF]
    # Eq. 9 on rows 2 and 3 of the printed A^X (Eq. 4): boxes {1,2,5} and {3,4}
    assert o["c_size"].tolist() == [3, 2]
    assert o["c_sum_tot"].tolist() == [350, 325] and o["c_sum_tot_x"].tolist() == [7000, 29300]
    assert o["c_cx"][0] == 20.0 and o["c_cx"][1] == np.float32(29300) / np.float32(325)


def _dense_localmax(x, y, toa, tot, wx, wy, wt, Pp):
    """The same from the paper's array formulation (oracle/bruteforce.py: Eq. 3-9 written out)."""
    toa_l = [int(t) for t in toa]
    shot = [t // Pp if Pp else 0 for t in toa_l]
    perm = sorted(range(len(toa_l)), key=lambda i: (shot[i], toa_l[i]))
    xs, ys, ts = np.asarray(x)[perm], np.asarray(y)[perm], np.asarray(tot)[perm]
    tl = np.array([toa_l[i] for i in perm], dtype=np.int64)
    sl = np.array([shot[i] for i in perm], dtype=np.int64)
    A = bf.adjacency(xs, ys, tl, wx, wy, wt, shot=sl)
    lm = bf.local_maxima(ts, A, "lex")
    tof = tl - sl * Pp
    return perm, lm, A, bf.box_centroid(xs, ts, A), bf.box_centroid(ys, ts, A), bf.box_centroid(tof, ts, A), ts


@pytest.mark.parametrize("seed", range(25))
def test_localmax_vs_dense_array_formulation(seed):
    rng = np.random.default_rng(1000 + seed)
    n = int(rng.integers(1, 60))
    x, y, toa, tot = tiny_random(rng, n, span_xy=9, span_t=1200, shots=2)
    tot = rng.integers(1, 4, n)  # many ties: the tie rule decides
    wx, wy, wt = int(rng.integers(0, 4)), int(rng.integers(0, 4)), int(rng.integers(0, 700))
    o = oracle.run_localmax(x, y, toa, tot, wx, wy, wt, P)
    perm, lm, A, cx, cy, ct, ts = _dense_localmax(x, y, toa, tot, wx, wy, wt, P)
    assert o["perm"].tolist() == perm
    assert o["c_label"].tolist() == sorted(lm.tolist())
    for c, i in enumerate(o["c_label"]):
        assert o["c_size"][c] == A[i].sum() and o["c_sum_tot"][c] == (A[i] * ts).sum()
        assert float(o["c_cx"][c]) == pytest.approx(cx[i], rel=1e-6)
        assert float(o["c_cy"][c]) == pytest.approx(cy[i], rel=1e-6)
        assert float(o["c_ctof"][c]) == pytest.approx(ct[i], rel=1e-6, abs=1e-6)


def test_localmax_tie_and_window_edges():
    # equal ToT: the later pixel of the sorted stream wins. Sorted positions: x = 10, 12, 11;
    # x=11 (pos 2) is adjacent to both others and is the latest -> the only hit; its box holds all three.
    o = oracle.run_localmax([10, 11, 12], [5, 5, 5], [100, 105, 103], [9, 9, 9], 1, 1, W, P)
    assert o["perm"].tolist() == [0, 2, 1]
    assert o["c_label"].tolist() == [2] and o["c_size"].tolist() == [3] and o["c_cx"].tolist() == [11.0]
    assert o["c_toa_peak"].tolist() == [105] and o["c_ctof"].tolist() == [np.float32(9 * 308) / np.float32(27)]
    # inclusive thresholds in all three coordinates, and no neighbourhood across a shot
    for dx, dy, dt, linked in [(2, 0, 0, True), (3, 0, 0, False), (0, 2, 0, True), (0, 3, 0, False),
                               (0, 0, 50, True), (0, 0, 51, False)]:
        o = oracle.run_localmax([100, 100 + dx], [100, 100 + dy], [1000, 1000 + dt], [5, 7], 2, 2, 50, P)
        assert o["n_clusters"] == (1 if linked else 2), (dx, dy, dt)
    o = oracle.run_localmax([100, 100], [100, 100], [P - 1, P], [5, 7], 2, 2, 50, P)
    assert o["n_clusters"] == 2 and o["c_shot"].tolist() == [0, 1]
    o = oracle.run_localmax([100, 100], [100, 100], [P - 1, P], [5, 7], 2, 2, 50, 0)
    assert o["n_clusters"] == 1
    # empty input
    z = np.zeros(0, dtype=np.uint16)
    assert oracle.run_localmax(z, z, np.zeros(0, dtype=np.uint64), z, 1, 1, W, P)["n_clusters"] == 0


def test_localmax_equals_components_when_boxes_cover_blobs():
    """Well-separated particles (centres >= 12 px apart, footprints within 2 px of the centre): a box of
    half-width 4 about ANY pixel of a blob holds the whole blob and nothing else, so the paper's hit
    (local maximum + box, Eq. 6-9) and the north_star's hit (connected component) are the same sets and
    every sum, peak and centroid must agree — the two oracles pin each other, and the generated truth
    pins the count."""
    w = gen.generate(5, shots=300, truth=True)
    a = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    b = oracle.run_localmax(w.x, w.y, w.toa, w.tot, 4, 4, W, P)
    assert b["n_clusters"] == a["n_clusters"] == len(w.truth["cx"])
    assert np.array_equal(a["perm"], b["perm"])
    # a component is listed at its first pixel, a paper hit at its brightest pixel: match through the label array
    comp_of_hit = a["label"][b["c_label"]]
    order = np.argsort(comp_of_hit, kind="stable")
    assert np.array_equal(comp_of_hit[order], a["c_label"])
    for k in ("c_size", "c_shot", "c_sum_tot", "c_sum_tot_x", "c_sum_tot_y", "c_sum_tot_tof", "c_toa_peak", "c_cx",
              "c_cy", "c_ctof"):
        assert np.array_equal(b[k][order], a[k]), k


def test_localmax_invariants():
    w = gen.generate(2, shots=40)
    o = oracle.run_localmax(w.x, w.y, w.toa, w.tot, 1, 1, W, P)
    a = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    n = w.n
    k = np.arange(n, dtype=np.uint32)
    assert np.all((o["lmax"] == k) | (o["lmax"] == 0xFFFFFFFF))
    assert np.array_equal(np.flatnonzero(o["lmax"] == k), o["c_label"])
    # at least one local maximum per connected component, all maxima inside components (links R2's two definitions)
    assert o["n_clusters"] >= a["n_clusters"]
    assert set(a["label"][o["c_label"]].tolist()) == set(a["c_label"].tolist())
    # a box at w = 1 is a subset of the pixel's component
    slot = np.searchsorted(a["c_label"], a["label"][o["c_label"]])
    assert np.all(o["c_size"] <= a["c_size"][slot]) and np.all(o["c_sum_tot"] <= a["c_sum_tot"][slot])
    assert np.all(o["c_size"] >= 1)
    # growing the box never adds hits
    assert oracle.run_localmax(w.x, w.y, w.toa, w.tot, 2, 2, W, P)["n_clusters"] <= o["n_clusters"]


# ------------------------------------------------------------------ ToA unwrapping (NEXT #4)
from oracle import preprocess as pp  # noqa: E402

TICK_NS = 1.5625
PIX_MOD = (1 << 42) // 256            # 2^42 units of 25/4096 ns in ticks of 256 units
JUMP_20S = int(20e9 / TICK_NS)        # "more than 20 seconds"


def test_unwrap_constants_match_the_paper():
    # 25/4096 ns x 2^42 = about 26.8 s for pixels, x 2^44 = about 107.4 s for the TDCs
    assert abs(PIX_MOD * TICK_NS * 1e-9 - 26.8) < 0.05
    assert abs(((1 << 44) // 256) * TICK_NS * 1e-9 - 107.4) < 0.05


def test_unwrap_hand_example_out_of_order_across_the_wrap():
    # a dim pixel with a LATER ToA (after the wrap) reports before a bright one whose ToA is
    # just before the wrap. Counter period 1024, threshold 600; true times 1000 1019 1027 1022 1031 1044.
    raw = [1000, 1019, 3, 1022, 7, 20]
    out, wraps = pp.unwrap_toa(raw, 1024, 600)
    assert out.tolist() == [1000, 1019, 1027, 1022, 1031, 1044] and wraps == 1
    # without the edge case: each large negative shift adds one period to everything after it
    out, wraps = pp.unwrap_toa([10, 500, 1000, 5, 400, 900, 2], 1024, 600)
    assert out.tolist() == [10, 500, 1000, 1029, 1424, 1924, 2050] and wraps == 2
    # strict threshold: a shift of exactly `jump` is not a wrap, jump + 1 is
    assert pp.unwrap_toa([700, 100], 1024, 600)[1] == 0 and pp.unwrap_toa([701, 100], 1024, 600)[1] == 1
    assert pp.unwrap_toa([100, 700], 1024, 600)[1] == 0 and pp.unwrap_toa([100, 701], 1024, 600)[1] == -1
    assert pp.unwrap_toa([], 1024, 600, wraps_in=3) [1] == 3


@pytest.mark.parametrize("seed", range(6))
def test_unwrap_recovers_true_times(seed):
    """Generated truth: true arrival times over several counter periods, delivered with local disorder
    (dim pixels report first), wrapped to 42 bits; unwrapping must give the true times back."""
    rng = np.random.default_rng(seed)
    n = 20000
    span = 3 * PIX_MOD + PIX_MOD // 3                     # about 3.3 wraps
    t = np.sort(rng.integers(0, span, n).astype(np.int64))
    t = t + rng.integers(0, 2000, n)                      # report order != ToA order (disorder up to 3 us)
    start = PIX_MOD - 5000                                # the first wrap comes early
    t = t + start
    raw = (t % PIX_MOD).astype(np.uint64)
    w0 = int(t[0] // PIX_MOD)                             # wraps before the first event: the caller's state
    out, wraps = pp.unwrap_toa(raw, PIX_MOD, JUMP_20S, wraps_in=w0)
    assert np.array_equal(out.astype(np.int64), t) and wraps == int(t[-1] // PIX_MOD) and wraps - w0 >= 3
    # chunked with carried state == whole
    cuts = [0, 1, 777, 778, 9000, n]
    w, prev, parts = w0, None, []
    for a, b in zip(cuts[:-1], cuts[1:]):
        o, w = pp.unwrap_toa(raw[a:b], PIX_MOD, JUMP_20S, wraps_in=w, prev_raw=prev)
        parts.append(o)
        prev = raw[b - 1]
    assert np.array_equal(np.concatenate(parts), out) and w == wraps


# ------------------------------------------------------------------ preprocessing (NEXT #3)
def test_timewalk_table_closed_forms():
    # Eq. 1 at d = 1 ("typically very close to 1", :76): a / (ToT + b) + c, by hand
    t = pp.timewalk_table(a=1000.0, b=10.0, c=-2.0, d=1.0, length=6)
    assert t.tolist() == [98, 89, 81, 75, 69, 65]      # 100-2, 90.909-2, 83.33-2, 76.92-2, 71.43-2, 66.67-2
    # monotone decreasing in ToT for a > 0 (dim pixels walk later), tends to c
    t = pp.timewalk_table(500.0, 3.0, 1.0, 1.2, 1024)
    assert np.all(np.diff(t) <= 0) and t[-1] == 1 and t[0] == int(np.floor(500.0 / 3.0 ** 1.2 + 1.0 + 0.5))
    # a = 0: the constant c, rounded half away from zero
    assert pp.timewalk_table(0.0, 1.0, 2.5, 1.0, 3).tolist() == [3, 3, 3]
    assert pp.timewalk_table(0.0, 1.0, -2.5, 1.0, 3).tolist() == [-3, -3, -3]


def test_preprocess_hand_example():
    # triggers at 1000, 2000, 3000 (ticks); cut 300; table: ToT 0..3 -> 9, 5, 2, 0; P_out = 640000
    trig = [1000, 2000, 3000]
    toa = [900, 1000, 1300, 1301, 2004, 2999, 3100, 2150, 3003]
    tot = [1, 1, 2, 2, 0, 3, 9, 1, 1]
    x = list(range(9)); y = [2 * v for v in x]
    xs, ys, ts, os_, idx = pp.preprocess(x, y, toa, tot, trig, 300, [9, 5, 2, 0], P)
    # 900: before the first trigger -> dropped; 1301: ToF 301 > cut -> dropped; 2999: ToF 999 -> dropped
    assert idx.tolist() == [1, 2, 4, 6, 7, 8]
    # 1000: ToF 0 - 5 -> clamped to 0; 1300: 300 - 2 = 298 (ToF == cut is kept, "does not exceed");
    # 2004: 4 - 9 -> 0; 3100: ToT 9 beyond the table -> last entry 0 -> 100; 2150 (out of order in the stream):
    # trigger 1, 150 - 5; 3003: 3 - 5 -> 0
    assert ts.tolist() == [0 * P + 0, 0 * P + 298, 1 * P + 0, 2 * P + 100, 1 * P + 145, 2 * P + 0]
    assert xs.tolist() == [1, 2, 4, 6, 7, 8] and ys.tolist() == [2, 4, 8, 12, 14, 16] and os_.tolist() == [1, 2, 0, 9, 1, 1]
    # shot_base shifts every shot number
    assert pp.preprocess(x, y, toa, tot, trig, 300, [9, 5, 2, 0], P, shot_base=7)[2].tolist() == [
        t + 7 * P for t in ts.tolist()]


def test_preprocess_recovers_the_generated_stream():
    """Generated truth: take a config-2 stream (shot s starts at s*P), move its shots onto irregular trigger
    times, add timewalk dToF(ToT) to every pixel and sprinkle dark counts later than the cut: preprocessing
    with the same table must give the original stream back, event for event."""
    w = gen.generate(2, shots=30)
    rng = np.random.default_rng(9)
    trig = np.cumsum(rng.integers(P - 2000, P + 2000, 30)).astype(np.int64) + 12345
    table = pp.timewalk_table(800.0, 4.0, 0.0, 1.0, 1024)
    shot = (w.toa // np.uint64(P)).astype(np.int64)
    tof = (w.toa % np.uint64(P)).astype(np.int64)
    raw = trig[shot] + tof + table[np.minimum(w.tot, 1023)]
    keep_cut = int(tof.max() + table.max())
    # dark counts: ToF beyond the cut, random pixels; merged into the stream by raw time
    nd = 5000
    dshot = rng.integers(0, 30, nd)
    draw = trig[dshot] + rng.integers(keep_cut + 1, P - 3000, nd)
    allx = np.concatenate([w.x, rng.integers(0, 256, nd).astype(np.uint16)])
    ally = np.concatenate([w.y, rng.integers(0, 256, nd).astype(np.uint16)])
    alltot = np.concatenate([w.tot, rng.integers(1, 30, nd).astype(np.uint16)])
    allraw = np.concatenate([raw, draw]).astype(np.uint64)
    is_dark = np.concatenate([np.zeros(w.n, bool), np.ones(nd, bool)])
    order = np.argsort(allraw, kind="stable")
    xs, ys, ts, os_, idx = pp.preprocess(allx[order], ally[order], allraw[order], alltot[order], trig, keep_cut,
                                         table, P)
    assert not np.any(is_dark[order][idx]) and len(idx) == w.n          # exactly the dark counts are cut
    back = np.argsort(order[idx], kind="stable")                        # original event order
    assert np.array_equal(ts[back], w.toa) and np.array_equal(xs[back], w.x) and np.array_equal(os_[back], w.tot)


# ------------------------------------------------------------------ chunked stream, unaligned cuts (NEXT #3)
def _stream_rows(model, chunks, W, P):
    """Push the chunks (the last one with final=True); cluster every emitted set with the batch oracle and
    concatenate the hit rows, labels made global with label_base."""
    cols = {k: [] for k in ("c_label", "c_size", "c_shot", "c_sum_tot", "c_sum_tot_x", "c_sum_tot_y",
                            "c_sum_tot_tof", "c_toa_peak", "c_cx", "c_cy", "c_ctof")}
    stats = []
    for i, (x, y, toa, tot) in enumerate(chunks):
        e = model.push(x, y, toa, tot, final=(i == len(chunks) - 1))
        stats.append((len(e["x"]), e["n_carry"], e["n_late"]))
        r = oracle.run(e["x"], e["y"], e["toa"], e["tot"], W, P)
        for k in cols:
            v = r[k]
            cols[k].append(v + np.uint32(e["label_base"]) if k == "c_label" else v)
    return {k: np.concatenate(v) for k, v in cols.items()}, stats


def _cut(w, sizes):
    out, i = [], 0
    for s in sizes:
        out.append((w.x[i:i + s], w.y[i:i + s], w.toa[i:i + s], w.tot[i:i + s]))
        i += s
    assert i == w.n
    return out


def _disorder(toa):
    t = toa.astype(np.int64)
    return int(np.max(np.maximum.accumulate(t) - t)) if len(t) else 0


def test_stream_hand_example_cluster_across_the_cut():
    """Two pixels of one hit on either side of a chunk cut, a second shot after them: the first push emits
    nothing (shot 0 is not complete), the second emits shot 0 as ONE hit of two pixels, final emits shot 1."""
    P, W = 1000, 5
    m = pp.StreamModel(P, 0)
    a = m.push([5], [5], [10], [3])
    assert (len(a["x"]), a["n_carry"], a["n_late"]) == (0, 1, 0)
    b = m.push([5, 9], [6, 9], [11, 1004], [4, 7])
    assert b["toa"].tolist() == [10, 11] and b["n_carry"] == 1 and b["label_base"] == 0
    r = oracle.run(b["x"], b["y"], b["toa"], b["tot"], W, P)
    assert r["n_clusters"] == 1 and r["c_size"].tolist() == [2] and r["c_sum_tot_y"].tolist() == [3 * 5 + 4 * 6]
    c = m.push([], [], [], [], final=True)
    assert c["toa"].tolist() == [1004] and c["label_base"] == 2 and c["n_carry"] == 0


def test_stream_late_event_is_counted_not_clustered():
    P = 100
    m = pp.StreamModel(P, 0)                     # the stream claims to be in order
    a = m.push([1, 2], [1, 2], [10, 250], [5, 5])
    assert a["toa"].tolist() == [10] and a["n_carry"] == 1
    b = m.push([3], [3], [20], [5])              # shot 0 went out already
    assert b["n_late"] == 1 and len(b["x"]) == 0 and m.late_total == 1
    m2 = pp.StreamModel(P, 240)                  # with the true disorder bound nothing is late
    a2 = m2.push([1, 2], [1, 2], [10, 250], [5, 5])
    assert len(a2["x"]) == 0 and a2["n_carry"] == 2
    b2 = m2.push([3], [3], [20], [5], final=True)
    assert b2["toa"].tolist() == [10, 250, 20] and b2["n_late"] == 0


@pytest.mark.parametrize("cfg,shots,sizes", [
    (0, 12, "ones"), (0, 40, 997), (0, 40, "random"), (0, 40, "whole"), (4, 6, 4099), (4, 6, "random"),
])
def test_stream_model_equals_batch(cfg, shots, sizes):
    """The definition: the hits of the chunked stream, in order, ARE the batch hits of the whole stream —
    every column, labels included — wherever the cuts fall (inside shots, inside hits, chunks of one event,
    one chunk for everything), for an in-order stream (D = 0) and a locally shuffled one (D = its bound)."""
    w = gen.generate(cfg, shots=shots)
    if cfg == 4:
        assert _disorder(w.toa) > 0
    rng = np.random.default_rng(5)
    if sizes == "ones":
        sz = [1] * w.n
    elif sizes == "whole":
        sz = [w.n]
    elif sizes == "random":
        sz = []
        while sum(sz) < w.n:
            sz.append(int(min(rng.integers(1, max(2, w.n // 9)), w.n - sum(sz))))
    else:
        sz = [sizes] * (w.n // sizes) + ([w.n % sizes] if w.n % sizes else [])
    m = pp.StreamModel(P, _disorder(w.toa))
    rows, stats = _stream_rows(m, _cut(w, sz), W, P)
    ref = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    assert m.late_total == 0 and sum(s[0] for s in stats) == w.n
    for k, v in rows.items():
        assert np.array_equal(v, ref[k]), k
    if sizes not in ("whole",):
        assert max(s[1] for s in stats) > 0          # something was carried: the cuts were not shot-aligned


def test_stream_carry_is_bounded_by_the_open_shots():
    """In-order stream: what is carried is never more than the events of the shot still open."""
    w = gen.generate(0, shots=30)
    m = pp.StreamModel(P, 0)
    per_shot = np.bincount((w.toa // np.uint64(P)).astype(np.int64)).max()
    for c in _cut(w, [500] * (w.n // 500) + [w.n % 500]):
        e = m.push(*c)
        assert e["n_carry"] <= per_shot
        assert all(t // P >= m.s_emitted for t in (ev[2] for ev in m.carry))


# ------------------------------------------------------------------ the oracle under the sanitizers
def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    """oracle/tpx3_oracle.cpp rebuilt with -fsanitize=address,undefined (any report aborts the program) and run
    on seeded inputs of every kind the pins use — in-order, shuffled, noise pixels, one event, none — gives the
    outputs of the ordinary build, digest for digest, with nothing on stderr."""
    import ctypes
    import shutil
    import subprocess

    if shutil.which("g++") is None:
        pytest.skip("g++ not available")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    exe = str(tmp_path / "oracle_asan")
    cmd = ["g++", "-O1", "-g", "-std=c++17", "-fopenmp", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           os.path.join(root, "oracle", "sanitize_driver.cpp"), os.path.join(root, "oracle", "tpx3_oracle.cpp"), "-o", exe]
    build = subprocess.run(cmd, capture_output=True, text=True)
    if build.returncode != 0 and "sanitize" in build.stderr.lower():
        pytest.skip("this toolchain has no sanitizer runtime: " + build.stderr[-200:])
    assert build.returncode == 0, build.stderr

    def fnv(h, a):
        for b in np.ascontiguousarray(a).view(np.uint8).tobytes():
            h = ((h ^ b) * 1099511628211) & 0xFFFFFFFFFFFFFFFF
        return h

    def digest(o, second):
        h = 1469598103934665603
        for k in ("perm", second, "c_label", "c_size", "c_shot", "c_sum_tot", "c_sum_tot_x", "c_sum_tot_y",
                  "c_toa_peak", "c_cx", "c_cy", "c_sum_tot_tof", "c_ctof"):
            h = fnv(h, o[k])
        return "%016x" % h

    cases = [gen.generate(0, shots=60), gen.generate(4, shots=12), gen.generate(3, shots=3)]
    one = gen.generate(0, shots=1)
    for w, n in [(c, c.n) for c in cases] + [(one, 1), (one, 0)]:
        d = tmp_path / ("case_%d_%d" % (w.cfg_id, n))
        d.mkdir()
        w.x[:n].tofile(d / "x.u16"); w.y[:n].tofile(d / "y.u16"); w.toa[:n].tofile(d / "toa.u64"); w.tot[:n].tofile(d / "tot.u16")
        for threads in (1, 3):
            r = subprocess.run([exe, str(d), str(W), str(P), "2", "1", "200", str(threads)], capture_output=True, text=True,
                               env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1"))
            assert r.returncode == 0 and r.stderr.strip() == "", (r.returncode, r.stderr[-2000:])
            lines = r.stdout.strip().splitlines()
            o = oracle.run(w.x[:n], w.y[:n], w.toa[:n], w.tot[:n], W, P, threads=1)
            lm = oracle.run_localmax(w.x[:n], w.y[:n], w.toa[:n], w.tot[:n], 2, 1, 200, P, threads=1)
            assert lines[0] == "run n=%d hits=%d digest=%s" % (n, o["n_clusters"], digest(o, "label"))
            assert lines[1] == "localmax n=%d hits=%d digest=%s" % (n, lm["n_clusters"], digest(lm, "lmax"))
