"""GPU fuzz: random shot-structured streams through every route of the library against the CPU oracle.

Bounded (a few hundred streams, about 20 s); the seeds are fixed, so a failure reproduces. Shot sizes are drawn
around the tile windows (2048 / 4096 / 8192 events), shot numbers have gaps, the order inside a shot is sorted or
shuffled, pixels repeat, and the link window runs from 0 to 3000 ticks. Every output is compared element by
element, as in tests/test_gpu_parity.py (whose helpers it uses).
"""
import numpy as np
import pytest

import oracle
from oracle import preprocess as opp

import test_gpu_parity as T

pytestmark = pytest.mark.gpu
P = T.P


@pytest.fixture(scope="module")
def tpx3():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    import paper_2603_04942_b200 as m

    m.load_library()
    return m


def _random_stream(rng):
    kind = int(rng.integers(0, 6))
    nshots = int(rng.integers(1, 40))
    if kind == 0:
        sizes = rng.integers(1, 50, nshots)
    elif kind == 1:
        sizes = rng.integers(1900, 2060, nshots)                     # around the 2048-event window
    elif kind == 2:
        sizes = rng.choice([1, 2, 7, 8, 9, 2039, 2040, 2041, 4088, 300], nshots)
    elif kind == 3:
        sizes = rng.integers(200, 1500, nshots)
    elif kind == 4:
        sizes = rng.choice([0, 0, 1, 5000, 3, 800], nshots)          # empty shots: gaps in the shot numbers
    else:
        sizes = rng.integers(3000, 8300, max(1, nshots // 6))
    shot_ids = np.cumsum(rng.integers(1, 4, len(sizes)))
    n = int(sizes.sum())
    shot = np.repeat(shot_ids, sizes)
    tof = rng.integers(0, int(rng.choice([64, 400, 5000, 60000])), n)
    side = int(rng.choice([8, 40, 256]))
    x = rng.integers(0, side, n).astype(np.uint16)
    y = rng.integers(0, side, n).astype(np.uint16)
    tot = rng.integers(1, 1024, n).astype(np.uint16)
    toa = (shot * P + tof).astype(np.uint64)
    idx = np.lexsort((tof, shot)) if rng.random() < 0.4 else np.lexsort((rng.random(n), shot))
    return x[idx], y[idx], toa[idx], tot[idx], sizes


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_fuzz_cluster_routes(tpx3, seed):
    """tpx3_cluster_centroid and tpx3_cluster + tpx3_centroid, tile kernel with every hint (the ladder included) and
    the forced general route (global sort + tile kernel through perm, slab hash for shots beyond a window)."""
    m = tpx3
    rng = np.random.default_rng(seed)
    done = 0
    while done < 60:
        x, y, toa, tot, sizes = _random_stream(rng)
        if len(x) == 0:
            continue
        done += 1
        hint = int(rng.choice([0, int(sizes.max()), 512, 1536, 3584, 8184]))
        flags = int(rng.choice([0, 0, 0, m.FLAG_FORCE_GENERAL]))
        Wr = int(rng.choice([0, 5, 320, 3000]))
        o = oracle.run(x, y, toa, tot, Wr, P)
        for mode in ("fused", "split"):
            g = T.run_gpu(m, x, y, toa, tot, Wr, P, mode=mode, flags=flags, max_shot_hits=hint)
            assert g["status"]["error"] == 0, g["status"]
            T.assert_parity(g, o, "seed %d stream %d hint %d flags %d W %d %s" % (seed, done, hint, flags, Wr, mode))
        if done % 10 == 0 and len(x) < 30000:
            T.check_localmax(m, x, y, toa, tot, int(rng.integers(0, 4)), int(rng.integers(0, 4)), int(rng.choice([0, 7, 320])),
                             what="seed %d stream %d" % (seed, done), hints=(hint,))


@pytest.mark.parametrize("seed", [21, 22])
def test_fuzz_preprocess_and_stream(tpx3, seed):
    """The fused preprocessing call against oracle.preprocess -> oracle.run, and the surviving stream through stream
    pushes of random sizes against the batch oracle."""
    import torch

    m = tpx3
    rng = np.random.default_rng(seed)
    W = T.W
    for it in range(60):
        nshots = int(rng.integers(1, 25))
        kind = int(rng.integers(0, 4))
        sizes = [rng.integers(1, 60, nshots), rng.integers(300, 1400, nshots), rng.choice([1, 2040, 7, 1900, 500], nshots),
                 rng.integers(1500, 3500, max(1, nshots // 3))][kind]
        n = int(sizes.sum())
        shot = np.repeat(np.arange(len(sizes)), sizes)
        trig = (np.cumsum(rng.integers(P - 3000, P + 3000, len(sizes))) + 777).astype(np.uint64)
        cut = int(rng.choice([100, 5000, 60000]))
        tof = rng.integers(0, int(cut * 1.3) + 2, n)
        tof[rng.random(n) < 0.02] += 200000                                  # dark counts far beyond the cut
        toa = trig[shot].astype(np.int64) + tof
        if rng.random() < 0.3 and sizes[0] > 3:
            toa[:3] = int(trig[0]) - rng.integers(1, 50, 3)                  # before the first trigger
        x = rng.integers(0, 40, n).astype(np.uint16)
        y = rng.integers(0, 40, n).astype(np.uint16)
        tot = rng.integers(1, 1500, n).astype(np.uint16)
        table = None if rng.random() < 0.2 else np.round(
            rng.integers(-30, 200) / (np.arange(int(rng.choice([4, 64, 1024]))) + 1.0) ** 0.7).astype(np.int32)
        idx = np.lexsort((toa, shot)) if rng.random() < 0.5 else np.lexsort((rng.random(n), shot))
        x, y, toa, tot = x[idx], y[idx], toa[idx].astype(np.uint64), tot[idx]
        sb = int(rng.integers(0, 1000))
        ex, ey, et, eo, ei = opp.preprocess(x, y, toa, tot, trig, cut, [] if table is None else table, P, sb)
        o = dict(oracle.run(ex, ey, et, eo, W, P))
        o["perm"] = ei[o["perm"]].astype(np.uint32)
        pl = m.plan(m.Config(max_hits=n, toa_window_ticks=W, shot_period_ticks=P, max_shot_hits=int(sizes.max())))
        cl = m.Clusters(n, pl.device)
        perm, label, nc, nk = pl.preprocess_cluster_centroid(T.to_dev(x), T.to_dev(y), T.to_dev(toa), T.to_dev(tot), T.to_dev(trig),
                                                             cut, None if table is None else T.to_dev(table), sb, cl)
        torch.cuda.synchronize()
        st = pl.status()
        assert st["error"] == 0, (seed, it, st)
        k, ncl = int(nk.cpu().numpy()[0]), int(nc.cpu().numpy()[0])
        assert k == len(ei)
        g = {"perm": perm[:k].cpu().numpy(), "label": label[:k].cpu().numpy(), "n_clusters": ncl}
        g.update(cl.numpy(ncl))
        T.assert_parity(g, o, "fused preprocessing, seed %d stream %d" % (seed, it))
        pl.free()
        if k and it % 2 == 0:
            w = type("W", (), {})()
            w.x, w.y, w.toa, w.tot, w.n = ex, ey, et, eo, k
            D = T._disorder(et)
            chunks = []
            while sum(chunks) < k:
                chunks.append(int(min(rng.choice([1, 13, 700, 5000, 40000]), k - sum(chunks))))
            rows, infos, _ = T.run_stream(m, w, chunks, D, max_carry=int(sizes.max()) * 4 + 64, max_shot_hits=int(sizes.max()))
            o2 = oracle.run(ex, ey, et, eo, W, P)
            for key in T._ROW_KEYS:
                np.testing.assert_array_equal(rows[key], o2[key], err_msg="stream, seed %d stream %d: %s" % (seed, it, key))
            T._check_push_properties(infos, et, chunks, D)
