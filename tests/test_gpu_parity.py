"""GPU parity tests: the CUDA path (through the C ABI, include/tpx3.h) against the CPU oracle,
element by element, on the same seeded inputs.

Bar (BASELINE.json north_star): perm, label, hit count and the integer sums bit-exact; toa_peak,
shot, size bit-exact; centroids within 1e-6 px absolute — asserted here as exact fp32 equality
as well, because both sides compute fp32(int64)/fp32(int64) with an IEEE RN divide (R12).
"""
import numpy as np
import pytest

import gen
import oracle

pytestmark = pytest.mark.gpu

W, P = 320, 640000
CENTROID_TOL = 1e-6  # px, north_star


@pytest.fixture(scope="module")
def tpx3():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    import paper_2603_04942_b200 as m

    m.load_library()
    return m


def to_dev(a):
    import torch

    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_gpu(m, x, y, toa, tot, W=W, P=P, mode="fused", flags=0, max_clusters=None, sensor=(256, 256),
            max_shot_hits=0):
    """mode: 'fused' = tpx3_cluster_centroid; 'split' = tpx3_cluster then tpx3_centroid."""
    import torch

    n = len(x)
    pl = m.plan(m.Config(sensor_w=sensor[0], sensor_h=sensor[1], toa_window_ticks=W, shot_period_ticks=P,
                         max_hits=max(n, 1), flags=flags, max_shot_hits=max_shot_hits))
    dx, dy, dtoa, dtot = (to_dev(np.asarray(x, dtype=np.uint16)), to_dev(np.asarray(y, dtype=np.uint16)),
                          to_dev(np.asarray(toa, dtype=np.uint64)), to_dev(np.asarray(tot, dtype=np.uint16)))
    cap = n if max_clusters is None else max_clusters
    cl = m.Clusters(cap, pl.device)
    if mode == "fused":
        perm, label, nc = pl.cluster_centroid(dx, dy, dtoa, dtot, cl)
    else:
        perm, label, nc = pl.cluster(dx, dy, dtoa, dtot)
        nc_a = int(nc.cpu().numpy()[0])
        nc = pl.centroid(dx, dy, dtoa, dtot, perm, label, cl)
        assert int(nc.cpu().numpy()[0]) == nc_a
    torch.cuda.synchronize()
    st = pl.status()
    ncl = int(nc.cpu().numpy()[0])
    out = {"perm": perm[:n].cpu().numpy(), "label": label[:n].cpu().numpy(), "n_clusters": ncl, "status": st}
    out.update(cl.numpy(min(ncl, cap)))
    pl.free()
    return out


def assert_parity(g, o, what=""):
    assert g["n_clusters"] == o["n_clusters"], what
    np.testing.assert_array_equal(g["perm"], o["perm"], err_msg=what + " perm")
    np.testing.assert_array_equal(g["label"], o["label"], err_msg=what + " label")
    for k in ("c_label", "c_size", "c_shot", "c_sum_tot", "c_sum_tot_x", "c_sum_tot_y", "c_toa_peak", "c_sum_tot_tof"):
        np.testing.assert_array_equal(g[k], o[k], err_msg=what + " " + k)
    np.testing.assert_array_equal(g["c_ctof"], o["c_ctof"], err_msg=what + " c_ctof (bitwise fp32)")
    for k in ("c_cx", "c_cy"):
        assert np.all(np.abs(g[k].astype(np.float64) - o[k].astype(np.float64)) <= CENTROID_TOL), what + " " + k
        np.testing.assert_array_equal(g[k], o[k], err_msg=what + " " + k + " (bitwise fp32)")


def check(m, x, y, toa, tot, W=W, P=P, modes=("fused", "split"), flags=0, what="", max_shot_hits=0):
    o = oracle.run(x, y, toa, tot, W, P, threads=0)
    res = None
    for mode in modes:
        res = run_gpu(m, x, y, toa, tot, W, P, mode=mode, flags=flags, max_shot_hits=max_shot_hits)
        assert res["status"]["error"] == 0
        assert_parity(res, o, "%s [%s]" % (what, mode))
    return res, o


# ------------------------------------------------------------------ the five configs
def test_cfg0_full(tpx3):
    w = gen.generate(0)  # ~75k hits, 1000 shots: several tiles and a ragged tail
    res, o = check(tpx3, w.x, w.y, w.toa, w.tot, modes=("split", "fused"), what="cfg0")
    assert o["n_clusters"] > 9000
    assert res["status"]["path"] == 1  # the fused shot-tile kernel served the call


@pytest.mark.parametrize("cfg,shots", [(1, 3000), (2, 1500), (3, 600), (4, 1500)])
def test_cfg_subsets(tpx3, cfg, shots):
    w = gen.generate(cfg, shots=shots)
    res, _ = check(tpx3, w.x, w.y, w.toa, w.tot, modes=("split", "fused"), what="cfg%d" % cfg)
    assert res["status"]["path"] == 1


@pytest.mark.parametrize("cfg,shots,hint", [(0, 1000, 256), (1, 3000, 640), (1, 3000, 1024), (2, 1200, 1536),
                                            (4, 1200, 1536), (4, 1200, 4096)])
def test_fused_tile_variants(tpx3, cfg, shots, hint):
    # max_shot_hits picks the tile variant (2048-event tiles for <= 512, 4096 for <= 1024, 8192 otherwise)
    # and the slice length
    w = gen.generate(cfg, shots=shots)
    res, _ = check(tpx3, w.x, w.y, w.toa, w.tot, modes=("fused",), max_shot_hits=hint, what="cfg%d hint %d" % (cfg, hint))
    assert res["status"]["path"] == 1


def test_fused_falls_back_when_a_shot_exceeds_the_hint(tpx3):
    w = gen.generate(3, shots=100)  # ~2100 events per shot
    res, _ = check(tpx3, w.x, w.y, w.toa, w.tot, modes=("fused",), max_shot_hits=512, what="cfg3 hint 512")
    assert res["status"]["path"] == 2


def test_fused_shots_aligned_with_slices(tpx3):
    # shots of exactly S = 4096 and 2048 events: shot starts fall exactly on slice boundaries
    rng = np.random.default_rng(3)
    for per in (4096, 2048, 1):
        shots = 40 if per > 1 else 9000
        n = per * shots
        x = rng.integers(0, 256, n); y = rng.integers(0, 256, n)
        toa = (np.repeat(np.arange(shots), per) * P + rng.integers(0, 60000, n)).astype(np.uint64)
        tot = rng.integers(1, 1024, n)
        res, _ = check(tpx3, x, y, toa, tot, modes=("fused",), what="aligned %d" % per)
        assert res["status"]["path"] == 1


def test_fused_sparse_shot_numbers(tpx3):
    # empty shots in between and a shot number jump too wide for the 32-bit tile key
    rng = np.random.default_rng(4)
    n = 30000
    shot = np.sort(rng.integers(0, 200, n)) * 37
    x = rng.integers(0, 64, n); y = rng.integers(0, 64, n)
    toa = (shot * P + rng.integers(0, 20000, n)).astype(np.uint64)
    tot = rng.integers(1, 1024, n)
    res, _ = check(tpx3, x, y, toa, tot, modes=("fused",), what="sparse shots")
    assert res["status"]["path"] == 1
    shot2 = shot.astype(np.uint64).copy()
    shot2[n // 2:] += np.uint64(1 << 40)
    toa2 = shot2 * np.uint64(P) + (toa % np.uint64(P))
    res, _ = check(tpx3, x, y, toa2, tot, modes=("fused",), what="shot jump")
    assert res["status"]["path"] in (1, 2)


def test_cfg4_requires_sort(tpx3):
    w = gen.generate(4, shots=300)
    assert np.any(np.diff(w.toa.astype(np.int64)) < 0)  # delivered out of order
    res, o = check(tpx3, w.x, w.y, w.toa, w.tot, what="cfg4")
    assert np.any(res["perm"] != np.arange(w.n))


def test_force_general_path(tpx3):
    w = gen.generate(2, shots=800)
    res, _ = check(tpx3, w.x, w.y, w.toa, w.tot, flags=tpx3.FLAG_FORCE_GENERAL, modes=("fused",), what="general")
    assert res["status"]["path"] == 2


def test_globally_shuffled_input(tpx3):
    # shots interleaved in the stream: not shot-contiguous, the general path (global sort) must run
    w = gen.generate(2, shots=500)
    rng = np.random.default_rng(7)
    p = rng.permutation(w.n)
    check(tpx3, w.x[p], w.y[p], w.toa[p], w.tot[p], modes=("split",), what="shuffled")
    res, _ = check(tpx3, w.x[p], w.y[p], w.toa[p], w.tot[p], modes=("fused",), what="shuffled")
    assert res["status"]["path"] == 2


def test_single_shot_P0(tpx3):
    # P = 0: the whole input is one shot (links may cross the 640000-tick boundaries)
    w = gen.generate(1, shots=400)
    check(tpx3, w.x, w.y, w.toa, w.tot, P=0, what="P=0")


def test_dense_single_shot_chain(tpx3):
    # one shot far larger than any tile, dense in time: long chains across slabs
    rng = np.random.default_rng(11)
    n = 300000
    x = rng.integers(0, 256, n); y = rng.integers(0, 256, n)
    toa = np.sort(rng.integers(0, 600000, n)).astype(np.uint64) + 5 * P
    tot = rng.integers(1, 1024, n)
    check(tpx3, x, y, toa, tot, what="dense shot")
    check(tpx3, x, y, toa, tot, W=3, what="dense shot W=3")


# ------------------------------------------------------------------ edge cases
def test_empty_and_single(tpx3):
    z16 = np.zeros(0, dtype=np.uint16); z64 = np.zeros(0, dtype=np.uint64)
    for mode in ("fused", "split"):
        r = run_gpu(tpx3, z16, z16, z64, z16, mode=mode)
        assert r["n_clusters"] == 0 and r["status"]["error"] == 0
    check(tpx3, [7], [9], [123456789], [55], what="single")


def test_all_identical(tpx3):
    n = 5000
    check(tpx3, np.full(n, 100), np.full(n, 17), np.full(n, 10**9), np.full(n, 3), what="identical")


def test_window_inclusive_and_shot_boundary(tpx3):
    # dt == W links, dt == W+1 does not ("<="); sP-1 | sP never link (R6)
    x = [10, 11, 50, 51, 90, 91]; y = [10, 10, 50, 50, 90, 90]
    toa = [1000, 1000 + W, 5000, 5000 + W + 1, 3 * P - 1, 3 * P]
    res, o = check(tpx3, x, y, toa, [5, 6, 7, 8, 9, 10], what="window")
    assert res["n_clusters"] == 5


def test_chain_longer_than_window(tpx3):
    # A-B-C with |tA - tC| > W: one component by transitivity
    n = 4000
    x = (np.arange(n) % 200) + 20; y = np.full(n, 100) + (np.arange(n) // 200 % 2)
    toa = 7 * P + np.arange(n) * 100
    res, o = check(tpx3, x, y, toa, np.full(n, 9), what="chain")


def test_corners_and_repeated_addresses(tpx3):
    x = [0, 0, 255, 255, 0, 255, 128, 128, 128]; y = [0, 0, 255, 255, 255, 0, 128, 128, 128]
    toa = [10, 20, 30, 40, 50, 60, 70, 70 + W, 70 + 2 * W]
    check(tpx3, x, y, toa, [1, 2, 3, 4, 5, 6, 7, 8, 9], what="corners")


def test_tie_break_later_pixel_wins(tpx3):
    res, o = check(tpx3, [10, 11, 12], [5, 5, 5], [100, 100, 100], [7, 9, 9], what="tie")
    assert res["c_toa_peak"].tolist() == [100]


@pytest.mark.parametrize("seed", range(6))
def test_random_small(tpx3, seed):
    rng = np.random.default_rng(100 + seed)
    n = int(rng.integers(2, 3000))
    side = int(rng.integers(4, 40))
    x = rng.integers(0, side, n); y = rng.integers(0, side, n)
    toa = rng.integers(0, 4 * P, n).astype(np.uint64)
    tot = rng.integers(1, 1024, n)
    Wr = int(rng.choice([0, 1, 320, 5000, 700000]))
    Pr = int(rng.choice([0, P, 1000]))
    check(tpx3, x, y, toa, tot, W=Wr, P=Pr, what="random %d" % seed)


def test_large_values(tpx3):
    # ToT up to 65535, ToA near 2^63: integer sums stay exact
    rng = np.random.default_rng(5)
    n = 20000
    x = rng.integers(250, 256, n); y = rng.integers(250, 256, n)
    toa = (np.uint64(1) << np.uint64(62)) + rng.integers(0, 10 * P, n).astype(np.uint64)
    tot = rng.integers(60000, 65536, n)
    check(tpx3, x, y, toa, tot, what="large values")


def test_centroid_accepts_oracle_labels(tpx3):
    # tpx3_centroid is defined on ANY valid (perm, label): feed it the oracle's
    import torch

    w = gen.generate(2, shots=300)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    pl = tpx3.plan(tpx3.Config(max_hits=w.n))
    cl = tpx3.Clusters(w.n, pl.device)
    nc = pl.centroid(to_dev(w.x), to_dev(w.y), to_dev(w.toa), to_dev(w.tot), to_dev(o["perm"]), to_dev(o["label"]), cl)
    torch.cuda.synchronize()
    ncl = int(nc.cpu().numpy()[0])
    g = {"perm": o["perm"], "label": o["label"], "n_clusters": ncl}
    g.update(cl.numpy(ncl))
    assert_parity(g, o, "oracle labels")


@pytest.mark.parametrize("cfg,shots,hint", [(1, 2000, 600), (4, 1200, 1500), (3, 300, 3360), (4, 1200, 0)])
def test_split_calls_take_the_tile_kernel(tpx3, cfg, shots, hint):
    """tpx3_cluster (S0-S3) and tpx3_centroid (S4-S5) run in the fused tile kernel too (labels only / labels
    given): same outputs as the oracle, and the status word says which path served each call."""
    import torch

    w = gen.generate(cfg, shots=shots)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    pl = tpx3.plan(tpx3.Config(max_hits=w.n, max_shot_hits=hint))
    dev = [to_dev(a) for a in (w.x, w.y, w.toa, w.tot)]
    perm, label, nc = pl.cluster(*dev)
    torch.cuda.synchronize()
    st = pl.status()
    assert st["error"] == 0 and st["path"] == 1, st
    assert int(nc.cpu().numpy()[0]) == o["n_clusters"]
    np.testing.assert_array_equal(perm[: w.n].cpu().numpy(), o["perm"])
    np.testing.assert_array_equal(label[: w.n].cpu().numpy(), o["label"])
    cl = tpx3.Clusters(w.n, pl.device)
    nc2 = pl.centroid(*dev, perm, label, cl)
    torch.cuda.synchronize()
    st = pl.status()
    assert st["error"] == 0 and st["path"] == 1, st
    ncl = int(nc2.cpu().numpy()[0])
    g = {"perm": o["perm"], "label": o["label"], "n_clusters": ncl}
    g.update(cl.numpy(ncl))
    assert_parity(g, o, "split cfg%d" % cfg)
    pl.free()


@pytest.mark.parametrize("off,poff", [(1, 0), (2, 3), (3, 1), (5, 2), (7, 7), (8, 5), (12347, 1)])
def test_chunks_of_a_resident_stream_at_any_offset(tpx3, off, poff):
    """Inputs (and outputs) that are views into larger device arrays at any element offset - a chunk of a resident
    stream cut at a shot boundary - are not 16-byte aligned; the tile kernel still serves them (the arrays are moved down
    to the boundary alike, FusedArgs::head): every route, outputs in the caller's numbering."""
    import torch

    w = gen.generate(4, shots=60)
    n = w.n
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    pad = lambda a: to_dev(np.concatenate([np.full(off, 7, a.dtype), a, np.full(9, 7, a.dtype)]))[off:off + n]  # noqa: E731
    dev = [pad(a) for a in (w.x, w.y, w.toa, w.tot)]
    assert dev[0].data_ptr() % 16 == (2 * off) % 16
    for flags, want_path in ((0, 1), (tpx3.FLAG_FORCE_GENERAL, 2)):
        pl = tpx3.plan(tpx3.Config(max_hits=n, max_shot_hits=1500, flags=flags))
        mk = lambda: torch.full((n + poff + 8,), 0xDEAD, dtype=torch.uint32, device="cuda")  # noqa: E731
        pbuf, lbuf = mk(), mk()
        perm, label = pbuf[poff:poff + n], lbuf[poff:poff + n]
        cl = tpx3.Clusters(n, pl.device)
        _, _, nc = pl.cluster_centroid(*dev, cl, perm=perm, label=label)
        torch.cuda.synchronize()
        st = pl.status()
        assert st["error"] == 0 and st["path"] == want_path, st
        ncl = int(nc.cpu().numpy()[0])
        g = {"perm": perm.cpu().numpy(), "label": label.cpu().numpy(), "n_clusters": ncl}
        g.update(cl.numpy(ncl))
        assert_parity(g, o, "offset %d flags %d" % (off, flags))
        assert int(pbuf[poff + n].cpu()) == 0xDEAD and (poff == 0 or int(pbuf[poff - 1].cpu()) == 0xDEAD)   # nothing beside the view
        assert int(lbuf[poff + n].cpu()) == 0xDEAD and (poff == 0 or int(lbuf[poff - 1].cpu()) == 0xDEAD)
        # the two calls: labels only, then the sums on those (perm is read by position there)
        pbuf2, lbuf2 = mk(), mk()
        perm2, label2 = pbuf2[poff:poff + n], lbuf2[poff:poff + n]
        pl.cluster(*dev, perm=perm2, label=label2)
        cl2 = tpx3.Clusters(n, pl.device)
        nc2 = pl.centroid(*dev, perm2, label2, cl2)
        torch.cuda.synchronize()
        st = pl.status()
        assert st["error"] == 0 and (flags or st["path"] == 1), st
        g2 = {"perm": perm2.cpu().numpy(), "label": label2.cpu().numpy(), "n_clusters": int(nc2.cpu().numpy()[0])}
        g2.update(cl2.numpy(g2["n_clusters"]))
        assert_parity(g2, o, "split, offset %d flags %d" % (off, flags))
        pl.free()
    # the paper-literal mode on the same views
    if off in (3, 12347):
        olm = oracle.run_localmax(w.x, w.y, w.toa, w.tot, 2, 1, 200, P)
        for flags in (0, tpx3.FLAG_FORCE_GENERAL):
            pl = tpx3.plan(tpx3.Config(max_hits=n, max_shot_hits=1500, flags=flags))
            pbuf, lbuf = torch.zeros(n + poff + 8, dtype=torch.uint32, device="cuda"), torch.zeros(n + poff + 8, dtype=torch.uint32, device="cuda")
            cl = tpx3.Clusters(n, pl.device)
            _, _, nh = pl.localmax_centroid(*dev, 2, 1, 200, cl, perm=pbuf[poff:poff + n], lmax=lbuf[poff:poff + n])
            torch.cuda.synchronize()
            st = pl.status()
            assert st["error"] == 0 and st["path"] == 3, st
            k = int(nh.cpu().numpy()[0])
            assert k == olm["n_clusters"]
            np.testing.assert_array_equal(pbuf[poff:poff + n].cpu().numpy(), olm["perm"])
            np.testing.assert_array_equal(lbuf[poff:poff + n].cpu().numpy(), olm["lmax"])
            got = cl.numpy(k)
            for key in LM_KEYS:
                np.testing.assert_array_equal(got[key], olm[key], err_msg="localmax offset %d flags %d %s" % (off, flags, key))
            pl.free()
    # arrays that are NOT aligned alike (x one element further than the others): still the right answer, general route
    if off == 1:
        pl = tpx3.plan(tpx3.Config(max_hits=n, max_shot_hits=1500))
        xs = to_dev(np.concatenate([np.zeros(2, np.uint16), w.x]))[2:]
        cl = tpx3.Clusters(n, pl.device)
        perm, label, nc = pl.cluster_centroid(xs, dev[1], dev[2], dev[3], cl)
        torch.cuda.synchronize()
        st = pl.status()
        assert st["error"] == 0 and st["path"] == 2, st
        g = {"perm": perm[:n].cpu().numpy(), "label": label[:n].cpu().numpy(), "n_clusters": int(nc.cpu().numpy()[0])}
        g.update(cl.numpy(g["n_clusters"]))
        assert_parity(g, o, "unlike alignment")
        pl.free()


def test_centroid_with_hits_that_cross_shots(tpx3):
    """tpx3_centroid takes ANY valid (perm, label): here every event of the stream is declared one hit (label 0),
    so the hit crosses every shot and every tile: the tile kernel gives up and the general kernels serve the
    call. Expected row recomputed with numpy from the definition (Eq. 8-9)."""
    import torch

    w = gen.generate(1, shots=40)
    n = w.n
    perm = np.argsort(w.toa, kind="stable").astype(np.uint32)
    label = np.zeros(n, dtype=np.uint32)
    # and a second variant: two hits, the second one starting in the middle of a shot
    cut = int(w.shot_offsets[17]) + 5
    label2 = np.where(np.arange(n) < cut, 0, cut).astype(np.uint32)
    for lab in (label, label2):
        pl = tpx3.plan(tpx3.Config(max_hits=n, max_shot_hits=600))
        cl = tpx3.Clusters(16, pl.device)
        nc = pl.centroid(to_dev(w.x), to_dev(w.y), to_dev(w.toa), to_dev(w.tot), to_dev(perm), to_dev(lab), cl)
        torch.cuda.synchronize()
        assert pl.status()["error"] == 0
        roots = np.flatnonzero(lab == np.arange(n))
        assert int(nc.cpu().numpy()[0]) == len(roots)
        g = cl.numpy(len(roots))
        x, y, tot, toa = (a[perm].astype(np.int64) for a in (w.x, w.y, w.tot, w.toa))
        for i, r in enumerate(roots):
            m = lab == r
            assert g["c_label"][i] == r and g["c_size"][i] == m.sum()
            assert g["c_sum_tot"][i] == tot[m].sum()
            assert g["c_sum_tot_x"][i] == (tot[m] * x[m]).sum()
            assert g["c_sum_tot_y"][i] == (tot[m] * y[m]).sum()
            best = np.flatnonzero(m)[np.lexsort((np.flatnonzero(m), tot[m]))[-1]]   # max (ToT, sorted position)
            assert g["c_toa_peak"][i] == toa[best]
            assert g["c_cx"][i] == np.float32(np.float32((tot[m] * x[m]).sum()) / np.float32(tot[m].sum()))
        pl.free()


# ------------------------------------------------------------------ error behaviour
def test_capacity_error(tpx3):
    w = gen.generate(0, shots=50)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    for mode in ("fused", "split"):
        r = run_gpu(tpx3, w.x, w.y, w.toa, w.tot, mode=mode, max_clusters=10)
        assert r["status"]["error"] == tpx3.ERR_CAPACITY
        assert r["n_clusters"] == o["n_clusters"]  # the true count is still reported
        np.testing.assert_array_equal(r["c_sum_tot"], o["c_sum_tot"][:10])


def test_validate_input(tpx3):
    r = run_gpu(tpx3, [1, 2, 300], [1, 2, 3], [10, 20, 30], [5, 5, 5], flags=tpx3.FLAG_VALIDATE_INPUT)
    assert r["status"]["error"] == tpx3.ERR_OUT_OF_RANGE
    r = run_gpu(tpx3, [1, 2, 3], [1, 2, 3], [10, 20, 30], [5, 0, 5], flags=tpx3.FLAG_VALIDATE_INPUT)
    assert r["status"]["error"] == tpx3.ERR_OUT_OF_RANGE
    r = run_gpu(tpx3, [1, 2, 3], [1, 2, 3], [10, 20, 30], [5, 5, 5], flags=tpx3.FLAG_VALIDATE_INPUT)
    assert r["status"]["error"] == 0


def test_invalid_args(tpx3):
    with pytest.raises(tpx3.Tpx3Error):
        tpx3.plan(tpx3.Config(sensor_w=0))
    with pytest.raises(tpx3.Tpx3Error):
        tpx3.plan(tpx3.Config(max_hits=(1 << 28) + 1))
    pl = tpx3.plan(tpx3.Config(max_hits=16))
    with pytest.raises(tpx3.Tpx3Error):
        w = gen.generate(0, shots=5)
        pl.cluster(to_dev(w.x), to_dev(w.y), to_dev(w.toa), to_dev(w.tot))


def test_process_host_end_to_end(tpx3):
    import torch

    w = gen.generate(1, shots=500)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    pl = tpx3.plan(tpx3.Config(max_hits=w.n))
    hx, hy, htoa, htot = (torch.from_numpy(a).pin_memory() for a in (w.x, w.y, w.toa, w.tot))
    cl = tpx3.Clusters(w.n, "cpu", pin=True)
    perm = torch.empty(w.n, dtype=torch.uint32).pin_memory()
    label = torch.empty(w.n, dtype=torch.uint32).pin_memory()
    ncl = pl.process_host(hx, hy, htoa, htot, cl, perm, label)
    g = {"perm": perm.numpy(), "label": label.numpy(), "n_clusters": ncl}
    g.update(cl.numpy(ncl))
    assert_parity(g, o, "process_host")


# ------------------------------------------------------------------ full bench sizes
def _full_size_check(m, w, windows, hint):
    """The bench launch configuration (bench.py: max_hits = n, max_shot_hits = the recipe's bound) at a
    BASELINE.json full size: sampled shot windows element by element against the oracle, plus the
    size-independent invariants on the whole output."""
    import torch

    n = w.n
    pl = m.plan(m.Config(max_hits=n, toa_window_ticks=W, shot_period_ticks=P, max_shot_hits=hint))
    dev = [to_dev(a) for a in (w.x, w.y, w.toa, w.tot)]
    cl = m.Clusters(max(n // 2, 1024), pl.device)
    perm, label, nc = pl.cluster_centroid(*dev, cl)
    torch.cuda.synchronize()
    st = pl.status()
    assert st["error"] == 0 and st["path"] == 1, st
    ncl = int(nc.cpu().numpy()[0])
    perm, label = perm[:n].cpu().numpy(), label[:n].cpu().numpy()
    c = cl.numpy(ncl)
    pl.free()
    # invariants that hold at any size
    k = np.arange(n, dtype=np.uint32)
    assert np.all(label <= k) and np.array_equal(label[label], label)
    assert int(np.count_nonzero(label == k)) == ncl
    assert np.array_equal(c["c_label"], np.flatnonzero(label == k).astype(np.uint32))
    assert int(c["c_size"].sum()) == n
    assert int(c["c_sum_tot"].sum()) == int(w.tot.astype(np.int64).sum())
    assert int(c["c_sum_tot_x"].sum()) == int((w.tot.astype(np.int64) * w.x.astype(np.int64)).sum())
    assert int(c["c_sum_tot_y"].sum()) == int((w.tot.astype(np.int64) * w.y.astype(np.int64)).sum())
    seen = np.zeros(n, dtype=bool)
    seen[perm] = True
    assert seen.all()                                                                     # a permutation
    del seen
    st_toa = w.toa[perm]
    assert np.all(st_toa[1:] >= st_toa[:-1])                                              # in ToA order
    del st_toa
    # sampled shot windows, element by element (shots are contiguous in the stream: a window of shots
    # is a window of input positions and of sorted positions)
    off = w.shot_offsets
    for s0, s1 in windows:
        a, b = int(off[s0]), int(off[s1])
        s = w.slice_shots(s0, s1)
        o = oracle.run(s.x, s.y, s.toa, s.tot, W, P, threads=0)
        what = "shots [%d, %d)" % (s0, s1)
        np.testing.assert_array_equal(perm[a:b], o["perm"] + np.uint32(a), err_msg=what + " perm")
        np.testing.assert_array_equal(label[a:b], o["label"] + np.uint32(a), err_msg=what + " label")
        i0, i1 = np.searchsorted(c["c_label"], [a, b])
        assert i1 - i0 == o["n_clusters"], what
        np.testing.assert_array_equal(c["c_label"][i0:i1], o["c_label"] + np.uint32(a), err_msg=what)
        for key in ("c_size", "c_shot", "c_sum_tot", "c_sum_tot_x", "c_sum_tot_y", "c_toa_peak", "c_cx", "c_cy",
                    "c_sum_tot_tof", "c_ctof"):
            np.testing.assert_array_equal(c[key][i0:i1], o[key], err_msg=what + " " + key)
    return ncl


def _windows(shots, width, count):
    starts = np.linspace(0, shots - width, count).astype(np.int64)
    return [(int(s), int(s) + width) for s in starts]


def test_full_size_cfg1(tpx3):
    """BASELINE.json configs[1] in full (100 000 shots, 3.6e7 hits): the workload bench.py times."""
    w = gen.generate(1)
    ncl = _full_size_check(tpx3, w, _windows(w.shots, 400, 7), gen.max_shot_hits(1))
    assert ncl > 2_800_000


def test_full_size_cfg4_chunk_16M(tpx3):
    """One 2^24-hit chunk of config 4 (locally shuffled: the in-tile sort runs), bench configuration."""
    chunk = 1 << 24
    w = gen.generate(4, shots=chunk // 850 + 64, max_hits=chunk)
    _full_size_check(tpx3, w, _windows(w.shots, 150, 6), gen.max_shot_hits(4))


def test_full_size_cfg3_quarter(tpx3):
    """A quarter of config 3 (12 500 shots, 2.6e7 hits, about 2 100 hits per shot: the 8192-event tiles)."""
    w = gen.generate(3, shots=12500)
    _full_size_check(tpx3, w, _windows(w.shots, 60, 5), gen.max_shot_hits(3))


def test_full_size_cfg2(tpx3):
    """BASELINE.json configs[2] in full (200 000 shots, 1.8e8 hits)."""
    w = gen.generate(2)
    ncl = _full_size_check(tpx3, w, _windows(w.shots, 120, 7), gen.max_shot_hits(2))
    assert ncl > 8_500_000


def test_full_size_cfg3(tpx3):
    """BASELINE.json configs[3] in full (50 000 shots, 1.05e8 hits, noise pixels chaining the blobs)."""
    w = gen.generate(3)
    ncl = _full_size_check(tpx3, w, _windows(w.shots, 50, 7), gen.max_shot_hits(3))
    assert ncl > 11_000_000


@pytest.mark.parametrize("log2_chunk,count", [(26, 6), (28, 8)])
def test_full_size_cfg4_chunk(tpx3, log2_chunk, count):
    """One 2^26- and one 2^28-hit chunk of config 4 (locally shuffled: the in-tile sort runs) — 2^28 is the
    configuration bench.py times by default and the largest a plan accepts: 32-bit positions, the 12.9 GB
    staging table and about 10^5 tiles are at their limits. Sampled shot windows (first, last and spread over
    the chunk) element by element against the oracle; the invariants on the whole output."""
    chunk = 1 << log2_chunk
    w = gen.generate(4, shots=chunk // 850 + 64, max_hits=chunk)
    assert w.n > chunk - 2000
    _full_size_check(tpx3, w, _windows(w.shots, 150, count), gen.max_shot_hits(4))


def test_cfg4_rows_do_not_depend_on_the_chunk_size(tpx3):
    """one stretch of config 4 (2^26 hits) cut at shot boundaries into chunks of 2^20, 2^24 and
    2^26 hits gives the same hit rows (labels made global by the chunk's first position): every column, in
    order, not only as a multiset."""
    import torch

    m = tpx3
    n_max = 1 << 26
    w = gen.generate(4, shots=n_max // 850 + 64, max_hits=n_max)
    pl = m.plan(m.Config(max_hits=w.n, toa_window_ticks=W, shot_period_ticks=P, max_shot_hits=gen.max_shot_hits(4)))
    dev = [to_dev(a) for a in (w.x, w.y, w.toa, w.tot)]
    cl = m.Clusters(max(w.n // 2, 1024), pl.device)
    perm = torch.empty(w.n, dtype=torch.uint32, device=pl.device)
    label = torch.empty(w.n, dtype=torch.uint32, device=pl.device)
    nc = torch.zeros(1, dtype=torch.uint32, device=pl.device)
    off = w.shot_offsets
    ref = None
    for log2 in (26, 24, 20):
        rows = {k: [] for k in LM_KEYS}
        perm_all = np.empty(w.n, dtype=np.uint32)
        for s0, s1 in w.chunks(1 << log2):
            a, b = int(off[s0]), int(off[s1])
            pl.cluster_centroid(*(d[a:b] for d in dev), cl, perm=perm, label=label, n_clusters=nc)
            torch.cuda.synchronize()
            k = int(nc.cpu().numpy()[0])
            c = cl.numpy(k)
            c["c_label"] = c["c_label"] + np.uint32(a)
            for key in LM_KEYS:
                rows[key].append(c[key])
            perm_all[a:b] = perm[: b - a].cpu().numpy() + np.uint32(a)
        assert pl.status()["error"] == 0
        rows = {k: np.concatenate(v) for k, v in rows.items()}
        if ref is None:
            ref, ref_perm = rows, perm_all
            assert len(ref["c_label"]) > 3_000_000
        else:
            for key in LM_KEYS:
                np.testing.assert_array_equal(rows[key], ref[key], err_msg="chunks of 2^%d: %s" % (log2, key))
            np.testing.assert_array_equal(perm_all, ref_perm, err_msg="chunks of 2^%d: perm" % log2)
    pl.free()


def test_small_tile_variant_with_in_tile_sort(tpx3):
    """Shots of <= 120 events delivered out of order inside each shot, hint 128: the 2048-event tile
    variant has to run its in-tile sort."""
    w = gen.generate(0, shots=600)
    rng = np.random.default_rng(21)
    p = np.arange(w.n)
    off = w.shot_offsets
    for s in range(w.shots):
        a, b = int(off[s]), int(off[s + 1])
        p[a:b] = a + rng.permutation(b - a)
    res, _ = check(tpx3, w.x[p], w.y[p], w.toa[p], w.tot[p], modes=("fused",), max_shot_hits=128, what="cfg0 shuffled")
    assert res["status"]["path"] == 1
    assert np.any(res["perm"] != np.arange(w.n))


@pytest.mark.parametrize("hint", [600, 2000, 4000])
def test_in_tile_order_with_many_events_per_key(tpx3, hint):
    """Electron VMI delivered out of order inside each shot: a shot's 360 events share 95 ticks, so up to 20 events
    of one (shot, ToF) key fall into one position block and the rank by counting needs its 8-bit counter fields."""
    w = gen.generate(1, shots=800)
    rng = np.random.default_rng(5)
    p = np.arange(w.n)
    off = w.shot_offsets
    for s in range(w.shots):
        a, b = int(off[s]), int(off[s + 1])
        p[a:b] = a + rng.permutation(b - a)
    res, _ = check(tpx3, w.x[p], w.y[p], w.toa[p], w.tot[p], modes=("fused", "split"), max_shot_hits=hint,
                   what="cfg1 shuffled, hint %d" % hint)
    assert res["status"]["path"] == 1
    assert np.any(res["perm"] != np.arange(w.n))


def test_in_tile_order_falls_back_to_the_radix_sort(tpx3):
    """Hundreds of events with ONE key inside one position block overflow even the 8-bit counter fields: the stable
    LSD radix sort of the tile takes over. Two time values per shot, the later one delivered first."""
    rng = np.random.default_rng(8)
    shots, per = 12, 1400
    n = shots * per
    x = rng.integers(0, 256, n); y = rng.integers(0, 256, n)
    tof = np.tile(np.concatenate([np.full(per // 2, 900), np.full(per - per // 2, 100)]), shots)
    toa = (np.repeat(np.arange(shots), per) * P + tof).astype(np.uint64)
    tot = rng.integers(1, 1024, n)
    for hint in (1500, 3000):
        res, _ = check(tpx3, x, y, toa, tot, modes=("fused",), max_shot_hits=hint, what="two keys per shot, hint %d" % hint)
        assert res["status"]["path"] == 1


# ------------------------------------------------------------------ paper-literal mode (NEXT #2)
LM_KEYS = ("c_label", "c_size", "c_shot", "c_sum_tot", "c_sum_tot_x", "c_sum_tot_y", "c_toa_peak", "c_sum_tot_tof",
           "c_cx", "c_cy", "c_ctof")


def check_localmax(m, x, y, toa, tot, wx, wy, wt, P=P, what="", hints=(0, 1024)):
    """Every route of tpx3_localmax_centroid against the plain-definition oracle: the fused tile kernel in its
    paper-literal mode (8192- and 4096-event tiles) and the general kernels (forced)."""
    import torch

    o = oracle.run_localmax(x, y, toa, tot, wx, wy, wt, P)
    n = len(x)
    dev = [to_dev(np.asarray(x, dtype=np.uint16)), to_dev(np.asarray(y, dtype=np.uint16)),
           to_dev(np.asarray(toa, dtype=np.uint64)), to_dev(np.asarray(tot, dtype=np.uint16))]
    for flags, hint in [(0, h) for h in hints] + [(m.FLAG_FORCE_GENERAL, 0)]:
        tag = "%s [flags %d hint %d]" % (what, flags, hint)
        pl = m.plan(m.Config(toa_window_ticks=W, shot_period_ticks=P, max_hits=max(n, 1), flags=flags,
                             max_shot_hits=hint))
        cl = m.Clusters(max(n, 1), pl.device)
        perm, lmax, nh = pl.localmax_centroid(*dev, wx, wy, wt, cl)
        torch.cuda.synchronize()
        st = pl.status()
        assert st["error"] == 0, tag
        nhits = int(nh.cpu().numpy()[0])
        assert nhits == o["n_clusters"], tag
        np.testing.assert_array_equal(perm[:n].cpu().numpy(), o["perm"], err_msg=tag + " perm")
        np.testing.assert_array_equal(lmax[:n].cpu().numpy(), o["lmax"], err_msg=tag + " lmax")
        g = cl.numpy(nhits)
        for k in LM_KEYS:   # integers bit-exact; centroids bitwise fp32 (same int64 sums, IEEE RN divide: R12)
            np.testing.assert_array_equal(g[k], o[k], err_msg=tag + " " + k)
        if n:
            assert st["path"] == 3, tag
        pl.free()
    return o


def test_localmax_paper_example(tpx3):
    # X of Eq. 2, ToT of :134, |D| <= 5 -> hits = pixel 2 and pixel 3
    X = np.array([20, 21, 90, 92, 18]); z = np.zeros(5, dtype=np.int64); T = np.array([50, 200, 300, 25, 100])
    o = check_localmax(tpx3, X, z, z, T, 5, 0, 0, P=0, what="paper example")
    assert (o["c_label"] + 1).tolist() == [2, 3]


@pytest.mark.parametrize("cfg,shots,w3", [(0, 1000, (1, 1, 320)), (1, 400, (1, 1, 320)), (1, 400, (5, 5, 320)),
                                          (2, 150, (2, 2, 40)), (3, 40, (1, 1, 320)), (4, 150, (3, 3, 320)),
                                          (5, 300, (4, 4, 320))])
def test_localmax_configs(tpx3, cfg, shots, w3):
    w = gen.generate(cfg, shots=shots)
    check_localmax(tpx3, w.x, w.y, w.toa, w.tot, *w3, what="cfg%d w=%s" % (cfg, w3), hints=(0, gen.max_shot_hits(cfg)))


def test_localmax_edges(tpx3):
    z16 = np.zeros(0, dtype=np.uint16)
    check_localmax(tpx3, z16, z16, np.zeros(0, dtype=np.uint64), z16, 1, 1, W, what="empty")
    check_localmax(tpx3, [7], [9], [123456789], [55], 1, 1, W, what="single")
    check_localmax(tpx3, np.full(300, 100), np.full(300, 17), np.full(300, 10**9), np.full(300, 3), 0, 0, 0, what="identical")
    check_localmax(tpx3, [100, 100], [100, 100], [P - 1, P], [5, 7], 2, 2, 50, what="shot boundary")
    check_localmax(tpx3, [100, 100], [100, 100], [P - 1, P], [5, 7], 2, 2, 50, P=0, what="P=0")
    rng = np.random.default_rng(5)
    for seed in range(4):
        n = 3000
        x = rng.integers(0, 40, n); y = rng.integers(0, 40, n)
        toa = (rng.integers(0, 3, n) * P + rng.integers(0, 3000, n)).astype(np.uint64)
        tot = rng.integers(1, 5, n)     # many ties
        check_localmax(tpx3, x, y, toa, tot, int(rng.integers(0, 4)), int(rng.integers(0, 4)), int(rng.integers(0, 900)),
                       what="random %d" % seed)
    # large values: ToA near 2^40, ToT up to 65535, window wider than the shot
    n = 2000
    x = rng.integers(0, 256, n); y = rng.integers(0, 256, n)
    toa = ((1 << 40) + rng.integers(0, 2 * P, n)).astype(np.uint64)
    tot = rng.integers(1, 65536, n)
    check_localmax(tpx3, x, y, toa, tot, 255, 255, 10 * P, what="large")


# ------------------------------------------------------------------ ToA unwrapping (NEXT #4)
def test_unwrap_toa(tpx3):
    import torch
    from oracle import preprocess as pp

    m = tpx3
    mod = (1 << 42) // 256
    jump = int(20e9 / 1.5625)
    rng = np.random.default_rng(17)

    def run(raw, modulus, jmp, wraps_in=0, prev=None):
        raw = np.asarray(raw, dtype=np.uint64)
        pl = m.plan(m.Config(max_hits=max(len(raw), 1)))
        out, w = pl.unwrap_toa(to_dev(raw) if len(raw) else torch.empty(0, dtype=torch.uint64, device="cuda"),
                               modulus, jmp, wraps_in=wraps_in, prev_raw=prev)
        torch.cuda.synchronize()
        o, wo = pp.unwrap_toa(raw, modulus, jmp, wraps_in=wraps_in, prev_raw=prev)
        np.testing.assert_array_equal(out[: len(raw)].cpu().numpy(), o)
        assert int(w.cpu().numpy()[0]) == wo
        pl.free()
        return o, wo

    # the paper's edge case by hand, empty and single inputs, carried state
    o, w = run([1000, 1019, 3, 1022, 7, 20], 1024, 600)
    assert o.tolist() == [1000, 1019, 1027, 1022, 1031, 1044] and w == 1
    run([], 1024, 600, wraps_in=5)
    run([17], 1024, 600, wraps_in=2, prev=900)
    run([701, 100, 700, 99, 700], 1024, 600, wraps_in=-1)
    # several tiles and a ragged tail: 3.3 counter periods with reporting disorder, whole and in chunks
    n = 300000 + 1234
    t = np.sort(rng.integers(0, 3 * mod + mod // 3, n).astype(np.int64)) + rng.integers(0, 2000, n) + mod - 5000
    raw = (t % mod).astype(np.uint64)
    w0 = int(t[0] // mod)
    o, w = run(raw, mod, jump, wraps_in=w0)
    assert np.array_equal(o.astype(np.int64), t)
    prev, wc = None, w0
    for a, b in [(0, 4096), (4096, 4097), (4097, 100000), (100000, n)]:
        oc, wc = run(raw[a:b], mod, jump, wraps_in=wc, prev=prev)
        assert np.array_equal(oc, o[a:b])
        prev = int(raw[b - 1])
    assert wc == w
    # adversarial: every event jumps (alternating +/-), counter swings negative and back
    alt = np.where(np.arange(50000) % 2 == 0, 5, 1000).astype(np.uint64)
    run(alt, 1024, 600)
    run(rng.integers(0, 1024, 70000), 1024, 300)
    # 1.3e7 events (3 000 blocks: the block-sum scan runs several rounds per thread): generated truth over 5.4 counter
    # periods (the sequential oracle is a Python loop; the true times are what it must give back)
    n = (1 << 23) + (1 << 22) + 54321
    mod2 = 1 << 30
    t = np.sort(rng.integers(0, 5 * mod2 + mod2 // 3, n).astype(np.int64)) + rng.integers(0, 3000, n) + mod2 - 7000
    w0 = int(t[0] // mod2)
    pl = m.plan(m.Config(max_hits=n))
    out, w = pl.unwrap_toa(to_dev((t % mod2).astype(np.uint64)), mod2, mod2 // 2, wraps_in=w0)
    torch.cuda.synchronize()
    assert np.array_equal(out[:n].cpu().numpy().astype(np.int64), t)
    assert int(w.cpu().numpy()[0]) == int(t[-1] // mod2) and int(w.cpu().numpy()[0]) >= 5
    pl.free()


# ------------------------------------------------------------------ preprocessing (NEXT #3)
def test_preprocess(tpx3):
    import torch
    from oracle import preprocess as pp

    m = tpx3

    def run(x, y, toa, tot, trig, cut, table, shot_base=0):
        x = np.asarray(x, dtype=np.uint16); y = np.asarray(y, dtype=np.uint16)
        toa = np.asarray(toa, dtype=np.uint64); tot = np.asarray(tot, dtype=np.uint16)
        trig = np.asarray(trig, dtype=np.uint64)
        n = len(x)
        pl = m.plan(m.Config(max_hits=max(n, 1), shot_period_ticks=P))
        dv = lambda a, dt: to_dev(a) if len(a) else torch.empty(0, dtype=dt, device="cuda")  # noqa: E731
        tb = None if table is None else to_dev(np.asarray(table, dtype=np.int32))
        xo, yo, to, oo, io, no = pl.preprocess(dv(x, torch.uint16), dv(y, torch.uint16), dv(toa, torch.uint64),
                                               dv(tot, torch.uint16), dv(trig, torch.uint64), cut, tb, shot_base)
        torch.cuda.synchronize()
        k = int(no.cpu().numpy()[0])
        ex, ey, et, eo, ei = pp.preprocess(x, y, toa, tot, trig, cut, [] if table is None else table, P, shot_base)
        assert k == len(ei)
        np.testing.assert_array_equal(xo[:k].cpu().numpy(), ex)
        np.testing.assert_array_equal(yo[:k].cpu().numpy(), ey)
        np.testing.assert_array_equal(to[:k].cpu().numpy(), et)
        np.testing.assert_array_equal(oo[:k].cpu().numpy(), eo)
        np.testing.assert_array_equal(io[:k].cpu().numpy().astype(np.int64), ei)
        pl.free()
        return k, (xo[:k], yo[:k], to[:k], oo[:k])

    # hand example of the oracle pins (cut edge, clamp, ToT beyond the table, out-of-order event, no trigger yet)
    k, _ = run(list(range(9)), [2 * v for v in range(9)], [900, 1000, 1300, 1301, 2004, 2999, 3100, 2150, 3003],
               [1, 1, 2, 2, 0, 3, 9, 1, 1], [1000, 2000, 3000], 300, [9, 5, 2, 0], shot_base=7)
    assert k == 6
    # degenerate inputs: nothing in, no triggers (everything dropped), no table
    run([], [], [], [], [5], 10, [1])
    assert run([1, 2], [3, 4], [100, 200], [5, 6], [], 10, [1])[0] == 0
    assert run([1, 2], [3, 4], [100, 200], [5, 6], [50], 1000, None)[0] == 2
    # a config-2 stream moved onto irregular triggers, with timewalk and dark counts: several tiles, ragged tail
    w = gen.generate(2, shots=400)
    rng = np.random.default_rng(9)
    trig = np.cumsum(rng.integers(P - 2000, P + 2000, w.shots)).astype(np.int64) + 12345
    table = pp.timewalk_table(800.0, 4.0, 0.0, 1.0, 1024)
    assert np.array_equal(table, m.timewalk_table(800.0, 4.0, 0.0, 1.0, 1024))
    shot = (w.toa // np.uint64(P)).astype(np.int64)
    tof = (w.toa % np.uint64(P)).astype(np.int64)
    raw = trig[shot] + tof + table[np.minimum(w.tot, 1023)]
    cut = int(tof.max() + table.max())
    nd = w.n // 10
    draw = trig[rng.integers(0, w.shots, nd)] + rng.integers(cut + 1, P - 3000, nd)
    allx = np.concatenate([w.x, rng.integers(0, 256, nd).astype(np.uint16)])
    ally = np.concatenate([w.y, rng.integers(0, 256, nd).astype(np.uint16)])
    alltot = np.concatenate([w.tot, rng.integers(1, 30, nd).astype(np.uint16)])
    allraw = np.concatenate([raw, draw]).astype(np.uint64)
    order = np.argsort(allraw, kind="stable")
    k, dev = run(allx[order], ally[order], allraw[order], alltot[order], trig, cut, table)
    assert k == w.n
    # and the preprocessed stream, clustered on the device, gives the hits of the original stream (the corrected
    # stream is ordered by raw time, i.e. out of ToA order inside a shot: the sort runs)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    pl = m.plan(m.Config(max_hits=k, toa_window_ticks=W, shot_period_ticks=P, max_shot_hits=gen.max_shot_hits(2)))
    cl = m.Clusters(k, pl.device)
    perm, label, nc = pl.cluster_centroid(*[t.contiguous() for t in dev], cl)
    torch.cuda.synchronize()
    assert pl.status()["error"] == 0
    ncl = int(nc.cpu().numpy()[0])
    assert ncl == o["n_clusters"]
    g = cl.numpy(ncl)
    # events of equal ToA are delivered in a different order here than in w, so the stable sort and with it the
    # listing order of hits inside a shot may differ: compare the hits as a set of rows
    keys = ("c_shot", "c_toa_peak", "c_sum_tot_x", "c_sum_tot_y", "c_sum_tot", "c_size", "c_sum_tot_tof")

    def rows(d):
        r = np.stack([d[k2].astype(np.int64) for k2 in keys] + [d["c_cx"].view(np.int32).astype(np.int64),
                     d["c_cy"].view(np.int32).astype(np.int64), d["c_ctof"].view(np.int32).astype(np.int64)], axis=1)
        return r[np.lexsort(r.T[::-1])]

    np.testing.assert_array_equal(rows(g), rows(o))
    pl.free()


@pytest.mark.parametrize("side,per_shot,hint,Wr", [(6, 900, 1024, 320), (12, 3000, 4096, 40), (3, 400, 512, 5),
                                                   (40, 2000, 2048, 2), (16, 1000, 1024, 100000)])
def test_fused_dense_repeated_addresses(tpx3, side, per_shot, hint, Wr):
    """Shot-contiguous streams whose events crowd a few pixels: many events per (shot, pixel), overflowing
    hash buckets, more deferred links than the list holds — the fused kernel's rare paths — in all three
    tile variants, delivered out of order inside each shot."""
    rng = np.random.default_rng(side * 1000 + per_shot)
    shots = 60
    n = shots * per_shot
    shot = np.repeat(np.arange(shots), per_shot)
    x = rng.integers(100, 100 + side, n); y = rng.integers(250 - side, 256, n) % 256
    tof = rng.integers(0, 3000, n)
    toa = (shot * P + tof).astype(np.uint64)
    tot = rng.integers(1, 1024, n)
    res, _ = check(tpx3, x, y, toa, tot, W=Wr, modes=("fused",), max_shot_hits=hint, what="dense %d" % side)
    assert res["status"]["path"] == 1


def test_localmax_capacity_and_args(tpx3):
    import torch

    m = tpx3
    w = gen.generate(1, shots=200)
    o = oracle.run_localmax(w.x, w.y, w.toa, w.tot, 1, 1, W, P)
    dev = [to_dev(a) for a in (w.x, w.y, w.toa, w.tot)]
    for flags in (0, m.FLAG_FORCE_GENERAL):
        pl = m.plan(m.Config(max_hits=w.n, shot_period_ticks=P, flags=flags))
        cap = o["n_clusters"] // 2
        cl = m.Clusters(cap, pl.device)
        perm, lmax, nh = pl.localmax_centroid(*dev, 1, 1, W, cl)
        torch.cuda.synchronize()
        st = pl.status()
        assert st["error"] == m.ERR_CAPACITY                       # reported, not silently truncated
        assert int(nh.cpu().numpy()[0]) == o["n_clusters"]           # the true count
        g = cl.numpy(cap)
        for k in LM_KEYS:
            np.testing.assert_array_equal(g[k], o[k][:cap], err_msg=k)   # the first `cap` rows are valid
        np.testing.assert_array_equal(lmax[: w.n].cpu().numpy(), o["lmax"])
        pl.free()
    pl = m.plan(m.Config(max_hits=10))
    with pytest.raises(m.Tpx3Error):
        pl.localmax_centroid(*dev, 1, 1, W, m.Clusters(16, pl.device))  # n > max_hits
    pl.free()


@pytest.mark.parametrize("per_shot,path", [(700, 1), (1500, 1), (3000, 1), (6000, 1), (9000, 2)])
def test_no_hint_ladder(tpx3, per_shot, path):
    """max_shot_hits = 0: windows of 2048, 4096 and 8192 events are tried in turn on the device (a failed rung
    stops in its first wave and the next one is launched from k_fallback_dispatch), then the general path."""
    rng = np.random.default_rng(per_shot)
    shots = 25
    n = shots * per_shot
    x = rng.integers(0, 256, n); y = rng.integers(0, 256, n)
    toa = (np.repeat(np.arange(shots), per_shot) * P + np.sort(rng.integers(0, 60000, (shots, per_shot)), axis=1).ravel()
           ).astype(np.uint64)
    tot = rng.integers(1, 1024, n)
    res, _ = check(tpx3, x, y, toa, tot, modes=("fused",), max_shot_hits=0, what="ladder %d" % per_shot)
    assert res["status"]["path"] == path
    check_localmax(tpx3, x, y, toa, tot, 1, 1, 200, what="ladder lm %d" % per_shot, hints=(0,))


def test_full_size_localmax_cfg1(tpx3):
    """BASELINE.json configs[1] in full through the paper-literal mode (the bench configuration of
    `bench.py --mode localmax`): sampled shot windows element by element, invariants on the whole output."""
    import torch

    m = tpx3
    w = gen.generate(1)
    n = w.n
    wx, wy, wt = 2, 2, 320
    pl = m.plan(m.Config(max_hits=n, toa_window_ticks=W, shot_period_ticks=P, max_shot_hits=gen.max_shot_hits(1)))
    dev = [to_dev(a) for a in (w.x, w.y, w.toa, w.tot)]
    cl = m.Clusters(max(n // 2, 1024), pl.device)
    perm, lmax, nh = pl.localmax_centroid(*dev, wx, wy, wt, cl)
    torch.cuda.synchronize()
    st = pl.status()
    assert st["error"] == 0 and st["path"] == 3, st
    nhits = int(nh.cpu().numpy()[0])
    perm, lmax = perm[:n].cpu().numpy(), lmax[:n].cpu().numpy()
    c = cl.numpy(nhits)
    pl.free()
    k = np.arange(n, dtype=np.uint32)
    assert np.all((lmax == k) | (lmax == 0xFFFFFFFF))
    assert np.array_equal(np.flatnonzero(lmax == k).astype(np.uint32), c["c_label"])
    assert np.array_equal(perm, k)                                    # cfg1 is delivered in ToA order
    assert np.all(c["c_size"] >= 1) and np.all(c["c_size"] <= 25 * 4)  # a 5 x 5 box, a few repeated addresses
    assert np.array_equal(c["c_toa_peak"], w.toa[c["c_label"]])
    off = w.shot_offsets
    for s0, s1 in _windows(w.shots, 300, 6):
        a, b = int(off[s0]), int(off[s1])
        s = w.slice_shots(s0, s1)
        o = oracle.run_localmax(s.x, s.y, s.toa, s.tot, wx, wy, wt, P)
        what = "shots [%d, %d)" % (s0, s1)
        exp = np.where(o["lmax"] == 0xFFFFFFFF, np.uint32(0xFFFFFFFF), o["lmax"] + np.uint32(a))
        np.testing.assert_array_equal(lmax[a:b], exp, err_msg=what + " lmax")
        i0, i1 = np.searchsorted(c["c_label"], [a, b])
        assert i1 - i0 == o["n_clusters"], what
        np.testing.assert_array_equal(c["c_label"][i0:i1], o["c_label"] + np.uint32(a), err_msg=what)
        for key in LM_KEYS[1:]:
            np.testing.assert_array_equal(c[key][i0:i1], o[key], err_msg=what + " " + key)


def test_time_cluster_hint_never_changes_results(tpx3):
    """One plan (one workspace) serving calls of different character: the hint the fused kernel leaves in the
    workspace (skip the time-cluster check after a call with hardly any tight tile) only selects between two
    exact code paths, so every call must match the oracle whatever came before it."""
    import torch

    m = tpx3
    loose = gen.generate(3, shots=300)      # noise hits chain the time clusters: no tight tiles
    multi = gen.generate(2, shots=700)      # separated mass peaks: tight tiles with several clusters
    narrow = gen.generate(1, shots=1500)    # all times of flight within W
    nmax = max(w.n for w in (loose, multi, narrow))
    pl = m.plan(m.Config(max_hits=nmax, toa_window_ticks=W, shot_period_ticks=P, max_shot_hits=gen.max_shot_hits(3)))
    cl = m.Clusters(nmax, pl.device)
    for name, w in [("loose", loose), ("loose again", loose), ("multi after loose", multi), ("multi again", multi),
                    ("narrow", narrow), ("loose after narrow", loose), ("multi", multi)] + [("multi x%d" % i, multi) for i in range(16)]:
        o = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
        dev = [to_dev(a) for a in (w.x, w.y, w.toa, w.tot)]
        perm, label, nc = pl.cluster_centroid(*dev, cl)
        torch.cuda.synchronize()
        st = pl.status()
        assert st["error"] == 0 and st["path"] == 1, name
        ncl = int(nc.cpu().numpy()[0])
        g = {"perm": perm[: w.n].cpu().numpy(), "label": label[: w.n].cpu().numpy(), "n_clusters": ncl}
        g.update(cl.numpy(ncl))
        assert_parity(g, o, name)
    pl.free()


# ------------------------------------------------------------------ chunked stream, cuts not shot-aligned (NEXT #3)
from oracle import preprocess as opp  # noqa: E402

_ROW_KEYS = ("c_label", "c_size", "c_shot", "c_sum_tot", "c_sum_tot_x", "c_sum_tot_y", "c_sum_tot_tof",
             "c_toa_peak", "c_cx", "c_cy", "c_ctof")


def _disorder(toa):
    t = np.asarray(toa).astype(np.int64)
    return int(np.max(np.maximum.accumulate(t) - t)) if len(t) else 0


def run_stream(m, w, sizes, D, max_carry, max_shot_hits=0, cap=None, final_empty=False, flags=0):
    """Push w in chunks of the given sizes through tpx3_stream_push; returns the concatenated hit rows,
    the per-push info and the StreamModel's per-push (n_emitted, n_carry, n_late) for the same chunks."""
    import torch

    max_chunk = max(max(sizes), 1)
    pl = m.plan(m.Config(toa_window_ticks=W, shot_period_ticks=P, max_hits=max_chunk + max_carry,
                         max_shot_hits=max_shot_hits, flags=flags))
    s = pl.stream_open(max_chunk, max_carry, D)
    cl = m.Clusters(cap or (max_chunk + max_carry), pl.device)
    dx, dy, dt, do = to_dev(w.x), to_dev(w.y), to_dev(w.toa), to_dev(w.tot)
    model = opp.StreamModel(P, D)
    rows = {k: [] for k in _ROW_KEYS}
    infos, want = [], []
    i = 0
    pushes = [(sz, False) for sz in sizes]
    if final_empty:
        pushes.append((0, True))
    else:
        pushes[-1] = (pushes[-1][0], True)
    for sz, fin in pushes:
        nh, info = s.push(dx[i:i + sz], dy[i:i + sz], dt[i:i + sz], do[i:i + sz], cl, final=fin)
        e = model.push(w.x[i:i + sz], w.y[i:i + sz], w.toa[i:i + sz], w.tot[i:i + sz], final=fin)
        i += sz
        torch.cuda.synchronize()
        assert pl.status()["error"] == 0
        k = int(nh.cpu().numpy()[0])
        got = cl.numpy(k)
        for key in _ROW_KEYS:
            rows[key].append(got[key].copy())
        infos.append(info)
        want.append((len(e["x"]), e["n_carry"], e["n_late"], e["label_base"]))
    s.close()
    pl.free()
    return {k: np.concatenate(v) for k, v in rows.items()}, infos, want


def _sizes(n, chunk):
    return [chunk] * (n // chunk) + ([n % chunk] if n % chunk else [])


DEVICE_TMAX_TAIL = 65536   # tpx3.h: a push takes the running maximum over the last 65536 events of its chunk


def _check_push_properties(infos, toa, sizes, D, honest=True):
    """What a push emits is not part of the definition (oracle/preprocess.py StreamModel: any lower bound of the
    running maximum is safe; the device samples the chunk's tail) — these properties are: nothing is lost or
    emitted twice, a shot goes out in one piece and only when complete, labels continue the batch numbering,
    and with an honest disorder bound D nothing is late and no shot goes out before it can be complete."""
    shot = (np.asarray(toa) // np.uint64(P)).astype(np.int64)
    n = len(shot)
    consumed = emitted = late = 0
    s_prev = 0
    for info, sz in zip(infos, sizes):
        consumed += sz
        assert info["label_base"] == emitted
        emitted += info["n_emitted"]
        late += info["n_late"]
        assert info["late_total"] == late
        assert emitted + late + info["n_carry"] == consumed          # every event is emitted, late or carried
        s_now = info["shots_emitted"]
        assert s_now >= s_prev
        s_prev = s_now
        seen = shot[:consumed]
        if honest:
            assert info["n_late"] == 0
            if consumed == n and info["n_carry"] == 0:                # the final push emits what is left
                assert emitted == n
                continue
            assert emitted == int(np.count_nonzero(seen < s_now))     # exactly the shots below s_now went out ...
            assert not np.any(shot[consumed:] < s_now)                # ... and they were complete
            if consumed < n or info["n_carry"]:
                t_seen = int(np.asarray(toa[:consumed]).max()) if consumed else 0
                assert s_now <= max(t_seen - D, 0) // P or s_now == 0 or consumed == n
    assert consumed == n and infos[-1]["n_carry"] == 0 and emitted + late == n


@pytest.mark.parametrize("cfg,shots,chunk", [(0, 1000, 997), (0, 300, 64), (1, 60, 100003), (1, 60, 1 << 20),
                                             (2, 8, 250007), (3, 40, 30011), (4, 1200, 65536), (4, 1200, 300001),
                                             (4, 1200, 1 << 22)])
def test_stream_equals_batch(tpx3, cfg, shots, chunk):
    """Chunks cut anywhere (inside shots and hits): the rows of all pushes, in order, are the oracle's rows for
    the whole stream, every column bit for bit; per push the emitted / carried / late counts are the model's."""
    w = gen.generate(cfg, shots=shots)
    D = _disorder(w.toa)
    assert (D > 0) == (cfg == 4)
    per_shot = int(np.bincount((w.toa // np.uint64(P)).astype(np.int64) - int(w.toa.min() // P)).max())
    rows, infos, want = run_stream(tpx3, w, _sizes(w.n, chunk), D, max_carry=4 * per_shot + 16)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P, threads=0)
    for k in _ROW_KEYS:
        np.testing.assert_array_equal(rows[k], o[k], err_msg=k)
    sizes = _sizes(w.n, chunk)
    _check_push_properties(infos, w.toa, sizes, D)
    if chunk <= DEVICE_TMAX_TAIL or D == 0:   # the device's tail sample holds the true maximum: the model's very pushes
        for info, (ne, nk, nl, lb) in zip(infos, want):
            assert (info["n_emitted"], info["n_carry"], info["n_late"], info["label_base"]) == (ne, nk, nl, lb)
    assert infos[-1]["late_total"] == 0 and infos[-1]["n_carry"] == 0
    if chunk < w.n:
        assert max(i["n_carry"] for i in infos) > 0       # the cuts were not shot-aligned


@pytest.mark.parametrize("cfg,shots,chunk,hint", [(1, 60, 7001, 600), (4, 200, 50021, 1500), (3, 12, 9973, 512)])
def test_stream_on_the_general_route(tpx3, cfg, shots, chunk, hint):
    """Stream pushes whose clustering takes the general route, sized and enqueued from the device (the emit count is
    device state): forced by the plan's flag (global sort, then the tile kernel through perm), and - last case,
    2100-event shots against 2048-event windows - after the tile kernel gave up."""
    w = gen.generate(cfg, shots=shots)
    D = _disorder(w.toa)
    per_shot = int(np.bincount((w.toa // np.uint64(P)).astype(np.int64) - int(w.toa.min() // P)).max())
    sizes = _sizes(w.n, chunk)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P, threads=0)
    for flags in ((tpx3.FLAG_FORCE_GENERAL, 0) if cfg != 3 else (0,)):
        rows, infos, _ = run_stream(tpx3, w, sizes, D, max_carry=4 * per_shot + 16, max_shot_hits=hint, flags=flags)
        for k in _ROW_KEYS:
            np.testing.assert_array_equal(rows[k], o[k], err_msg="%s flags %d" % (k, flags))
        _check_push_properties(infos, w.toa, sizes, D)


def test_shot_period_beyond_the_tile_key(tpx3):
    """P > 2^24 ticks: the time of flight does not fit the tile kernel's 32-bit key, the plan has no tile kernel and
    every call runs the slab-hash kernels: batch call, split calls, and stream pushes (device-sized, labels offset)."""
    import torch

    P2 = (1 << 25) + 12345
    w = gen.generate(0, shots=400)
    shot = (w.toa // np.uint64(P)).astype(np.uint64)
    toa = shot * np.uint64(P2) + (w.toa % np.uint64(P)) * np.uint64(37)          # ToF spread over 2.3e6 ticks
    Wr = 320 * 37
    o = oracle.run(w.x, w.y, toa, w.tot, Wr, P2, threads=0)
    res, _ = check(tpx3, w.x, w.y, toa, w.tot, W=Wr, P=P2, modes=("split", "fused"), what="P > 2^24")
    assert res["status"]["path"] == 2
    chunk, carry = 5003, 2048
    pl = tpx3.plan(tpx3.Config(toa_window_ticks=Wr, shot_period_ticks=P2, max_hits=chunk + carry))
    s = pl.stream_open(chunk, carry, 0)
    cl = tpx3.Clusters(chunk + carry, pl.device)
    dev = [to_dev(a) for a in (w.x, w.y, toa, w.tot)]
    rows = {k: [] for k in _ROW_KEYS}
    sizes = _sizes(w.n, chunk)
    i = 0
    for j, sz in enumerate(sizes):
        nh, info = s.push(*(d[i:i + sz] for d in dev), cl, final=(j == len(sizes) - 1))
        i += sz
        torch.cuda.synchronize()
        assert pl.status()["error"] == 0
        got = cl.numpy(int(nh.cpu().numpy()[0]))
        for k in _ROW_KEYS:
            rows[k].append(got[k].copy())
    s.close()
    pl.free()
    for k in _ROW_KEYS:
        np.testing.assert_array_equal(np.concatenate(rows[k]), o[k], err_msg=k)


def test_stream_random_chunks_and_empty_pushes(tpx3):
    w = gen.generate(1, shots=40)
    rng = np.random.default_rng(11)
    sizes = []
    while sum(sizes) < w.n:
        sizes.append(int(min(rng.choice([0, 1, 17, 5000, 70000, 200000]), w.n - sum(sizes))))
    rows, infos, want = run_stream(tpx3, w, sizes, 0, max_carry=200000, final_empty=True)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P, threads=0)
    for k in _ROW_KEYS:
        np.testing.assert_array_equal(rows[k], o[k], err_msg=k)
    _check_push_properties(infos, w.toa, sizes + [0], 0)
    # a stream in ToA order: the chunk's largest ToA is its last event, so the device's tail sample is exact
    assert [(i["n_emitted"], i["n_carry"], i["n_late"]) for i in infos] == [t[:3] for t in want]


@pytest.mark.parametrize("cfg,shots,chunk,hint", [(1, None, 4000037, 1024), (4, 24000, (1 << 22) + 12345, 1536)])
def test_stream_full_size(tpx3, cfg, shots, chunk, hint):
    """configs[1] whole (3.6e7 hits) and a 1.7e7-hit stretch of configs[4], pushed in chunks of about 2^22
    events cut anywhere: all rows against the oracle's for the whole stream."""
    w = gen.generate(cfg, shots=shots) if shots else gen.generate(cfg)
    D = _disorder(w.toa)
    import torch

    pl = tpx3.plan(tpx3.Config(toa_window_ticks=W, shot_period_ticks=P, max_hits=chunk + (1 << 18), max_shot_hits=hint))
    s = pl.stream_open(chunk, 1 << 18, D)
    cl = tpx3.Clusters(chunk + (1 << 18), pl.device)
    dx, dy, dt, do = to_dev(w.x), to_dev(w.y), to_dev(w.toa), to_dev(w.tot)
    rows = {k: [] for k in _ROW_KEYS}
    sizes = _sizes(w.n, chunk)
    i = emitted = 0
    for j, sz in enumerate(sizes):
        nh, info = s.push(dx[i:i + sz], dy[i:i + sz], dt[i:i + sz], do[i:i + sz], cl, final=(j == len(sizes) - 1))
        i += sz
        torch.cuda.synchronize()
        st = pl.status()
        assert st["error"] == 0 and st["path"] == 1 and info["n_late"] == 0 and info["label_base"] == emitted
        emitted += info["n_emitted"]
        got = cl.numpy(int(nh.cpu().numpy()[0]))
        for k in _ROW_KEYS:
            rows[k].append(got[k].copy())
    assert emitted == w.n
    s.close()
    pl.free()
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P, threads=0)
    for k in _ROW_KEYS:
        np.testing.assert_array_equal(np.concatenate(rows[k]), o[k], err_msg=k)


def test_stream_late_events_are_dropped_and_counted(tpx3):
    """A stream that breaks its promise (D = 0, but the pixels of some shots arrive three shots later): those are
    late. The rows are then the oracle's rows of what the model emitted (not the batch result), and the counts
    match the model."""
    import types

    w0 = gen.generate(0, shots=400)
    shot = (w0.toa // np.uint64(P)).astype(np.int64)
    shot -= shot.min()
    moved = (shot % 50 == 7) & (np.arange(w0.n) % 3 == 0)
    key = np.where(moved, shot + 3, shot) * 4 + moved           # stable: behind the events of shot + 3
    order = np.argsort(key, kind="stable")
    w = types.SimpleNamespace(x=w0.x[order], y=w0.y[order], toa=w0.toa[order], tot=w0.tot[order], n=w0.n)
    sizes = _sizes(w.n, 1013)
    rows, infos, want = run_stream(tpx3, w, sizes, 0, max_carry=1 << 20)
    assert infos[-1]["late_total"] > 0
    assert [(i["n_emitted"], i["n_carry"], i["n_late"]) for i in infos] == [t[:3] for t in want]
    model = opp.StreamModel(P, 0)
    i, exp = 0, {k: [] for k in _ROW_KEYS}
    for j, sz in enumerate(sizes):
        e = model.push(w.x[i:i + sz], w.y[i:i + sz], w.toa[i:i + sz], w.tot[i:i + sz], final=(j == len(sizes) - 1))
        i += sz
        r = oracle.run(e["x"], e["y"], e["toa"], e["tot"], W, P, threads=0)
        for k in _ROW_KEYS:
            exp[k].append(r[k] + np.uint32(e["label_base"]) if k == "c_label" else r[k])
    for k in _ROW_KEYS:
        np.testing.assert_array_equal(rows[k], np.concatenate(exp[k]), err_msg=k)


def test_stream_carry_overflow_is_an_error(tpx3):
    w = gen.generate(1, shots=50)
    with pytest.raises(tpx3.Tpx3Error) as ei:
        run_stream(tpx3, w, _sizes(w.n, 4000), 0, max_carry=8)
    assert ei.value.code == tpx3.ERR_CAPACITY


def test_stream_rejects_bad_arguments(tpx3):
    pl = tpx3.plan(tpx3.Config(toa_window_ticks=W, shot_period_ticks=P, max_hits=1000))
    with pytest.raises(tpx3.Tpx3Error):
        pl.stream_open(900, 200, 0)               # max_chunk + max_carry > max_hits
    pl.free()
    pl0 = tpx3.plan(tpx3.Config(toa_window_ticks=W, shot_period_ticks=0, max_hits=1000))
    with pytest.raises(tpx3.Tpx3Error):
        pl0.stream_open(500, 200, 0)              # no shot period: nothing is ever complete
    pl0.free()


def test_stream_pushes_without_info_do_not_wait_and_give_the_same_rows(tpx3):
    """info = NULL: the push only enqueues (the emit count sizes the clustering launch on the device). The rows of
    all pushes — read back once, at the end, from one table per push — are the batch oracle's; a carry overflow is
    reported by the status word."""
    import torch

    w = gen.generate(4, shots=900)
    D = _disorder(w.toa)
    chunk, carry = 100003, 8192
    pl = tpx3.plan(tpx3.Config(toa_window_ticks=W, shot_period_ticks=P, max_hits=chunk + carry, max_shot_hits=1500))
    s = pl.stream_open(chunk, carry, D)
    dev = [to_dev(a) for a in (w.x, w.y, w.toa, w.tot)]
    sizes = _sizes(w.n, chunk)
    tabs = [tpx3.Clusters(chunk + carry, pl.device) for _ in sizes]
    counts = [torch.zeros(1, dtype=torch.uint32, device=pl.device) for _ in sizes]
    i = 0
    for j, sz in enumerate(sizes):
        _, info = s.push(*(d[i:i + sz] for d in dev), tabs[j], final=(j == len(sizes) - 1), n_hits=counts[j],
                         want_info=False)
        assert info is None
        i += sz
    torch.cuda.synchronize()
    assert pl.status()["error"] == 0
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P, threads=0)
    rows = {k: np.concatenate([t.numpy(int(c.cpu().numpy()[0]))[k] for t, c in zip(tabs, counts)]) for k in _ROW_KEYS}
    for k in _ROW_KEYS:
        np.testing.assert_array_equal(rows[k], o[k], err_msg=k)
    s.close()
    # overflow: a carry capacity below one shot
    s = pl.stream_open(chunk, 64, D)
    s.push(*(d[:chunk] for d in dev), tabs[0], n_hits=counts[0], want_info=False)
    torch.cuda.synchronize()
    assert pl.status()["error"] == tpx3.ERR_CAPACITY
    s.push(*(d[chunk:2 * chunk] for d in dev), tabs[0], n_hits=counts[0], want_info=False)   # the stream stays dead
    torch.cuda.synchronize()
    assert pl.status()["error"] == tpx3.ERR_CAPACITY and int(counts[0].cpu().numpy()[0]) == 0
    with pytest.raises(tpx3.Tpx3Error):
        s.push(*(d[:chunk] for d in dev), tabs[0], n_hits=counts[0])       # with info: the call itself reports it
    s.close()
    pl.free()


def test_stream_takes_nothing_after_the_final_push(tpx3):
    """tpx3.h: final "ends the stream". A later push is refused (it would cluster shots a second time)."""
    w = gen.generate(0, shots=30)
    pl = tpx3.plan(tpx3.Config(toa_window_ticks=W, shot_period_ticks=P, max_hits=w.n + 1000))
    s = pl.stream_open(w.n, 1000, 0)
    cl = tpx3.Clusters(w.n, pl.device)
    dev = [to_dev(a) for a in (w.x, w.y, w.toa, w.tot)]
    _, info = s.push(*dev, cl, final=True)
    assert info["n_emitted"] == w.n
    with pytest.raises(tpx3.Tpx3Error) as e:
        s.push(*dev, cl, final=False)
    assert e.value.code == tpx3.ERR_INVALID_ARG
    s.close()
    pl.free()


def _raw_stream(cfg, shots, seed, dark_every=10, shuffle=False):
    """A config stream moved onto irregular trigger times with timewalk added and dark counts beyond the cut,
    in raw-time order (or as delivered by config 4: locally shuffled). Returns the raw arrays and the call's
    parameters; the original stream comes back from oracle.preprocess (tests/test_oracle_pins.py pins that)."""
    from oracle import preprocess as pp

    w = gen.generate(cfg, shots=shots)
    rng = np.random.default_rng(seed)
    trig = np.cumsum(rng.integers(P - 2000, P + 2000, w.shots)).astype(np.int64) + 12345
    table = pp.timewalk_table(800.0, 4.0, 0.0, 1.0, 1024)
    shot = (w.toa // np.uint64(P)).astype(np.int64)
    shot -= shot.min()
    tof = (w.toa % np.uint64(P)).astype(np.int64)
    raw = trig[shot] + tof + table[np.minimum(w.tot, 1023)]
    cut = int(tof.max() + table.max())
    nd = w.n // dark_every if dark_every else 0
    dshot = rng.integers(0, w.shots, nd)
    draw = trig[dshot] + rng.integers(cut + 1, P - 3000, nd)
    allx = np.concatenate([w.x, rng.integers(0, 256, nd).astype(np.uint16)])
    ally = np.concatenate([w.y, rng.integers(0, 256, nd).astype(np.uint16)])
    alltot = np.concatenate([w.tot, rng.integers(1, 30, nd).astype(np.uint16)])
    allraw = np.concatenate([raw, draw]).astype(np.uint64)
    if shuffle:   # keep config 4's delivery order inside a shot; dark counts go behind their shot's events
        order = np.argsort(np.concatenate([shot, dshot]), kind="stable")
    else:
        order = np.argsort(allraw, kind="stable")
    per_shot = int(np.bincount(np.concatenate([shot, dshot])).max())
    return allx[order], ally[order], allraw[order], alltot[order], trig.astype(np.uint64), cut, table, per_shot


@pytest.mark.parametrize("cfg,shots,dark,shuffle", [(2, 300, 10, False), (1, 1500, 0, False), (4, 300, 7, True),
                                                    (0, 900, 3, False), (3, 60, 10, False)])
def test_preprocess_fused_into_the_clustering_call(tpx3, cfg, shots, dark, shuffle):
    """tpx3_preprocess_cluster_centroid (SURVEY 8f NEXT #3 as worded): the oracle's preprocessing followed by the
    oracle's clustering, element by element — perm (as input positions), labels, every hit column — and the
    two-call device route gives the same."""
    import torch
    from oracle import preprocess as pp

    x, y, raw, tot, trig, cut, table, per_shot = _raw_stream(cfg, shots, 100 + cfg, dark, shuffle)
    n = len(x)
    ex, ey, et, eo, ei = pp.preprocess(x, y, raw, tot, trig, cut, table, P, 5)
    o = oracle.run(ex, ey, et, eo, W, P)
    pl = tpx3.plan(tpx3.Config(max_hits=n, toa_window_ticks=W, shot_period_ticks=P, max_shot_hits=per_shot))
    dev = [to_dev(a) for a in (x, y, raw, tot)]
    dtrig, dtab = to_dev(trig), to_dev(np.asarray(table, dtype=np.int32))
    cl = tpx3.Clusters(n, pl.device)
    perm, label, nc, nk = pl.preprocess_cluster_centroid(*dev, dtrig, cut, dtab, 5, cl)
    torch.cuda.synchronize()
    st = pl.status()
    assert st["error"] == 0 and st["path"] == 1, st
    k = int(nk.cpu().numpy()[0])
    assert k == len(ei)
    ncl = int(nc.cpu().numpy()[0])
    g = {"perm": perm[:k].cpu().numpy(), "label": label[:k].cpu().numpy(), "n_clusters": ncl}
    g.update(cl.numpy(ncl))
    want = dict(o)
    want["perm"] = ei[o["perm"]].astype(np.uint32)          # input positions
    assert_parity(g, want, "fused preprocessing cfg%d" % cfg)
    # the two calls on the device: same hits
    xo, yo, to, oo, io, no = pl.preprocess(*dev, dtrig, cut, dtab, 5)
    torch.cuda.synchronize()
    k2 = int(no.cpu().numpy()[0])
    assert k2 == k
    cl2 = tpx3.Clusters(n, pl.device)
    perm2, label2, nc2 = pl.cluster_centroid(xo[:k].contiguous(), yo[:k].contiguous(), to[:k].contiguous(),
                                             oo[:k].contiguous(), cl2)
    torch.cuda.synchronize()
    assert int(nc2.cpu().numpy()[0]) == ncl
    np.testing.assert_array_equal(io[:k].cpu().numpy()[perm2[:k].cpu().numpy()], g["perm"])
    np.testing.assert_array_equal(label2[:k].cpu().numpy(), g["label"])
    g2 = cl2.numpy(ncl)
    for key in LM_KEYS:
        np.testing.assert_array_equal(g2[key], g[key], err_msg=key)
    pl.free()


def test_preprocess_fused_edge_cases(tpx3):
    import torch
    from oracle import preprocess as pp

    def run(x, y, toa, tot, trig, cut, table, shot_base, hint=64):
        x = np.asarray(x, dtype=np.uint16); y = np.asarray(y, dtype=np.uint16)
        toa = np.asarray(toa, dtype=np.uint64); tot = np.asarray(tot, dtype=np.uint16)
        trig = np.asarray(trig, dtype=np.uint64)
        n = len(x)
        pl = tpx3.plan(tpx3.Config(max_hits=max(n, 1), toa_window_ticks=W, shot_period_ticks=P, max_shot_hits=hint))
        dv = lambda a, dt: to_dev(a) if len(a) else torch.empty(0, dtype=dt, device="cuda")  # noqa: E731
        tb = None if table is None else to_dev(np.asarray(table, dtype=np.int32))
        cl = tpx3.Clusters(max(n, 1), pl.device)
        perm, label, nc, nk = pl.preprocess_cluster_centroid(dv(x, torch.uint16), dv(y, torch.uint16), dv(toa, torch.uint64),
                                                             dv(tot, torch.uint16), dv(trig, torch.uint64), cut, tb,
                                                             shot_base, cl)
        torch.cuda.synchronize()
        st = pl.status()
        k, ncl = int(nk.cpu().numpy()[0]), int(nc.cpu().numpy()[0])
        g = {"perm": perm[:k].cpu().numpy(), "label": label[:k].cpu().numpy(), "n_clusters": ncl}
        g.update(cl.numpy(ncl))
        pl.free()
        return st, k, g

    def want(x, y, toa, tot, trig, cut, table, shot_base):
        ex, ey, et, eo, ei = pp.preprocess(np.asarray(x, np.uint16), np.asarray(y, np.uint16), np.asarray(toa, np.uint64),
                                           np.asarray(tot, np.uint16), np.asarray(trig, np.uint64), cut,
                                           [] if table is None else table, P, shot_base)
        o = dict(oracle.run(ex, ey, et, eo, W, P))
        o["perm"] = ei[o["perm"]].astype(np.uint32)
        return len(ei), o

    # the hand example of the oracle pins, with the triggers a shot period apart so that it is shot-contiguous:
    # cut edge, clamp at 0, ToT beyond the table, an event before the first trigger
    base = [1000, 1000 + P, 1000 + 2 * P]
    toa = [900, 1000, 1300, 1301, base[1] + 4, base[1] + 150, base[1] + 999, base[2] + 100, base[2] + 3]
    args = (list(range(9)), [2 * v for v in range(9)], toa, [1, 1, 2, 2, 3, 3, 9, 1, 1], base, 300, [9, 5, 2, 0], 7)
    st, k, g = run(*args)
    kk, o = want(*args)
    assert st["error"] == 0 and k == kk
    assert_parity(g, o, "hand example")
    # nothing in; no triggers (everything dropped); no table
    st, k, g = run([], [], [], [], [5], 10, [1], 0)
    assert st["error"] == 0 and k == 0 and g["n_clusters"] == 0
    st, k, g = run([1, 2], [3, 4], [100, 200], [5, 6], [], 10, [1], 0)
    assert st["error"] == 0 and k == 0 and g["n_clusters"] == 0
    args = ([1, 2], [3, 4], [100, 200], [5, 6], [50], 1000, None, 3)
    st, k, g = run(*args)
    kk, o = want(*args)
    assert st["error"] == 0 and k == kk == 2
    assert_parity(g, o, "no table")
    # a stream that is not shot-contiguous (shots interleaved) and one whose shots exceed the window: reported
    x, y, raw, tot, trig, cut, table, per_shot = _raw_stream(1, 200, 3, 10, False)
    rng = np.random.default_rng(0)
    p = rng.permutation(len(x))
    st, _, _ = run(x[p], y[p], raw[p], tot[p], trig, cut, table, 0, hint=per_shot)
    assert st["error"] == tpx3.ERR_NOT_CONTIGUOUS
    x, y, raw, tot, trig, cut, table, per_shot = _raw_stream(3, 20, 4, 10, False)
    st, _, _ = run(x, y, raw, tot, trig, cut, table, 0, hint=512)      # 2100-event shots, 2048-event windows
    assert st["error"] == tpx3.ERR_NOT_CONTIGUOUS


def test_preprocess_rejects_a_cut_beyond_int64(tpx3):
    import torch

    pl = tpx3.plan(tpx3.Config(max_hits=16))
    z16 = torch.zeros(4, dtype=torch.uint16, device="cuda")
    z64 = torch.zeros(4, dtype=torch.uint64, device="cuda")
    with pytest.raises(tpx3.Tpx3Error) as e:
        pl.preprocess(z16, z16, z64, z16, z64, 1 << 63)
    assert e.value.code == tpx3.ERR_INVALID_ARG
    pl.free()


def test_two_devices_in_one_process(tpx3):
    """The opt-in to large dynamic shared memory is per device: a plan on cuda:1 made after one on cuda:0 must
    serve the fused path too. Skipped on a box with one GPU."""
    import torch

    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    w = gen.generate(1, shots=300)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P)
    for dev in (0, 1):
        with torch.cuda.device(dev):
            pl = tpx3.plan(tpx3.Config(max_hits=w.n, device=dev, max_shot_hits=600))
            d = [torch.from_numpy(a).to("cuda:%d" % dev) for a in (w.x, w.y, w.toa, w.tot)]
            cl = tpx3.Clusters(w.n, pl.device)
            perm, label, nc = pl.cluster_centroid(*d, cl)
            torch.cuda.synchronize(dev)
            st = pl.status()
            assert st["error"] == 0 and st["path"] == 1, (dev, st)
            g = {"perm": perm[: w.n].cpu().numpy(), "label": label[: w.n].cpu().numpy(), "n_clusters": int(nc.cpu().numpy()[0])}
            g.update(cl.numpy(g["n_clusters"]))
            assert_parity(g, o, "device %d" % dev)
            pl.free()


@pytest.mark.parametrize("cfg,shots,hint,pipelined", [(1, 24000, 1024, True), (4, 13000, 1536, True), (1, 24000, 1024, False)])
def test_process_host_pipelined(tpx3, cfg, shots, hint, pipelined):
    """Calls of >= 2^23 events go up in 2^22-event chunks pushed through the stream calls while later chunks
    are still being copied (tpx3_process_host): all rows against the oracle. The last case asks for perm and
    label as well, which takes the one-piece route on the same input: same rows."""
    import torch

    w = gen.generate(cfg, shots=shots)
    assert w.n >= 1 << 23
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P, threads=0)
    pl = tpx3.plan(tpx3.Config(max_hits=w.n, max_shot_hits=hint))
    hx, hy, htoa, htot = (torch.from_numpy(a).pin_memory() for a in (w.x, w.y, w.toa, w.tot))
    cap = w.n // 2
    cl = tpx3.Clusters(cap, "cpu", pin=True)
    extra = () if pipelined else (torch.empty(w.n, dtype=torch.uint32).pin_memory(),
                                  torch.empty(w.n, dtype=torch.uint32).pin_memory())
    for _ in range(2):                      # the second call reuses the device buffers of the first
        l0 = pl.launch_count()
        ncl = pl.process_host(hx, hy, htoa, htot, cl, *extra)
        launches = pl.launch_count() - l0
        assert ncl == o["n_clusters"]
        g = cl.numpy(ncl)
        for k in _ROW_KEYS:
            np.testing.assert_array_equal(g[k], o[k], err_msg=k)
        assert pl.host_route() == (1 if pipelined else 0)
        if pipelined:
            assert launches > 12            # several pushes, not one call
        else:
            assert launches <= 8
            np.testing.assert_array_equal(extra[0].numpy(), o["perm"])
            np.testing.assert_array_equal(extra[1].numpy(), o["label"])
    pl.free()


def test_process_host_pipelined_falls_back_on_a_broken_promise(tpx3):
    """Pixels that arrive four shots late, behind a chunk cut, break the half-period disorder bound the pipelined route assumes: it
    notices (late events) and redoes the call in one piece; the rows are the oracle's all the same."""
    import torch

    w0 = gen.generate(1, shots=24000)
    shot = (w0.toa // np.uint64(P)).astype(np.int64)
    shot -= shot.min()
    s_b = shot[1 << 22]                       # the shot the first chunk cut falls into
    moved = (shot == s_b - 3) & (np.arange(w0.n) % 3 == 0)      # ... arrive in the second chunk, 4 shots late
    order = np.argsort(np.where(moved, shot + 4, shot) * 4 + moved, kind="stable")
    x, y, toa, tot = w0.x[order], w0.y[order], w0.toa[order], w0.tot[order]
    o = oracle.run(x, y, toa, tot, W, P, threads=0)
    pl = tpx3.plan(tpx3.Config(max_hits=w0.n))
    cl = tpx3.Clusters(w0.n // 2, "cpu", pin=True)
    ncl = pl.process_host(*(torch.from_numpy(a).pin_memory() for a in (x, y, toa, tot)), cl)
    assert ncl == o["n_clusters"] and pl.host_route() == 2
    g = cl.numpy(ncl)
    for k in _ROW_KEYS:
        np.testing.assert_array_equal(g[k], o[k], err_msg=k)
    pl.free()


def test_process_host_pipelined_capacity(tpx3):
    """A host table too small for the hits of a pipelined call: TPX3_ERR_CAPACITY, the rows that fit are the
    first rows of the oracle's table, and the plan serves the next call as usual."""
    import torch

    w = gen.generate(1, shots=24000)
    o = oracle.run(w.x, w.y, w.toa, w.tot, W, P, threads=0)
    pl = tpx3.plan(tpx3.Config(max_hits=w.n, max_shot_hits=1024))
    host = [torch.from_numpy(a).pin_memory() for a in (w.x, w.y, w.toa, w.tot)]
    small = tpx3.Clusters(400001, "cpu", pin=True)
    with pytest.raises(tpx3.Tpx3Error) as ei:
        pl.process_host(*host, small)
    assert ei.value.code == tpx3.ERR_CAPACITY and pl.host_route() == 1
    g = small.numpy(400001)
    for k in _ROW_KEYS:
        np.testing.assert_array_equal(g[k], o[k][:400001], err_msg=k)
    cl = tpx3.Clusters(w.n // 2, "cpu", pin=True)
    assert pl.process_host(*host, cl) == o["n_clusters"]
    np.testing.assert_array_equal(cl.numpy(o["n_clusters"])["c_sum_tot_tof"], o["c_sum_tot_tof"])
    pl.free()


def test_preprocess_long_trigger_list(tpx3):
    """More than 512^2 triggers (the block-wide window search finishes with a binary search), events scattered
    over the whole list, some before the first trigger and some beyond the cut: against the oracle."""
    import torch
    from oracle import preprocess as pp

    rng = np.random.default_rng(23)
    nt, n = 300000, 30011
    trig = np.cumsum(rng.integers(500, 900, nt)).astype(np.uint64) + np.uint64(1000)
    toa = np.sort(rng.integers(0, int(trig[-1]) + 2000, n)).astype(np.uint64)
    swap = rng.integers(0, n - 1, 500)                       # a little disorder
    toa[swap], toa[swap + 1] = toa[swap + 1].copy(), toa[swap].copy()
    x = rng.integers(0, 256, n).astype(np.uint16)
    y = rng.integers(0, 256, n).astype(np.uint16)
    tot = rng.integers(1, 1024, n).astype(np.uint16)
    table = tpx3.timewalk_table(300.0, 1.0, 2.0, 1.1, 64)
    pl = tpx3.plan(tpx3.Config(max_hits=n, shot_period_ticks=P))
    xo, yo, to, oo, io, no = pl.preprocess(to_dev(x), to_dev(y), to_dev(toa), to_dev(tot), to_dev(trig), 400,
                                           to_dev(table), 5)
    torch.cuda.synchronize()
    k = int(no.cpu().numpy()[0])
    ex, ey, et, eo, ei = pp.preprocess(x, y, toa, tot, trig, 400, table, P, 5)
    assert k == len(ei) and 0 < k < n
    np.testing.assert_array_equal(to[:k].cpu().numpy(), et)
    np.testing.assert_array_equal(io[:k].cpu().numpy().astype(np.int64), ei)
    np.testing.assert_array_equal(xo[:k].cpu().numpy(), ex)
    np.testing.assert_array_equal(oo[:k].cpu().numpy(), eo)
    pl.free()
