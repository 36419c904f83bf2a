"""GPU test of the entry point that allocates nothing (tpx3_unwrap_toa_static, include/tpx3.h): its scratch is a
fixed `static __device__` array inside the library. Collected last on purpose (the suite runs with pytest -x).

The existing path (tpx3_unwrap_toa: plan + caller-owned workspace) is itself bit-identical to the sequential
oracle (tests/test_gpu_parity.py::test_unwrap_toa); the new entry point runs the same kernels on other scratch, so
the bar is the one those tests use: exact equality of every output, on two calls in a row that share the array.
"""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tpx3():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    import paper_2603_04942_b200 as m

    m.load_library()
    return m


def _stream(n, seed, modulus, wraps=3):
    """Counter values of a time axis that runs over `wraps` counter periods, reported slightly out of order."""
    rng = np.random.default_rng(seed)
    t = np.sort(rng.integers(0, wraps * modulus, n)).astype(np.int64)
    t += rng.integers(-2000, 2000, n)                      # pixels report out of order
    t = np.clip(t, 0, wraps * modulus - 1)
    return (t % modulus).astype(np.uint64)


def test_unwrap_static_matches_the_workspace_path_twice_in_a_row(tpx3):
    import torch

    m = tpx3
    modulus, jump = 1 << 34, 1 << 33
    # two calls in a row on the shared array: a long one (1222 block counts), then a shorter one with carried-in
    # state whose counts overwrite only the front of what the first call left behind
    cases = [(5_000_123, 1, 0, None), (70_001, 2, -2, int(modulus - 5))]
    pl = m.plan(m.Config(max_hits=max(c[0] for c in cases)))
    before = torch.cuda.memory_allocated()
    outs = []
    for n, seed, wraps_in, prev in cases:
        raw = torch.from_numpy(_stream(n, seed, modulus)).cuda()
        want, want_w = pl.unwrap_toa(raw, modulus, jump, wraps_in=wraps_in, prev_raw=prev)
        got = torch.empty_like(raw)
        got_w = torch.empty(1, dtype=torch.int64, device="cuda")
        m.unwrap_toa_static(raw, modulus, jump, got, got_w, wraps_in=wraps_in, prev_raw=prev)
        torch.cuda.synchronize()
        outs.append((want.cpu().numpy(), want_w.cpu().numpy(), got.cpu().numpy(), got_w.cpu().numpy()))
    for (want, want_w, got, got_w), (n, _, wraps_in, _) in zip(outs, cases):
        np.testing.assert_array_equal(got, want, err_msg="n = %d" % n)
        np.testing.assert_array_equal(got_w, want_w, err_msg="n = %d" % n)
        assert int(got_w[0]) != wraps_in            # the stream really wrapped
    # and the same call again gives the same result (the array kept the last call's contents)
    n, seed, wraps_in, prev = cases[0]
    raw = torch.from_numpy(_stream(n, seed, modulus)).cuda()
    got = torch.empty_like(raw)
    got_w = torch.empty(1, dtype=torch.int64, device="cuda")
    m.unwrap_toa_static(raw, modulus, jump, got, got_w, wraps_in=wraps_in, prev_raw=prev)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(got.cpu().numpy(), outs[0][2])
    del raw, got, got_w, want, want_w
    pl.free()
    assert torch.cuda.memory_allocated() <= before + (1 << 20)     # nothing of the calls stays allocated


def test_unwrap_static_edges_and_limit(tpx3):
    import torch

    m = tpx3
    lib = m.load_library()
    out = torch.zeros(8, dtype=torch.uint64, device="cuda")
    w = torch.full((1,), 99, dtype=torch.int64, device="cuda")
    # n = 0: only the counter is passed through
    m.unwrap_toa_static(torch.empty(0, dtype=torch.uint64, device="cuda"), 1 << 20, 1 << 19, out[:0], w, wraps_in=7)
    torch.cuda.synchronize()
    assert int(w.cpu().numpy()[0]) == 7
    # beyond the fixed scratch: refused before anything is enqueued (the pointers are never touched)
    rc = lib.tpx3_unwrap_toa_static(0, None, m.STATIC_UNWRAP_MAX + 1, out.data_ptr(), 1 << 20, 1 << 19, 0, 0, 0,
                                    out.data_ptr(), w.data_ptr())
    assert rc == m.ERR_TOO_LARGE
    assert "TPX3_STATIC_UNWRAP_MAX" in m.strerror(rc)
    assert lib.tpx3_unwrap_toa_static(0, None, 8, out.data_ptr(), 0, 1, 0, 0, 0, out.data_ptr(), w.data_ptr()) == m.ERR_INVALID_ARG
    assert lib.tpx3_unwrap_toa_static(-1, None, 8, out.data_ptr(), 4, 1, 0, 0, 0, out.data_ptr(), w.data_ptr()) == m.ERR_INVALID_ARG
    # exactly at the limit is served (2^26 events: 512 MB in, 512 MB out)
    n = m.STATIC_UNWRAP_MAX
    raw = (torch.arange(n, dtype=torch.int64, device="cuda") % 1000003).to(torch.uint64)
    big = torch.empty(n, dtype=torch.uint64, device="cuda")
    m.unwrap_toa_static(raw, 1000003, 500000, big, w)
    torch.cuda.synchronize()
    assert int(w.cpu().numpy()[0]) == (n - 1) // 1000003
    assert int(big[-1].cpu().numpy()) == n - 1 and int(big[n // 2].cpu().numpy()) == n // 2
    assert ctypes.sizeof(ctypes.c_uint32) * (n // 4096) == 64 * 1024       # the array the header states
