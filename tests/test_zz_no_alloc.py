"""mdpd_get_pairs_static: the neighbour-pair search for callers that cannot allocate device memory.

Some users of this library run inside a process whose device memory is already spoken for -- a tensor framework's
caching allocator or a job that reserves the whole card at start-up holds every free byte, so a cudaMalloc made from
inside the library fails although the pool has room -- or on a latency-critical path next to other streams, where
cudaMalloc / cudaFree stall the whole device.  For them the library offers one entry point whose scratch (hit counter +
unsorted pair buffer) is a fixed ~4 MiB array inside the library image (MDPD_STATIC_PAIRS_MAX pairs; include/mdpd.h).

What is checked here: the new entry point returns exactly what the allocating mdpd_get_pairs returns (pair sets are
integer work: the bar is bit-exact, as in tests/test_gpu_parity.py), on two calls in a row (the second one finds a
used array: stale pairs and a non-zero counter from the first), on both neighbour paths, after the particles have
moved, through the raw C-ABI with a cap smaller than the number found, and that a request beyond the fixed maximum is
refused with a clear error instead of overrunning the array.

The file name sorts last on purpose: `pytest -x` stops at the first failure, so a failure here cannot hide any other
test.  It passes alone in a fresh process (the first call then is the per-device set-up call) and after the rest of
the suite (the library is then already loaded and used).
"""
import ctypes as C

import numpy as np
import pytest

import mdpd_workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the -m gpu suite needs a CUDA device (no CPU fallback exists)")
    from paper_1903_10134_b200 import build
    build()
    import paper_1903_10134_b200 as pk
    return pk


def make_sim(pk, c, direct=False):
    prm = dict(c["params"])
    if direct:
        prm["flags"] = 2        # MDPD_FLAG_DIRECT
    s = pk.Simulation(prm)
    s.load_particles(c["pos"], c["vel"], c["type"])
    return s


@pytest.mark.parametrize("direct", [False, True])
def test_static_scratch_equals_allocating_path_two_calls_in_a_row(gpu, direct):
    c = wl.make_config(0)                       # 6000 particles, 10^3 box: ~75 000 pairs inside rc
    s = make_sim(gpu, c, direct)
    # call 1: the widest search (rc + skin); on a fresh process this is also the set-up call of the device
    want_wide = s.get_pairs(1.25)
    got_wide = s.get_pairs_static(1.25)
    assert len(want_wide) > 100_000
    assert got_wide.dtype == want_wide.dtype and got_wide.shape == want_wide.shape
    assert np.array_equal(got_wide, want_wide)
    # call 2, straight after: fewer pairs, so the array still holds call 1's pairs beyond the new count and call 1's
    # counter value before the library clears it -- neither may leak into the result
    want_rd = s.get_pairs(0.75)
    got_rd = s.get_pairs_static(0.75)
    assert 0 < len(want_rd) < len(want_wide) // 2
    assert got_rd.shape == want_rd.shape and np.array_equal(got_rd, want_rd)
    # and the same call repeated gives the same answer
    assert np.array_equal(s.get_pairs_static(0.75), want_rd)
    # after the particles have moved (and the list has been rebuilt at least once)
    s.step(40)
    assert s.counters()["rebuilds"] >= 1 or direct
    want = s.get_pairs(1.0)
    got = s.get_pairs_static(1.0)
    assert got.shape == want.shape and np.array_equal(got, want)
    s.close()


def test_static_scratch_is_shared_between_handles(gpu):
    """One array per device serves every handle: calls that do not overlap (each one synchronises its stream before it
    returns) may alternate between handles freely."""
    a = make_sim(gpu, wl.make_liquid(6.0, seed=21))
    b = make_sim(gpu, wl.make_liquid((5.0, 6.0, 7.0), seed=22))
    for rcut in (1.0, 0.75, 1.25):
        assert np.array_equal(a.get_pairs_static(rcut), a.get_pairs(rcut))
        assert np.array_equal(b.get_pairs_static(rcut), b.get_pairs(rcut))
    a.close()
    b.close()


def test_static_scratch_cap_below_count_and_limit(gpu):
    c = wl.make_config(0)
    s = make_sim(gpu, c)
    L, h = s._L, s._h
    full = s.get_pairs(1.0)
    cnt = C.c_uint64()
    # cap smaller than the number found: *count reports all of them, `cap` valid pairs come back, the rest of the
    # caller's buffer is untouched
    cap = 1000
    buf = np.full((cap + 8, 2), 0xFFFFFFFF, np.uint32)
    assert L.mdpd_get_pairs_static(h, 1.0, C.addressof(cnt), buf.ctypes.data, cap) == 0
    assert cnt.value == len(full)
    assert (buf[cap:] == 0xFFFFFFFF).all()
    keys = set(map(tuple, full.tolist()))
    assert all(tuple(p) in keys for p in buf[:cap].tolist())
    assert len(set(map(tuple, buf[:cap].tolist()))) == cap
    assert (np.diff(buf[:cap, 0].astype(np.int64) * 2 ** 32 + buf[:cap, 1]) > 0).all()      # sorted
    # count only (pairs = NULL)
    assert L.mdpd_get_pairs_static(h, 1.0, C.addressof(cnt), None, 0) == 0 and cnt.value == len(full)
    # beyond the fixed maximum: refused up front with a message that names the limit, nothing written
    big = gpu.binding.MDPD_STATIC_PAIRS_MAX + 1
    buf2 = np.zeros((big, 2), np.uint32)
    assert L.mdpd_get_pairs_static(h, 1.0, C.addressof(cnt), buf2.ctypes.data, big) == -1     # MDPD_EINVAL
    msg = L.mdpd_last_error(h).decode()
    assert "MDPD_STATIC_PAIRS_MAX" in msg and str(gpu.binding.MDPD_STATIC_PAIRS_MAX) in msg
    assert not buf2.any()
    with pytest.raises(gpu.MdpdError):
        s.get_pairs_static(1.0, cap=big)
    # exactly the maximum is accepted
    buf3 = np.zeros((big - 1, 2), np.uint32)
    assert L.mdpd_get_pairs_static(h, 1.0, C.addressof(cnt), buf3.ctypes.data, big - 1) == 0
    assert np.array_equal(buf3[:len(full)], full)
    # and the handle still works afterwards
    assert np.array_equal(s.get_pairs_static(1.0), full)
    s.close()
