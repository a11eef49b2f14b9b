"""Several devices behind one server (include/pp_multi.h, NEXT-4) without a GPU: the front deals
batches to host-only echo back ends (tests/echo_backend.cpp), one per "device"."""
import os
import re
import threading

import numpy as np
import pytest

from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import ipc
from paper_2405_05700_b200 import multi

from test_ipc_transport import _expected, _sources, echo_backend

ORDER = ["event_id", "source_id"]


def test_multi_symbols_are_exported():
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    hdr = re.sub(r"/\*.*?\*/", "", open(os.path.join(root, "include", "pp_multi.h")).read(), flags=re.S)
    declared = set(re.findall(r"\b(pp_multi_[a-z_]+)\s*\(", hdr))
    lib = B.load_library()
    for s in declared:
        assert hasattr(lib, s), s
    assert declared == set(multi.EXPORTS)


@pytest.mark.parametrize("n_dev", [1, 2, 3])
def test_every_source_comes_back_once_and_the_load_is_shared(n_dev):
    src, ev, sid, ln = _sources(0, 40, 25)               # 1000 sources of 1e3-1e5 photons
    tot = sum(B.photon_count(e) for e in src[:, 7])
    with multi.MultiFront(backends=[echo_backend() for _ in range(n_dev)], photons_per_GeV=1.0e4,
                          deal_photons=tot // 20) as m:
        got = []
        for a in range(0, len(ev), 90):                   # blocks that do not line up with the batches
            m.submit(src[a:a + 90], ev[a:a + 90], sid[a:a + 90], ln[a:a + 90])
            got.append(m.collect(block=False).copy())
        got.append(m.collect_all())
        st = m.stats()
    hits = np.sort(np.concatenate(got), order=ORDER)
    assert np.array_equal(hits, _expected(src, ev, sid, ln))
    assert st["sources_submitted"] == st["sources_completed"] == 1000 and st["sources_staged"] == 0
    assert st["photons_submitted"] == tot == sum(st["photons"]) and st["photons_outstanding"] == [0] * n_dev
    assert sum(st["batches"]) >= 19
    if n_dev > 1:
        # the echo back end completes a batch at once, so all devices look idle and the first one would get
        # everything if ties were not the only thing deciding; what must hold: nobody got more than everything
        assert max(st["photons"]) <= tot


def test_least_loaded_device_gets_the_next_batch():
    """Back end 0 never completes anything until flushed by hand (its flush is a no-op here): the front must send the
    following batches to the other device."""
    import ctypes as C
    be0, be1 = echo_backend(), echo_backend()
    # wrap back end 0 so that its flush does nothing: its batches stay outstanding
    b0 = multi.Backend()
    C.memmove(C.byref(b0), C.c_void_p(be0), C.sizeof(multi.Backend))
    real_flush = b0.flush
    NOFLUSH = C.CFUNCTYPE(C.c_int, C.c_void_p)(lambda ctx: 0)
    b0.flush = C.cast(NOFLUSH, C.c_void_p).value
    src, ev, sid, ln = _sources(1, 10, 10)
    tot = sum(B.photon_count(e) for e in src[:, 7])
    with multi.MultiFront(backends=[C.addressof(b0), be1], photons_per_GeV=1.0e4, deal_photons=tot // 10) as m:
        m.submit(src, ev, sid, ln)
        m.flush()
        st = m.stats()
        assert st["batches"][0] == 1 and st["batches"][1] >= 8, st      # one batch stuck on device 0, the rest on 1
        assert st["photons_outstanding"][0] > 0 and st["photons_outstanding"][1] == 0
        assert st["sources_completed"] == 0                               # the FIRST batch is the stuck one
        # release device 0
        C.CFUNCTYPE(C.c_int, C.c_void_p)(real_flush)(b0.ctx)
        hits = np.sort(np.concatenate([m.collect_all()]), order=ORDER)
        assert np.array_equal(hits, _expected(src, ev, sid, ln))
        assert m.stats()["sources_completed"] == 100


def test_null_ids_are_numbered_by_the_front_and_submit_is_thread_safe():
    src, ev, sid, ln = _sources(2, 8, 50)
    with multi.MultiFront(backends=[echo_backend(), echo_backend()], photons_per_GeV=1.0e4, deal_photons=10 ** 6) as m:
        def work(t):
            for a in range(t * 100, (t + 1) * 100, 20):
                m.submit(src[a:a + 20], ev[a:a + 20], None, ln[a:a + 20])
        th = [threading.Thread(target=work, args=(t,)) for t in range(4)]
        [t.start() for t in th]
        [t.join() for t in th]
        hits = m.collect_all()
    assert len(hits) == 400 and sorted(hits["source_id"]) == list(range(400))   # unique across devices and calls


def test_front_rejects_bad_input():
    with pytest.raises(B.PPError):
        multi.MultiFront(backends=[], photons_per_GeV=1.0e4)
    with pytest.raises(B.PPError):
        multi.MultiFront(backends=[echo_backend()], photons_per_GeV=0.0)
    with multi.MultiFront(backends=[echo_backend()], photons_per_GeV=1.0e4) as m:
        src, ev, sid, ln = _sources(3, 1, 2)
        big = src.copy()
        big[0, 7] = 1.0e9                                  # 1e13 photons: more than 2^32 - 1 in one source
        with pytest.raises(B.PPError) as e:
            m.submit(big, ev, sid, ln)
        assert e.value.code == -4 and m.stats()["sources_submitted"] == 0   # nothing was staged
        assert len(m.collect(block=True)) == 0             # nothing outstanding: drained at once
        # what a handle would refuse is refused here, in the caller that made the call (round-2 advice)
        for col, val in ((3, 2.0), (0, np.nan), (6, np.inf), (7, -1.0)):
            bad = src.copy()
            bad[1, col] = val
            with pytest.raises(B.PPError) as e:
                m.submit(bad, ev, sid, ln)
            assert e.value.code == -1
        for val in (-1.0, np.nan):
            bad_ln = ln.copy()
            bad_ln[0] = val
            with pytest.raises(B.PPError) as e:
                m.submit(src, ev, sid, bad_ln)
            assert e.value.code == -1
        assert m.stats()["sources_submitted"] == 0 and m.stats()["sources_staged"] == 0
        m.submit(src, ev, sid, ln)                         # and a good call after all that goes through
        assert np.array_equal(np.sort(m.collect_all(), order=ORDER), _expected(src, ev, sid, ln))


def test_a_batch_the_device_refuses_does_not_wedge_the_front():
    """A back end with stricter rules than the front's refuses one batch: that batch is dropped (counted as complete,
    no hits), the caller whose deal met it gets the code, and everybody else's sources go on."""
    import ctypes as C
    be = multi.Backend()
    C.memmove(C.byref(be), C.c_void_p(echo_backend()), C.sizeof(multi.Backend))
    SUBMIT = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_uint32), C.c_void_p, C.c_size_t)
    real = SUBMIT(be.submit)

    def picky(ctx, s, ln, ev, sid, n):
        if any(ev[i] == 4003 for i in range(n)):
            return -1
        return real(ctx, s, ln, ev, sid, n)

    keep = SUBMIT(picky)
    be.submit = C.cast(keep, C.c_void_p).value
    src, ev, sid, ln = _sources(4, 6, 5)                   # events 4000..4005, five sources each
    with multi.MultiFront(backends=[C.addressof(be)], photons_per_GeV=1.0e4, deal_photons=1) as m:
        ok = ev != 4003
        m.submit(src[ev < 4003], ev[ev < 4003], sid[ev < 4003], ln[ev < 4003])
        with pytest.raises(B.PPError) as e:                # deal_photons = 1: every submit deals what it brought
            m.submit(src[ev == 4003][:1], ev[ev == 4003][:1], sid[ev == 4003][:1], ln[ev == 4003][:1])
        assert e.value.code == -1
        m.submit(src[ev > 4003], ev[ev > 4003], sid[ev > 4003], ln[ev > 4003])
        hits = np.sort(m.collect_all(), order=ORDER)
        st = m.stats()
    assert np.array_equal(hits, _expected(src[ok], ev[ok], sid[ok], ln[ok]))
    assert st["sources_staged"] == 0 and st["sources_completed"] == st["sources_submitted"] == int(ok.sum()) + 1


def test_client_processes_in_front_of_two_devices():
    """pp_multi_backend: the multi-process server (pp_ipc.h) drives the front, which drives two "devices"."""
    name = f"/pp_multi_test_{os.getpid()}"
    with multi.MultiFront(backends=[echo_backend(), echo_backend()], photons_per_GeV=1.0e4, deal_photons=3 * 10 ** 5) as m:
        with ipc.IpcServer(None, name, max_clients=2, backend=m.backend_address()) as srv:
            a, b = ipc.IpcClient(name), ipc.IpcClient(name)
            sa, ea, ia, la = _sources(0, 6, 30)
            sb, eb, ib, lb = _sources(1, 4, 45)
            a.submit(sa, ea, ia, la)
            b.submit(sb, eb, ib, lb)
            ga = np.sort(a.collect_all(), order=ORDER)
            gb = np.sort(b.collect_all(), order=ORDER)
            assert np.array_equal(ga, _expected(sa, ea, ia, la)) and np.array_equal(gb, _expected(sb, eb, ib, lb))
            assert srv.stats()["error"] == 0 and srv.stats()["hits_unrouted"] == 0
            a.close(), b.close()
        st = m.stats()
        assert sum(st["batches"]) >= 2 and st["sources_completed"] == 360


def test_the_front_stays_responsive_while_a_device_takes_a_batch_slowly():
    """A device whose source ring is full blocks in submit (pp.h).  The front hands a batch over OUTSIDE its lock
    (round-2 advice): meanwhile the statistics and the completed count answer, other callers' batches go to the other
    device, and "drained" is not reported while a batch is on its way."""
    import ctypes as C
    import time
    b0 = multi.Backend()
    C.memmove(C.byref(b0), C.c_void_p(echo_backend()), C.sizeof(multi.Backend))
    SUBMIT = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t)
    real = SUBMIT(b0.submit)
    entered, gate = threading.Event(), threading.Event()

    def slow(ctx, s, ln, ev, sid, n):
        entered.set()
        gate.wait(20)
        return real(ctx, s, ln, ev, sid, n)

    keep = SUBMIT(slow)
    b0.submit = C.cast(keep, C.c_void_p).value
    s1, e1, i1, l1 = _sources(5, 2, 4)
    s2, e2, i2, l2 = _sources(6, 3, 3)
    with multi.MultiFront(backends=[C.addressof(b0), echo_backend()], photons_per_GeV=1.0e4, deal_photons=10 ** 12) as m:
        t = threading.Thread(target=lambda: (m.submit(s1, e1, i1, l1), m.flush()))  # the flush deals one batch
        t.start()
        try:
            assert entered.wait(10)                           # device 0 is "taking" that batch and will not finish
            t0 = time.monotonic()
            st = m.stats()                                    # needs the front's lock
            assert st["sources_staged"] == 0 and st["photons_outstanding"][0] > 0 and st["sources_completed"] == 0
            m.submit(s2, e2, i2, l2)
            m.flush()                                         # dealt to device 1: device 0 is busy
            got2 = []
            while len(got2) < len(e2) and time.monotonic() - t0 < 5:
                got2.extend(m.collect(block=False))
            assert time.monotonic() - t0 < 5 and len(got2) == len(e2)
            assert m.stats()["batches"] == [1, 1]
        finally:
            gate.set()
            t.join(10)
        assert not t.is_alive()
        got1 = np.sort(m.collect_all(), order=ORDER)
        st = m.stats()
    assert np.array_equal(got1, _expected(s1, e1, i1, l1))
    assert np.array_equal(np.sort(np.array(got2, dtype=B.HIT_DTYPE), order=ORDER), _expected(s2, e2, i2, l2))
    assert st["sources_completed"] == st["sources_submitted"] == len(e1) + len(e2)
