"""The multi-process front end (include/pp_ipc.h, NEXT-3) without a GPU: client processes
ship blocks through shared memory to a server bound to the host-only echo back end of tests/echo_backend.cpp (one hit
per source), plugged in through pp_ipc_server_create_backend."""
import multiprocessing as mp
import os

import numpy as np
import pytest

from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import ipc
from paper_2405_05700_b200 import workloads as W


def _echo_lib():
    import ctypes as C
    from conftest import build_echo_backend
    L = C.CDLL(build_echo_backend())
    L.echo_backend_new.restype = C.c_void_p
    L.echo_set_hits_per_source.argtypes = [C.c_void_p, C.c_uint32]
    L.echo_set_collect_delay_us.argtypes = [C.c_void_p, C.c_uint32]
    return L


def echo_backend(hits_per_source: int = 1) -> int:
    """Address of a fresh host-only back end (tests/echo_backend.cpp): one hit per source at the next flush."""
    L = _echo_lib()
    be = L.echo_backend_new()
    if hits_per_source != 1:
        L.echo_set_hits_per_source(be, hits_per_source)
    return be


def _sources(client: int, n_events: int, per_event: int):
    """Deterministic sources of one client: event ids client*1000 + e."""
    rng = np.random.default_rng(100 + client)
    n = n_events * per_event
    d = rng.normal(size=(n, 3))
    d /= np.linalg.norm(d, axis=1)[:, None]
    src = np.zeros((n, 8), np.float32)
    src[:, 0:3] = rng.uniform(-100, 100, size=(n, 3))
    src[:, 3:6] = d
    src[:, 6] = rng.uniform(0, 1000, size=n)
    src[:, 7] = rng.uniform(0.1, 10.0, size=n)
    ev = (client * 1000 + np.repeat(np.arange(n_events), per_event)).astype(np.uint32)
    sid = np.tile(np.arange(per_event), n_events).astype(np.uint32)
    ln = rng.uniform(0, 5, size=n).astype(np.float32)
    return src, ev, sid, ln


def _expected(src, ev, sid, ln):
    out = np.zeros(len(ev), dtype=B.HIT_DTYPE)
    out["event_id"], out["source_id"] = ev, sid
    out["photon_idx"] = [B.photon_count(e) for e in src[:, 7]]
    out["time_ns"] = src[:, 6].astype(np.float64) + ln.astype(np.float64)
    out["weight"] = src[:, 7]
    return np.sort(out, order=["event_id", "source_id"])


def _client_main(name, client, n_events, per_event, block, q):
    try:
        src, ev, sid, ln = _sources(client, n_events, per_event)
        got = []
        with ipc.IpcClient(name) as c:
            for a in range(0, len(ev), block):  # ship block by block, collecting in between (streaming)
                c.submit(src[a:a + block], ev[a:a + block], sid[a:a + block], ln[a:a + block])
                h = c.collect(block=False)
                if len(h):
                    got.append(h.copy())
            got.append(c.collect_all())
        hits = np.sort(np.concatenate(got), order=["event_id", "source_id"])
        q.put((client, hits.tobytes()))
    except Exception as e:  # pragma: no cover
        q.put((client, repr(e)))


@pytest.mark.parametrize("n_clients,ring_kib", [(1, 4096), (4, 4096), (8, 8)])
def test_clients_get_exactly_their_events_back(n_clients, ring_kib):
    """n client processes, one server; tiny rings (8 KiB = 170 sources / 256 hits) force back-pressure both ways."""
    name = f"/pp_ipc_test_{os.getpid()}_{n_clients}_{ring_kib}"
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    n_events, per_event, block = 20, 37, 111
    with ipc.IpcServer(None, name, max_clients=n_clients, source_ring_bytes=ring_kib * 1024,
                       hit_ring_bytes=ring_kib * 1024, backend=echo_backend()) as srv:
        procs = [ctx.Process(target=_client_main, args=(name, c, n_events, per_event, block, q)) for c in range(n_clients)]
        for p in procs:
            p.start()
        res = dict(q.get(timeout=120) for _ in procs)
        for p in procs:
            p.join(timeout=60)
        st = srv.stats()
    assert st["error"] == 0 and st["hits_unrouted"] == 0
    # (a client that has finished may leave its slot to a later one: at most n_clients distinct slots)
    assert 1 <= st["clients_attached"] <= n_clients and st["sources_ingested"] == n_clients * n_events * per_event
    assert st["hits_routed"] == st["sources_ingested"]
    for c in range(n_clients):
        assert isinstance(res[c], bytes), res[c]
        hits = np.frombuffer(res[c], dtype=B.HIT_DTYPE)
        assert np.array_equal(hits, _expected(*_sources(c, n_events, per_event)))


def test_open_errors_and_slot_limit():
    with pytest.raises(B.PPError) as e:
        ipc.IpcClient(f"/pp_ipc_nobody_{os.getpid()}")
    assert e.value.code == -7  # PP_E_STATE: no server
    name = f"/pp_ipc_test_{os.getpid()}_lim"
    with ipc.IpcServer(None, name, max_clients=2, backend=echo_backend()):
        with pytest.raises(B.PPError):
            ipc.IpcServer(None, name, backend=echo_backend())  # the segment exists already
        a, b = ipc.IpcClient(name), ipc.IpcClient(name)
        with pytest.raises(B.PPError) as e:
            ipc.IpcClient(name)
        assert e.value.code == -2  # PP_E_NOMEM: no free slot
        src, ev, sid, ln = _sources(0, 2, 3)
        bad = src.copy()
        bad[0, 3:6] = 0.0
        with pytest.raises(B.PPError):
            a.submit(bad, ev, sid, ln)
        with pytest.raises(B.PPError):
            a.submit(src, ev, sid, -ln - 1.0)
        assert len(a.collect_all()) == 0  # nothing was shipped: drained at once
        b.submit(src, ev, sid, ln)
        assert np.array_equal(np.sort(b.collect_all(), order=["event_id", "source_id"]), _expected(src, ev, sid, ln))
        a.close(), b.close()
    with pytest.raises(B.PPError):
        ipc.IpcClient(name)  # unlinked with the server


def test_a_client_drains_without_waiting_for_the_others():
    """Steady state (clients keep queueing steps): client A must see its own work drained while client B
    still has a block in the server that nobody flushed."""
    name = f"/pp_ipc_test_{os.getpid()}_own"
    with ipc.IpcServer(None, name, max_clients=2, backend=echo_backend()) as srv:
        a, b = ipc.IpcClient(name), ipc.IpcClient(name)
        sa, ea, ia, la = _sources(0, 5, 11)
        sb, eb, ib, lb = _sources(1, 3, 7)
        a.submit(sa, ea, ia, la)
        got_a = np.sort(a.collect_all(), order=["event_id", "source_id"])   # flushes A's block
        assert np.array_equal(got_a, _expected(sa, ea, ia, la))
        b.submit(sb, eb, ib, lb)                                            # shipped, never flushed
        import time
        time.sleep(0.05)
        sa2, ea2, ia2, la2 = _sources(2, 2, 5)
        a.submit(sa2, ea2, ia2, la2)
        got_a2 = a.collect_all()             # A's flush makes the server launch B's block too ...
        assert len(got_a2) == len(ea2)
        got_b = np.sort(b.collect_all(), order=["event_id", "source_id"])   # ... and B finds its hits
        assert np.array_equal(got_b, _expected(sb, eb, ib, lb))
        # now B ships a block that stays unflushed while A runs a whole cycle: A must not hang
        b.submit(sb, eb + 500, ib, lb)
        time.sleep(0.05)
        assert len(a.collect(block=True)) == 0      # nothing outstanding for A: drained at once
        assert srv.stats()["error"] == 0
        a.close(), b.close()


def test_slots_are_recycled():
    """Clients come and go on a long-running server: a slot is handed out again once its client has left and the
    server has run dry."""
    import time
    name = f"/pp_ipc_test_{os.getpid()}_recycle"
    with ipc.IpcServer(None, name, max_clients=2, backend=echo_backend()) as srv:
        keep = ipc.IpcClient(name)
        for round_ in range(5):
            c = None
            for _ in range(200):            # the slot of the previous round comes back within milliseconds
                try:
                    c = ipc.IpcClient(name)
                    break
                except B.PPError as e:
                    assert e.code == -2
                    time.sleep(0.005)
            assert c is not None, "slot was not recycled"
            src, ev, sid, ln = _sources(round_, 3, 9)
            c.submit(src, ev + np.uint32(10000 * round_), sid, ln)
            if round_ % 2:
                got = np.sort(c.collect_all(), order=["event_id", "source_id"])
                exp = _expected(src, ev + np.uint32(10000 * round_), sid, ln)
                assert np.array_equal(got, exp)
            else:
                c.flush()                   # leaves without reading its hits: they must not reach the next client
            c.close()
        assert srv.stats()["clients_attached"] == 2 and srv.stats()["error"] == 0
        keep.close()


def test_server_gone_and_client_gone():
    """A client that outlives the server gets PP_E_STATE instead of hanging; a client that leaves without reading its
    hits does not wedge the server (its hits are dropped), and the other client still drains."""
    name = f"/pp_ipc_test_{os.getpid()}_gone"
    src, ev, sid, ln = _sources(0, 4, 50)
    srv = ipc.IpcServer(None, name, max_clients=2, hit_ring_bytes=32 * 8, backend=echo_backend())  # hit ring of 8 hits
    a, b = ipc.IpcClient(name), ipc.IpcClient(name)
    a.submit(src, ev, sid, ln)          # 200 hits will come back into a ring of 8 ...
    a.flush()
    assert len(a.collect(cap=4, block=True)) > 0
    a.close()                           # ... but the client leaves after reading a few
    s2, e2, i2, l2 = _sources(1, 3, 20)
    b.submit(s2, e2, i2, l2)
    got = np.sort(b.collect_all(), order=["event_id", "source_id"])
    assert np.array_equal(got, _expected(s2, e2, i2, l2))
    st = srv.stats()
    assert st["error"] == 0 and st["sources_ingested"] == 260
    b.submit(s2[:5], e2[:5] + 500, i2[:5], l2[:5])  # shipped but never flushed: not drained ...
    srv.close()                                       # ... when the server goes away
    with pytest.raises(B.PPError) as e:
        b.collect(block=True)
    assert e.value.code == -7
    with pytest.raises(B.PPError):
        b.submit(s2[:1], e2[:1], i2[:1], l2[:1])
    b.close()


def test_ipc_symbols_are_exported():
    """Every function include/pp_ipc.h declares is exported by the library and bound in ipc.py."""
    import re
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    hdr = re.sub(r"/\*.*?\*/", "", open(os.path.join(root, "include", "pp_ipc.h")).read(), flags=re.S)
    declared = set(re.findall(r"\b(pp_ipc_[a-z_]+)\s*\(", hdr))
    lib = B.load_library()
    for s in declared:
        assert hasattr(lib, s), s
    assert declared == set(ipc.EXPORTS)


def _stuck_client_main(name, q):
    """Ships work whose hits overflow its hit ring many times over, reads nothing, reports its pid and waits to be
    killed (jobs die at their memory limit)."""
    import time
    src, ev, sid, ln = _sources(7, 4, 50)
    c = ipc.IpcClient(name)
    c.submit(src, ev, sid, ln)
    c.flush()
    q.put(os.getpid())
    time.sleep(600)


def test_a_killed_client_with_a_full_hit_ring_does_not_wedge_the_server():
    """a client that dies without closing (SIGKILL) while its hit ring is full used to stall the dispatch
    thread for ever.  Its hits are parked, the others are served meanwhile, and once its process is gone the server
    drops them and hands the slot out again."""
    import signal
    import time
    name = f"/pp_ipc_test_{os.getpid()}_kill"
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    # hit ring of 8 hits; every source echoes 40 hits: 200 sources -> 8000 hits against a ring of 8
    with ipc.IpcServer(None, name, max_clients=2, hit_ring_bytes=32 * 8, backend=echo_backend(40)) as srv:
        p = ctx.Process(target=_stuck_client_main, args=(name, q))
        p.start()
        pid = q.get(timeout=60)
        b = ipc.IpcClient(name)
        s2, e2, i2, l2 = _sources(1, 3, 20)
        t0 = time.time()
        b.submit(s2, e2, i2, l2)
        got = b.collect_all()                       # served although the other client's ring is full and unread
        assert len(got) == 40 * len(e2) and time.time() - t0 < 20
        assert set(np.unique(got["event_id"])) == set(np.unique(e2))
        os.kill(pid, signal.SIGKILL)
        p.join(timeout=30)
        c = None
        for _ in range(400):                        # the dead client's slot comes back
            try:
                c = ipc.IpcClient(name)
                break
            except B.PPError as e:
                assert e.code == -2
                time.sleep(0.01)
        assert c is not None, "the slot of the killed client was never recycled"
        s3, e3, i3, l3 = _sources(2, 2, 5)
        c.submit(s3, e3 + np.uint32(9000), i3, l3)
        assert len(c.collect_all()) == 40 * len(e3)
        st = srv.stats()
        assert st["error"] == 0 and st["clients_dropped"] == 1 and st["hits_dropped"] > 0 and st["hits_unrouted"] == 0
        b.close(), c.close()


def test_owner_table_and_slots_stay_bounded_while_the_server_never_runs_dry():
    """in steady state the server as a whole never runs dry.  One client keeps a block in the
    server at all times (shipped, never flushed by itself) while others come and go: their events must leave the
    owner table when their blocks complete, and their slots must be handed out again."""
    import time
    name = f"/pp_ipc_test_{os.getpid()}_busy"
    with ipc.IpcServer(None, name, max_clients=2, backend=echo_backend()) as srv:
        keep = ipc.IpcClient(name)
        sk, ek, ik, lk = _sources(9, 2, 5)
        n_keep = 0
        for round_ in range(12):
            keep.submit(sk, ek + np.uint32(50000 + 10 * round_), ik, lk)   # keeps the server from running dry
            n_keep += len(ek)
            c = None
            for _ in range(400):
                try:
                    c = ipc.IpcClient(name)
                    break
                except B.PPError as e:
                    assert e.code == -2
                    time.sleep(0.005)
            assert c is not None, f"round {round_}: slot not recycled while another client keeps the server busy"
            src, ev, sid, ln = _sources(round_ % 5, 30, 3)
            ev = ev + np.uint32(100000 * (round_ + 1))
            c.submit(src, ev, sid, ln)
            got = np.sort(c.collect_all(), order=["event_id", "source_id"])   # its flush also launches keep's block
            assert np.array_equal(got, _expected(src, ev, sid, ln))
            c.close()
            st = srv.stats()
            # at most: this round's 30 events (about to be forgotten) + the keeper's outstanding events
            assert st["events_tracked"] <= 30 + 2 * (round_ + 1), st
        assert len(keep.collect_all()) == n_keep
        for _ in range(200):
            if srv.stats()["events_tracked"] == 0:
                break
            time.sleep(0.005)
        st = srv.stats()
        assert st["events_tracked"] == 0 and st["error"] == 0 and st["clients_attached"] == 2
        keep.close()


def test_null_source_ids_do_not_collide_across_submits():
    """with source_ids == NULL two blocks of one event must not reuse ids 0..n-1 (identical Philox
    streams): the client's running record number is used."""
    name = f"/pp_ipc_test_{os.getpid()}_null"
    with ipc.IpcServer(None, name, max_clients=1, backend=echo_backend()) as srv:
        with ipc.IpcClient(name) as c:
            src, ev, sid, ln = _sources(0, 1, 20)
            c.submit(src[:10], ev[:10], None, ln[:10])
            c.submit(src[10:], ev[10:], None, ln[10:])
            got = c.collect_all()
        assert len(got) == 20 and len(np.unique(got["source_id"])) == 20
        assert srv.stats()["error"] == 0


def test_a_block_shipped_to_an_idle_server_is_never_declared_complete_before_it_ran():
    """Regression (round-2 advice): the dispatch thread asked the back end "anything left?" (drained), and only
    afterwards looked at how many sources had been handed over.  A block that arrived in between -- on an idle server,
    with the dispatch thread preempted -- was then taken for complete: its client saw "drained" without hits, and the
    hits turned up later with no owner.  The echo back end's empty-handed collect is made slow here, so that nearly
    every block lands inside that window; completion must follow the back end's completed count alone."""
    name = f"/pp_ipc_test_{os.getpid()}_idle"
    be = echo_backend()
    _echo_lib().echo_set_collect_delay_us(be, 3000)
    with ipc.IpcServer(None, name, max_clients=2, backend=be) as srv:
        total = 0
        for it in range(25):
            with ipc.IpcClient(name) as c:
                src, ev, sid, ln = _sources(it % 7, 3, 5)
                ev = ev + np.uint32(10000 * it)
                c.submit(src, ev, sid, ln)
                got = np.sort(c.collect_all(), order=["event_id", "source_id"])
                assert np.array_equal(got, _expected(src, ev, sid, ln)), f"iteration {it}: {len(got)} of {len(ev)} hits"
                total += len(ev)
        st = srv.stats()
        assert st["error"] == 0 and st["hits_unrouted"] == 0 and st["hits_routed"] == total


def test_a_block_of_one_source_events_with_interleaved_ids():
    """A block whose sources all belong to different events, some ids recurring out of order within the block: every
    id is announced once (the owner count per block is 1 however often the id recurs), all hits are routed, and the
    owner table empties.  (Round-2 advice: the ids are de-duplicated by sort + unique outside the routing lock.)"""
    import time
    name = f"/pp_ipc_test_{os.getpid()}_ids"
    with ipc.IpcServer(None, name, max_clients=1, backend=echo_backend()) as srv:
        with ipc.IpcClient(name) as c:
            n = 6000
            src, _, _, ln = _sources(3, n, 1)
            ev = (np.arange(n) % 4500 * 7 + 20000).astype(np.uint32)   # 4500 distinct ids, 1500 of them twice, far apart
            sid = (np.arange(n) // 4500).astype(np.uint32)
            c.submit(src, ev, sid, ln)
            got = np.sort(c.collect_all(), order=["event_id", "source_id"])
            assert np.array_equal(got, _expected(src, ev, sid, ln))
        for _ in range(200):
            if srv.stats()["events_tracked"] == 0:
                break
            time.sleep(0.005)
        st = srv.stats()
        assert st["events_tracked"] == 0 and st["hits_unrouted"] == 0 and st["hits_routed"] == n and st["error"] == 0


def test_a_block_the_back_end_refuses_fails_its_client_only():
    """What the client-side checks cannot judge (a photon count beyond 32 bits at the server's light yield, say) is
    refused by the back end.  That used to stop the server for everybody (round-2 advice); now the refused block is
    dropped, its client gets the back end's code from every later call, the others are served, and the slot comes
    back once the failed client has closed."""
    import ctypes as C
    import time
    from paper_2405_05700_b200 import multi
    be = multi.Backend()
    C.memmove(C.byref(be), C.c_void_p(echo_backend()), C.sizeof(multi.Backend))
    SUBMIT = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_uint32), C.c_void_p, C.c_size_t)
    real = SUBMIT(be.submit)

    def picky(ctx, s, ln, ev, sid, n):
        if any(ev[i] == 777 for i in range(n)):
            return -4
        return real(ctx, s, ln, ev, sid, n)

    keep = SUBMIT(picky)
    be.submit = C.cast(keep, C.c_void_p).value
    name = f"/pp_ipc_test_{os.getpid()}_refuse"
    with ipc.IpcServer(None, name, max_clients=2, backend=C.addressof(be)) as srv:
        a, b = ipc.IpcClient(name), ipc.IpcClient(name)
        sa, ea, ia, la = _sources(0, 2, 4)
        a.submit(sa, ea, ia, la)
        assert len(a.collect_all()) == len(ea)             # a good block first: A works
        a.submit(sa, np.full(len(ea), 777, np.uint32), ia, la)
        with pytest.raises(B.PPError) as e:
            a.collect_all()
        assert e.value.code == -4
        with pytest.raises(B.PPError) as e:
            a.submit(sa, ea + np.uint32(50), ia, la)
        assert e.value.code == -4
        sb, eb, ib, lb = _sources(1, 5, 6)
        b.submit(sb, eb, ib, lb)                           # B is served as if nothing had happened
        assert np.array_equal(np.sort(b.collect_all(), order=["event_id", "source_id"]), _expected(sb, eb, ib, lb))
        st = srv.stats()
        assert st["error"] == 0 and st["clients_failed"] == 1 and st["hits_unrouted"] == 0
        a.close()
        c = None
        for _ in range(400):                               # A's slot is handed out again
            try:
                c = ipc.IpcClient(name)
                break
            except B.PPError as e2:
                assert e2.code == -2
                time.sleep(0.005)
        assert c is not None
        c.submit(sa, ea + np.uint32(900), ia, la)
        assert len(c.collect_all()) == len(ea)
        assert srv.stats()["events_tracked"] == 0 or time.sleep(0.2) or srv.stats()["events_tracked"] == 0
        b.close(), c.close()
