"""The multi-process front end on the GPU (include/pp_ipc.h, NEXT-3): client processes ship blocks of C2's light sources
to one server process that owns the propagator; every client gets exactly the hits of its own events, and their
union is the hit list of a single-process run (the results contract of pp.h)."""
import multiprocessing as mp
import os

import numpy as np
import pytest

from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import ipc
from paper_2405_05700_b200 import workloads as W

from oracle import oracle as O

from gpu_util import KEY, compare_hits, sort_hits

pytestmark = pytest.mark.gpu
N_EVENTS = 120


def _case():
    src = W.sources_c2(n_events=N_EVENTS)
    order = np.argsort(src.event_id, kind="stable")
    return src.src[order], src.event_id[order], src.source_id[order]


def _client_main(name, client, n_clients, block, q):
    try:
        s, ev, sid = _case()
        mine = (ev % n_clients) == client
        s, ev, sid = s[mine], ev[mine], sid[mine]
        got = []
        with ipc.IpcClient(name) as c:
            for a in range(0, len(ev), block):
                c.submit(s[a:a + block], ev[a:a + block], sid[a:a + block])
                h = c.collect(block=False)
                if len(h):
                    got.append(h.copy())
            got.append(c.collect_all())
        q.put((client, np.concatenate(got).tobytes()))
    except Exception as e:  # pragma: no cover
        q.put((client, repr(e)))


@pytest.mark.parametrize("n_clients,ring_kib", [(1, 4096), (4, 4096), (8, 64)])
def test_clients_share_one_gpu_server(n_clients, ring_kib):
    geo, ice = W.geometry_full(radius=0.6), W.ice_layered()
    s, ev, sid = _case()
    with B.Propagator(geo, ice, seed=12, launch_photons_target=2 * 10 ** 6) as p:
        ref = sort_hits(p.run(s, ev, sid))
        n_ref_launches = p.stats().launches
    assert len(ref) > 2000 and n_ref_launches >= 3
    if n_clients == 4:
        # ... and that single-process run is what the oracle computes (once is enough: the other cases compare with
        # the same list, bit for bit)
        ref_o = O.propagate(geo, ice, W.Sources(s, ev, sid), seed=12)
        c = compare_hits(ref, ref_o.hits, ref_o.photons)
        assert c["frac_hit"] >= 0.99 and c["frac_all"] >= 0.999, c
    name = f"/pp_ipc_gpu_{os.getpid()}_{n_clients}"
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    with B.Propagator(geo, ice, seed=12, launch_photons_target=2 * 10 ** 6) as p:
        with ipc.IpcServer(p, name, max_clients=n_clients, source_ring_bytes=ring_kib * 1024,
                           hit_ring_bytes=ring_kib * 1024) as srv:
            procs = [ctx.Process(target=_client_main, args=(name, c, n_clients, 1500, q)) for c in range(n_clients)]
            for pr in procs:
                pr.start()
            res = dict(q.get(timeout=300) for _ in procs)
            for pr in procs:
                pr.join(timeout=60)
            st = srv.stats()
        pst = p.stats()
    assert st["error"] == 0 and st["hits_unrouted"] == 0 and st["sources_ingested"] == len(ev)
    assert pst.photons_done == pst.photons_submitted and pst.photons_aborted == 0
    parts = []
    for c in range(n_clients):
        assert isinstance(res[c], bytes), res[c]
        h = np.frombuffer(res[c], dtype=B.HIT_DTYPE)
        assert np.all(h["event_id"] % n_clients == c)  # only its own events
        parts.append(h)
    allh = np.sort(np.concatenate(parts), order=KEY)
    assert st["hits_routed"] == len(allh) == len(ref)
    assert np.array_equal(allh, ref)


def test_completion_is_tracked_source_by_source():
    """pp_stats.sources_completed: monotone, in submit order, equal to sources_submitted once drained; and through
    the front end a client drains while another client's block sits unlaunched in the server (steady state)."""
    import time
    geo, ice = W.geometry_full(radius=0.6), W.ice_layered()
    s, ev, sid = _case()
    with B.Propagator(geo, ice, seed=12, launch_photons_target=10 ** 9) as p:   # target never reached: flush decides
        assert p.stats().sources_completed == 0
        p.submit(s[:1000], ev[:1000], sid[:1000])
        p.flush()
        h1 = p.collect_all()
        st = p.stats()
        assert st.sources_completed == st.sources_submitted == 1000
        p.submit(s[1000:1200], ev[1000:1200], sid[1000:1200])       # queued, not flushed: below target / 8
        time.sleep(0.1)
        st = p.stats()
        assert st.sources_submitted == 1200 and st.sources_completed == 1000 and st.photons_done < st.photons_submitted
        name = f"/pp_ipc_gpu_{os.getpid()}_own"
        p.collect_all()
        assert p.stats().sources_completed == 1200
        with ipc.IpcServer(p, name, max_clients=2) as srv:
            a, b = ipc.IpcClient(name), ipc.IpcClient(name)
            ma, mb = (ev % 2) == 0, (ev % 2) == 1
            a.submit(s[ma][:3000], ev[ma][:3000], sid[ma][:3000])
            ha = a.collect_all()                                     # A's flush launches A's block
            assert len(ha) > 0 and np.all(ha["event_id"] % 2 == 0)
            b.submit(s[mb][:300], ev[mb][:300], sid[mb][:300])       # B's block stays queued in the server
            time.sleep(0.1)
            assert len(a.collect(block=True)) == 0                   # A is drained although the server is not
            pst = p.stats()
            assert pst.photons_done < pst.photons_submitted
            hb = b.collect_all()
            assert len(hb) > 0 and np.all(hb["event_id"] % 2 == 1)
            assert srv.stats()["hits_unrouted"] == 0
            a.close(), b.close()
