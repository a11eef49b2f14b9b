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

from gpu_util import KEY, sort_hits

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
