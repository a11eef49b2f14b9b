"""-m gpu: several devices behind one server (include/pp_multi.h, NEXT-4).  Only one GPU is here, so the "devices"
are two handles on cuda:0 -- the dispatcher, the merged collect and the results contract are what is tested: the
multiset of hits is bit-identical to one handle's, whatever the dealing."""
import numpy as np
import pytest

from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import multi
from paper_2405_05700_b200 import workloads as W

from gpu_util import gpu_run, sort_hits, total_photons

pytestmark = pytest.mark.gpu


def _job():
    geo, ice = W.geometry_full(radius=1.0), W.ice_layered()
    src = W.sources_c2(seed=2, n_events=40)
    return geo, ice, src


def test_two_handles_behind_one_front_give_one_handles_hits():
    geo, ice, src = _job()
    n_ph = total_photons(src, ice)
    ref, st_ref = gpu_run(geo, ice, src, 3)
    assert len(ref) > 1000
    for deal in (n_ph // 7, n_ph // 2, 10 ** 9):
        with multi.MultiFront.over_devices(geo, ice, [0, 0], seed=3, launch_photons_target=max(1, n_ph // 7),
                                           deal_photons=deal) as m:
            got = []
            for a in range(0, len(src), 5000):                       # blocks that do not line up with the batches
                m.submit(src.src[a:a + 5000], src.event_id[a:a + 5000], src.source_id[a:a + 5000])
                got.append(m.collect(block=False))
            got.append(m.collect_all())
            st = m.stats()
        hits = sort_hits(np.concatenate(got))
        assert np.array_equal(hits, ref), deal                        # bit for bit: ids, DOMs, times, weights
        assert st["sources_completed"] == len(src) and sum(st["photons"]) == n_ph
        if deal < n_ph // 2:
            assert min(st["batches"]) >= 1, st                        # both "devices" worked


def test_front_with_null_ids_matches_explicit_running_numbers():
    geo, ice, src = _job()
    src = src.subset(slice(0, 3000))
    ids = np.arange(len(src), dtype=np.uint32)
    ref, _ = gpu_run(geo, ice, W.Sources(src.src, src.event_id, ids), 5)
    with multi.MultiFront.over_devices(geo, ice, [0, 0], seed=5, deal_photons=total_photons(src, ice) // 5) as m:
        m.submit(src.src[:1000], src.event_id[:1000], None)
        m.submit(src.src[1000:], src.event_id[1000:], None)
        hits = sort_hits(m.collect_all())
    assert np.array_equal(hits, ref)
