"""-m gpu: several devices behind one server (include/pp_multi.h, NEXT-4).  Only one GPU is here, so the "devices"
are two handles on cuda:0 -- the dispatcher, the merged collect and the results contract are what is tested: the
multiset of hits is bit-identical to one handle's, whatever the dealing."""
import numpy as np
import pytest

from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import multi
from paper_2405_05700_b200 import workloads as W

from oracle import oracle as O

from gpu_util import compare_hits, gpu_run, sort_hits, total_photons

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
    ref_o = O.propagate(geo, ice, src, seed=3)  # what one handle gives is what the oracle computes
    c = compare_hits(ref, ref_o.hits, ref_o.photons)
    assert c["frac_hit"] >= 0.99 and c["frac_all"] >= 0.999, c
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


def test_two_physical_devices_behind_one_front():
    """NEXT-4 on real hardware: one handle per device ordinal.  Needs two GPUs (the round's boxes have one: skipped
    there).  Checks what a single device cannot: that ordinal 0 can be named while another device is current
    (PP_FLAG_DEVICE_ORDINAL), that pp_create leaves the caller's current device alone, and that hits do not depend
    on which device ran a source."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    geo, ice, src = _job()
    n_ph = total_photons(src, ice)
    ref, _ = gpu_run(geo, ice, src, 3)
    with torch.cuda.device(1):
        with B.Propagator(geo, ice, seed=3, device=0) as p:          # device 0 named while device 1 is current
            assert p.device.index == 0 and torch.cuda.current_device() == 1
            assert np.array_equal(sort_hits(p.run(src.src, src.event_id, src.source_id)), ref)
        with multi.MultiFront.over_devices(geo, ice, [0, 1], seed=3, launch_photons_target=max(1, n_ph // 8),
                                           deal_photons=n_ph // 8) as m:
            assert torch.cuda.current_device() == 1
            hits = sort_hits(m.run(src.src, src.event_id, src.source_id))
            st = m.stats()
    assert np.array_equal(hits, ref)
    assert min(st["batches"]) >= 1 and sum(st["photons"]) == n_ph, st


def test_create_leaves_the_current_device_alone_and_honours_ordinal_zero():
    import torch
    geo, ice, src = _job()
    before = torch.cuda.current_device()
    with B.Propagator(geo, ice, seed=3, device=0, use_torch_memory=False) as p:   # library-owned memory and streams
        assert torch.cuda.current_device() == before and p.device.index == 0
        sub = src.subset(slice(0, 500))
        hits = sort_hits(p.run(sub.src, sub.event_id, sub.source_id))
    ref, _ = gpu_run(geo, ice, src.subset(slice(0, 500)), 3)
    assert np.array_equal(hits, ref)
