"""-m gpu: the batching server (a1), the bounded hit ring with its replay protocol (a8) and hit
streaming (a9).  Results contract (include/pp.h): the multiset of hits depends only on (geometry, ice,
seed, sources), never on batching, thread count, launch size or ring size -- bit for bit."""
import threading

import numpy as np
import pytest

from oracle import oracle as O
from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import workloads as W

from gpu_util import compare_hits, gpu_run, gpu_run_resident, sort_hits, total_photons

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def case():
    geo, ice = W.geometry_full(radius=1.5), W.ice_layered()
    src = W.sources_c2(seed=5, n_events=40)  # tiny + large cascades, several events
    src.src[:, 7] *= 3.0
    return geo, ice, src


@pytest.fixture(scope="module")
def reference_hits(case):
    geo, ice, src = case
    hits, st = gpu_run(geo, ice, src, 9)
    assert len(hits) > 2000
    return hits


@pytest.mark.parametrize("target", [10 ** 4, 123457, 10 ** 6, 10 ** 9])
def test_launch_size_invariance(case, reference_hits, target):
    geo, ice, src = case
    hits, st = gpu_run(geo, ice, src, 9, launch_photons_target=target)
    assert np.array_equal(hits, reference_hits)
    n = total_photons(src, ice)
    assert st.launches == -(-n // target)


def test_launch_that_starts_a_few_photons_into_a_source():
    """A launch whose first photon is the 8th of its source, with thousands of warps that get no work item: their
    (empty) photon range then sits just below 2^32 in launch-relative numbering, where "next photon + lane rank" wraps
    (regression: such warps once refilled themselves for ever)."""
    geo, ice = W.geometry_full(radius=2.0), W.ice_layered()
    src = W.sources_c1().subset(slice(0, 6))
    src.src[:, 7] = np.array([0.9993, 5.0, 0.0031, 2.0, 0.0007, 1.5], np.float32)  # 9993, 50000, 31, 20000, 7, 15000 photons
    ref, _ = gpu_run(geo, ice, src, 4)
    hits, st = gpu_run(geo, ice, src, 4, launch_photons_target=10000)  # launch 2 starts at photon 7 of source 1
    assert st.photons_done == total_photons(src, ice) and st.launches == -(-st.photons_done // 10000)
    assert len(ref) > 50 and np.array_equal(hits, ref)


def test_packed_records_equal_separate_arrays(case, reference_hits):
    """pp_submit_packed (one 48-byte record per source: what the multi-process front end hands over) gives the hits of
    pp_submit; bad records are rejected before anything is queued."""
    geo, ice, src = case
    rec = B.pack_records(src.src, src.event_id, src.source_id)
    with B.Propagator(geo, ice, seed=9) as p:
        for part in np.array_split(rec, 7):
            p.submit_packed(part)
        hits = sort_hits(p.collect_all())
        bad = rec[:3].copy()
        bad["src"][1, 3] = 2.0  # not a unit direction
        with pytest.raises(B.PPError):
            p.submit_packed(bad)
    assert np.array_equal(hits, reference_hits)


def test_resident_path_equals_server_path(case, reference_hits):
    geo, ice, src = case
    hits, _, st = gpu_run_resident(geo, ice, src, 9, launch_photons_target=300000)
    assert np.array_equal(hits, reference_hits)


@pytest.mark.parametrize("n_threads", [1, 2, 8, 16])
def test_thread_count_and_submit_order_invariance(case, reference_hits, n_threads):
    """1, 2, 4, 8, 16 client instances share one photon server."""
    geo, ice, src = case
    rng = np.random.default_rng(n_threads)
    order = rng.permutation(len(src))
    chunks = np.array_split(order, n_threads * 5)
    with B.Propagator(geo, ice, seed=9, launch_photons_target=200000, source_ring_bytes=48 * 4096) as p:
        def work(t):
            for c in chunks[t::n_threads]:
                p.submit(src.src[c], src.event_id[c], src.source_id[c])
        th = [threading.Thread(target=work, args=(t,)) for t in range(n_threads)]
        [x.start() for x in th]
        [x.join() for x in th]
        hits = sort_hits(p.collect_all())
        st = p.stats()
    assert np.array_equal(hits, reference_hits)
    assert st.source_ring_high_water <= 48 * 4096  # bounded host memory: the ring never outgrows its size


@pytest.mark.parametrize("ring_bytes", [64 * 1024, 2 * 32 * 40, 1 << 20])
def test_hit_ring_overflow_replay_protocol(case, reference_hits, ring_bytes):
    """C4's forced-tiny-cap variant: a hit ring far smaller than a launch's hits forces stop/replay
    relaunches; the hit list must not change and memory stays bounded."""
    geo, ice, src = case
    hits, st = gpu_run(geo, ice, src, 9, launch_photons_target=500000, hit_ring_bytes=ring_bytes)
    assert np.array_equal(hits, reference_hits)
    cap_hits = ring_bytes // 2 // 32
    if cap_hits < len(reference_hits) / 4:
        assert st.relaunches > 0
    assert st.hit_ring_high_water <= max(ring_bytes // 2, 32 * 32)
    n = total_photons(src, ice)
    assert st.photons_done == n == st.photons_absorbed + st.photons_hit
    assert st.photons_hit == len(hits)


def test_ring_overflow_with_unfetched_resume_items():
    """Hits so frequent (5 m DOMs) that a 32-hit ring fills up again before the warps have fetched the whole resume
    list of a relaunch: the unfetched items must be carried over to the next relaunch, not dropped."""
    geo, ice = W.geometry_full(radius=5.0), W.ice_layered()
    src = W.sources_c1().subset(slice(0, 8))
    src.src[:, 7] = 2.0  # 2e4 photons per cascade
    n = total_photons(src, ice)
    ref, st0 = gpu_run(geo, ice, src, 4)
    assert st0.relaunches == 0 and len(ref) > 5000
    hits, st = gpu_run(geo, ice, src, 4, launch_photons_target=10 ** 6, hit_ring_bytes=2 * 32 * 32)
    assert st.relaunches > 100
    assert st.photons_done == n == st.photons_absorbed + st.photons_hit and st.flights == st0.flights
    assert np.array_equal(hits, ref)


def test_streaming_collect_while_producing(case, reference_hits):
    """Hits of one event may arrive across several pp_collect calls; a consumer thread drains while
    producers are still submitting."""
    geo, ice, src = case
    got = []
    with B.Propagator(geo, ice, seed=9, launch_photons_target=100000) as p:
        done = threading.Event()

        def consume():
            while True:
                h = p.collect(cap=257, block=False)
                if len(h):
                    got.append(h.copy())
                elif done.is_set():
                    break
        th = threading.Thread(target=consume)
        th.start()
        for c in np.array_split(np.arange(len(src)), 50):
            p.submit(src.src[c], src.event_id[c], src.source_id[c])
        p.flush()
        rest = []
        while True:
            h = p.collect(cap=1000, block=True)
            if len(h) == 0:
                break
            rest.append(h.copy())
        done.set()
        th.join()
    allh = sort_hits(np.concatenate(got + rest))
    assert np.array_equal(allh, reference_hits)


def test_nonblocking_submit_reports_wouldblock():
    geo, ice = W.geometry_full(), W.ice_layered()
    src = W.sources_c3(3.0e9)  # a few huge cascades keep the GPU busy for a while
    with B.Propagator(geo, ice, seed=0, launch_photons_target=10 ** 9, source_ring_bytes=48 * 64,
                      flags=B.FLAG_NONBLOCKING_SUBMIT) as p:
        small = W.sources_c2(n_events=3)
        codes = []
        for k in range(200):
            try:
                p.submit(small.src[:32], small.event_id[:32], small.source_id[:32])
                codes.append(0)
            except B.PPError as e:
                codes.append(e.code)
        assert -5 in codes and 0 in codes
        with pytest.raises(B.PPError) as e:
            p.submit(small.src[:100], small.event_id[:100], small.source_id[:100])  # larger than the ring
        assert e.value.code == -2
        p.collect_all()


def test_c3_launch_size_sweep_same_hits():
    """C3 shape (1-100 TeV cascades cut at N photons): the launch size must not change the result."""
    geo, ice = W.geometry_full(), W.ice_layered()
    src = W.sources_c3(1.0e7)
    n = total_photons(src, ice)
    assert abs(n - 1.0e7) <= 100
    ref = None
    for target in (10 ** 5, 10 ** 6, 10 ** 7):
        hits, st = gpu_run(geo, ice, src, 3, launch_photons_target=target)
        assert st.photons_done == n
        if ref is None:
            ref = hits
        assert np.array_equal(hits, ref)
    o = O.propagate(geo, ice, src, seed=3, stride=8)
    c = compare_hits(ref[ref["photon_idx"] % 8 == 0], o.hits, o.photons)
    assert c["frac_all"] >= 0.999, c
    assert c["n_union"] > 10 and (1.0 - c["frac_hit"]) * c["n_union"] <= 2.0, c  # few hits: at most two outliers


def test_c4_extreme_event_bounded_memory():
    """C4: one 1e8 GeV bundle, 500 muons, ~5e9 photons, hit ring capped at 2 GB (never approached, as
    SURVEY 8(d) computes) -- and the same event with a 256 KiB ring (approached all the time).  Per-DOM hit
    counts and per-photon hits against the oracle on the 1e7-photon subsample photon_idx % 500 == 0."""
    import torch
    geo, ice, src = W.geometry_full(), W.ice_layered(), W.sources_c4()
    n = total_photons(src, ice)
    assert 4.9e9 < n < 5.1e9
    torch.cuda.synchronize()
    torch.cuda.reset_peak_memory_stats()
    mem_before = torch.cuda.memory_allocated()
    with B.Propagator(geo, ice, seed=0, launch_photons_target=5 * 10 ** 8, hit_ring_bytes=2 << 30,
                      source_ring_bytes=16 << 20) as p:
        ws = p.device_workspace_bytes
        hits = sort_hits(p.run(src.src, src.event_id, src.source_id))
        st = p.stats()
        peak = torch.cuda.max_memory_allocated()
    assert st.photons_done == n and st.photons_aborted == 0 and st.relaunches == 0
    assert peak - mem_before <= ws + (16 << 20)  # predictable peak device memory: the workspace is all there is
    assert st.hit_ring_high_water < (2 << 30) / 2
    hits_small, st2 = gpu_run(geo, ice, src, 0, launch_photons_target=5 * 10 ** 8, hit_ring_bytes=256 * 1024,
                              source_ring_bytes=16 << 20)
    assert st2.relaunches > 0
    assert np.array_equal(hits_small, hits)
    ref = O.propagate(geo, ice, src, seed=0, stride=500)
    assert 0.9e7 < ref.photons < 1.1e7
    sub = hits[hits["photon_idx"] % 500 == 0]
    c = compare_hits(sub, ref.hits, ref.photons)
    # ~100 hits in the subsample: too few for the 0.99 gate of the large samples (profiles/r02_parity.md)
    assert c["frac_all"] >= 0.999 and c["frac_hit"] >= 0.95, c
    dom_gpu = np.bincount(sub["dom_id"], minlength=geo.n_dom)
    dom_ref = np.bincount(ref.hits["dom_id"], minlength=geo.n_dom)
    assert np.abs(dom_gpu - dom_ref).sum() <= 0.05 * max(1, dom_ref.sum())


def test_null_source_ids_are_unique_across_calls():
    """one event shipped in two pp_submit calls with source_ids == NULL used to reuse ids 0..n-1, i.e. the
    same Philox streams twice (duplicated hits).  NULL now means the handle's running record number."""
    geo, ice = W.geometry_single_string(radius=2.0), W.ice_homogeneous()
    src = W.sources_c0(seed=0, n_photons=2.0e5, toward_string=True)
    two = np.concatenate([src.src, src.src])
    ev = np.zeros(2, np.uint32)
    with B.Propagator(geo, ice, seed=1) as p:
        p.submit(two[:1], ev[:1], None)
        p.submit(two[1:], ev[1:], None)          # the same cascade again, same event, second call
        h = p.collect_all()
        assert sorted(np.unique(h["source_id"])) == [0, 1]
        a, b = h[h["source_id"] == 0], h[h["source_id"] == 1]
        assert len(a) > 20 and len(b) > 20
        assert not np.array_equal(np.sort(a["photon_idx"]), np.sort(b["photon_idx"]))  # independent streams
        # explicit equal ids reproduce the collision the header warns about: identical hits twice
        p.submit(two[:1], ev[:1], np.array([7], np.uint32))
        p.submit(two[1:], ev[1:], np.array([7], np.uint32))
        h2 = p.collect_all()
        assert len(h2) % 2 == 0 and len(np.unique(h2["photon_idx"])) == len(h2) // 2
        # the resident path numbers on from the same count
        d = p.upload(two, ev, None)
        p.run_resident(*d)
        h3 = p.drain()
        assert sorted(np.unique(h3["source_id"])) == [4, 5]
