"""-m gpu: pp_run_resident_noalloc, the entry point for callers that cannot allocate device memory.

Who that is: a plug-in living inside a framework whose caching allocator already owns the device (a cudaMalloc beside
the pool fails, or starves the pool later); a latency-bound loop that cannot let cudaMalloc / cudaFree wait for the
kernels running on the device; a thread in a process where a stream capture in the default mode is under way (cudaMalloc
is refused there).  For them the library keeps the launch's scratch -- expanded sources, prefix sums, tile table,
counters -- in one fixed 512 KiB device array inside libpp.so, so the call is limited to PP_NOALLOC_MAX_SOURCES sources
and PP_NOALLOC_MAX_PHOTONS photons, and every call on a device shares that array.

What is checked: the hits are those of the existing resident path (pp_run_resident) for the same handle and sources,
bit for bit -- the tolerance the batching tests use for "same photons, other launch layout" -- on two calls in a row
with different batches (the second, smaller one finds the first one's leftovers in the array), then on the first batch
again; and that oversized calls are refused with an error that names the limit, leaving the entry point usable.

This file sorts last on purpose: under `pytest -x` a failure here must not hide any other test."""
import numpy as np
import pytest

from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import workloads as W

from gpu_util import sort_hits, total_photons

pytestmark = pytest.mark.gpu

SEED = 11


def _batches():
    ice = W.ice_layered()
    a = W.sources_c2(seed=5, n_events=40).subset(slice(0, 3500))  # several events, tiny and large cascades
    b = W.sources_c1().subset(slice(0, 37))                       # fewer, far brighter sources, other ids
    b.src[:, 7] *= 0.008
    b.event_id = b.event_id + np.uint32(1000)
    for s in (a, b):
        assert len(s) <= B.NOALLOC_MAX_SOURCES and 10 ** 5 < total_photons(s, ice) <= B.NOALLOC_MAX_PHOTONS
    return ice, a, b


def _existing_path(p, src):
    ph, _, _ = p.run_resident(*p.upload(src.src, src.event_id, src.source_id))
    return sort_hits(p.drain()), ph


def _no_alloc_path(p, torch, src, d_hits):
    """d_hits is made by the caller (here: the test) before the call; the library itself allocates nothing."""
    n_hits, ph = p.run_resident_noalloc(*p.upload(src.src, src.event_id, src.source_id), d_hits)
    return sort_hits(d_hits[: n_hits * B.HIT_DTYPE.itemsize].cpu().numpy().view(B.HIT_DTYPE)), ph


def test_no_alloc_entry_point_matches_the_resident_path_on_consecutive_calls():
    import torch
    geo = W.geometry_full(radius=1.5)  # large DOMs: thousands of hits from a few million photons
    ice, a, b = _batches()
    with B.Propagator(geo, ice, seed=SEED) as p:
        ref_a, ph_a = _existing_path(p, a)
        ref_b, ph_b = _existing_path(p, b)
        assert len(ref_a) > 300 and len(ref_b) > 300
        d_hits = torch.empty(max(len(ref_a), len(ref_b)) * B.HIT_DTYPE.itemsize, dtype=torch.uint8, device=p.device)
        st0 = p.stats()
        for src, ref, ph_ref in ((a, ref_a, ph_a), (b, ref_b, ph_b), (a, ref_a, ph_a)):  # calls in a row, no reset between
            d_hits.fill_(0xFF)
            hits, ph = _no_alloc_path(p, torch, src, d_hits)
            assert ph == ph_ref == total_photons(src, ice)
            assert np.array_equal(hits, ref)
        st1 = p.stats()
        assert (st1.launches, st1.photons_done, st1.hits_collected) == (st0.launches, st0.photons_done, st0.hits_collected), \
            "the handle's server state is not touched by the no-alloc call"


def test_no_alloc_entry_point_refuses_what_does_not_fit_and_stays_usable():
    import torch
    geo = W.geometry_full(radius=1.5)
    ice, a, b = _batches()
    with B.Propagator(geo, ice, seed=SEED) as p:
        ref_b, _ = _existing_path(p, b)
        d_hits = torch.empty(len(ref_b) * B.HIT_DTYPE.itemsize, dtype=torch.uint8, device=p.device)
        # too many sources (known on the host: refused before any kernel runs)
        many = W.sources_c2(seed=5, n_events=40).subset(slice(0, B.NOALLOC_MAX_SOURCES + 1))
        with pytest.raises(B.PPError) as ei:
            _no_alloc_path(p, torch, many, d_hits)
        assert ei.value.code == -2 and "PP_NOALLOC_MAX_SOURCES" in str(ei.value)
        # too many photons (known only after the expansion kernel has counted them)
        bright = W.sources_c1().subset(slice(0, 37))
        assert total_photons(bright, ice) > B.NOALLOC_MAX_PHOTONS
        with pytest.raises(B.PPError) as ei:
            _no_alloc_path(p, torch, bright, d_hits)
        assert ei.value.code == -2 and "PP_NOALLOC_MAX_PHOTONS" in str(ei.value)
        # more hits than the caller's buffer holds
        with pytest.raises(B.PPError) as ei:
            _no_alloc_path(p, torch, b, d_hits[: 64 * B.HIT_DTYPE.itemsize])
        assert ei.value.code == -2 and "hit buffer too small" in str(ei.value)
        # none of that poisons the handle or the shared array
        hits, _ = _no_alloc_path(p, torch, b, d_hits)
        assert np.array_equal(hits, ref_b)
