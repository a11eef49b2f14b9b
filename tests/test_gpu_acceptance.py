"""GPU parity of the DOM acceptance (NEXT-1, R-17) against the oracle, through the C ABI."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import workloads as W

from gpu_util import compare_hits, sort_hits, total_photons, flights_agree

pytestmark = pytest.mark.gpu
COEF = W.ACCEPTANCE_COEF


def run(geo, ice, src, seed, mode, coef=COEF, **kw):
    with B.Propagator(geo, ice, seed=seed, **kw) as p:
        p.set_acceptance(mode, coef)
        hits = sort_hits(p.run(src.src, src.event_id, src.source_id))
        st = p.stats()
    return hits, st


@pytest.mark.parametrize("mode", ["probabilistic", "weighted"])
def test_layered_oversized_doms_per_photon(mode):
    """Full detector with oversized DOMs (many hits), layered ice: same accepted photons, DOMs, times and weights."""
    geo, ice = W.geometry_full(radius=1.0), W.ice_layered()
    src = W.sources_c1().subset(slice(0, 40))
    src.src[:, 7] = 5.0  # 5e4 photons per cascade
    n = total_photons(src, ice)
    hits, st = run(geo, ice, src, 5, mode, launch_photons_target=700000)
    ref = O.propagate(geo, ice, src, seed=5, acceptance_mode=mode, acceptance_coef=COEF)
    assert st.photons_done == n == ref.photons
    assert st.photons_done == st.photons_absorbed + st.photons_hit + st.photons_aborted + st.photons_rejected
    assert flights_agree(st.flights, ref.flights)
    assert ref.hit > 300
    assert abs(st.photons_hit - ref.hit) <= 2 and abs(st.photons_rejected - ref.rejected) <= 2
    c = compare_hits(hits, ref.hits, n)
    assert c["frac_all"] >= 0.999 and c["frac_hit"] >= 0.97, c
    # weights of the common hits
    kr = {(int(a), int(b), int(c_)): float(w) for a, b, c_, w in
          zip(ref.hits["event_id"], ref.hits["source_id"], ref.hits["photon_idx"], ref.hits["weight"])}
    dw = [abs(float(h["weight"]) - kr[k]) for h in hits
          for k in [(int(h["event_id"]), int(h["source_id"]), int(h["photon_idx"]))] if k in kr]
    assert len(dw) >= 0.97 * len(hits)
    if mode == "weighted":
        assert max(dw) <= 2e-5, max(dw)  # p(eta) in fp32 with eta from an fp32 trajectory
        assert 0.0 < hits["weight"].min() and hits["weight"].max() <= 1.0 and hits["weight"].std() > 0.05
    else:
        assert np.all(hits["weight"] == 1.0)


def test_closed_forms_on_the_gpu():
    """The oracle's own pins, run on the CUDA path: photons born inside a DOM, and a pencil beam from the side."""
    ice = W.ice_homogeneous()
    geo = W.Geometry(xyz=np.array([[0.0, 0.0, 0.0]], np.float32), radius=W.DOM_RADIUS)
    n = 400000
    for axis_z, p_exp in ((1.0, 0.8111), (-1.0, 0.0587)):
        src = W.pencil_beam([0.01, 0.0, 0.02], [0, 0, axis_z], float(n))
        hits, st = run(geo, ice, src, 3, "probabilistic", flags=B.FLAG_BRUTE_FORCE_DOMS)
        eta = axis_z * float(np.float32(ice.cos_cherenkov))
        p = min(1.0, max(0.0, 0.35 + 0.5 * eta + 0.15 * eta * eta))
        assert p == pytest.approx(p_exp, abs=2e-4)
        assert st.photons_hit + st.photons_rejected == n
        assert st.photons_hit / n == pytest.approx(p, abs=4 * math.sqrt(p * (1 - p) / n))
        hits2, st2 = run(geo, ice, src, 3, "weighted", flags=B.FLAG_BRUTE_FORCE_DOMS)
        assert st2.photons_hit == n and np.allclose(hits2["weight"], p, atol=2e-6)
    dist = 20.0
    geo = W.Geometry(xyz=np.array([[dist, 0.0, 0.0]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous(scat_len=1.0e30, cos_cherenkov=1.0)
    src = W.pencil_beam([0, 0, 0], [1, 0, 0], float(n))
    hits, st = run(geo, ice, src, 11, "probabilistic", flags=B.FLAG_BRUTE_FORCE_DOMS)
    e = math.exp(-(dist - float(np.float32(W.DOM_RADIUS))) / 100.0) * 0.35
    assert st.photons_hit / n == pytest.approx(e, abs=4 * math.sqrt(e * (1 - e) / n))


def test_off_mode_is_the_default_and_batching_invariance():
    """Acceptance off = the acceptance-free path bit for bit; with acceptance on, the hit multiset does not depend on
    the launch size or on a tiny hit ring (deferred photons are replayed together with their acceptance draw)."""
    geo, ice = W.geometry_full(radius=1.0), W.ice_layered()
    src = W.sources_c1().subset(slice(0, 20))
    src.src[:, 7] = 5.0  # 1e6 photons in all
    with B.Propagator(geo, ice, seed=2) as p:
        base = sort_hits(p.run(src.src, src.event_id, src.source_id))
    off, _ = run(geo, ice, src, 2, "off", ())
    assert np.array_equal(base, off) and np.all(off["weight"] == 1.0)
    a, st_a = run(geo, ice, src, 2, "probabilistic")
    b, st_b = run(geo, ice, src, 2, "probabilistic", launch_photons_target=200000, hit_ring_bytes=2 * 32 * 32)
    assert st_b.relaunches > 0 and st_b.launches > st_a.launches
    assert np.array_equal(a, b)
    assert st_a.photons_rejected == st_b.photons_rejected and st_a.flights == st_b.flights
    assert 0 < len(a) < len(base)
    # the accepted hits are a subset of the acceptance-free hits, same DOM and time
    kb = {(int(h["event_id"]), int(h["source_id"]), int(h["photon_idx"])): (int(h["dom_id"]), float(h["time_ns"])) for h in base}
    for h in a:
        assert kb[(int(h["event_id"]), int(h["source_id"]), int(h["photon_idx"]))] == (int(h["dom_id"]), float(h["time_ns"]))


def test_set_acceptance_argument_checks():
    geo, ice = W.geometry_single_string(), W.ice_homogeneous()
    with B.Propagator(geo, ice, seed=0) as p:
        for mode, coef in (("probabilistic", ()), ("weighted", [0.1] * 9), ("probabilistic", [float("nan")])):
            with pytest.raises(B.PPError) as e:
                p.set_acceptance(mode, coef)
            assert e.value.code == -1
        p.set_acceptance("off", ())
        p.set_acceptance("weighted", [0.5])
