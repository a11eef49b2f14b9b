"""GPU parity of the extended (track-segment) sources (NEXT-2, R-18) against the oracle, through the C ABI."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import workloads as W

from gpu_util import compare_hits, sort_hits, total_photons, flights_agree

pytestmark = pytest.mark.gpu
C = W.C_VACUUM
V = C / float(np.float32(W.N_GROUP))


def run(geo, ice, src, seed, lengths, acceptance=None, **kw):
    with B.Propagator(geo, ice, seed=seed, **kw) as p:
        if acceptance:
            p.set_acceptance(acceptance, W.ACCEPTANCE_COEF)
        hits = sort_hits(p.run(src.src, src.event_id, src.source_id, lengths))
        st = p.stats()
    return hits, st


def test_track_with_cascades_per_photon():
    """A muon as 100 track segments of 10 m plus 20 point cascades, full detector with oversized DOMs, layered ice."""
    geo, ice = W.geometry_full(radius=1.0), W.ice_layered()
    src = W.sources_track()
    src.src[:, 7] = np.minimum(src.src[:, 7], 2.0) + 1.0
    n = total_photons(src, ice)
    assert n > 1.0e6
    hits, st = run(geo, ice, src, 6, src.length, launch_photons_target=400000)
    ref = O.propagate(geo, ice, src, seed=6)
    assert st.photons_done == n == ref.photons and st.launches >= 3
    assert flights_agree(st.flights, ref.flights)
    assert ref.hit > 1000 and abs(st.photons_hit - ref.hit) <= 2
    c = compare_hits(hits, ref.hits, n)
    assert c["frac_all"] >= 0.999 and c["frac_hit"] >= 0.97, c
    # the lengths matter: the same list as point sources gives a different hit list
    pts, _ = run(geo, ice, src, 6, None, launch_photons_target=400000)
    assert not np.array_equal(pts, hits)
    # ... and lengths of zero are the point sources bit for bit
    zer, _ = run(geo, ice, src, 6, np.zeros(len(src), np.float32), launch_photons_target=400000)
    assert np.array_equal(pts, zer)
    # batching invariance with segments on (a launch of point sources only next to launches with segments)
    one, st1 = run(geo, ice, src, 6, src.length, launch_photons_target=10 ** 8)
    assert st1.launches == 1 and np.array_equal(one, hits)


def test_closed_form_on_the_gpu():
    """The oracle's pin: beam along the axis from a 20 m segment at a DOM 30 m ahead, scattering off."""
    lam, L, D, n = 100.0, 20.0, 30.0, 400000
    R = float(np.float32(W.DOM_RADIUS))
    geo = W.Geometry(xyz=np.array([[0.0, 0.0, D]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous(scat_len=1.0e30, cos_cherenkov=1.0)
    src = W.pencil_beam([0, 0, 0], [0, 0, 1], float(n), t0=7.0)
    hits, st = run(geo, ice, src, 21, [L], flags=B.FLAG_BRUTE_FORCE_DOMS)
    frac = lam / L * math.exp(-(D - R) / lam) * (math.exp(L / lam) - 1.0)
    assert st.photons_hit / n == pytest.approx(frac, abs=4 * math.sqrt(frac * (1 - frac) / n))
    t = hits["time_ns"] - 7.0
    t_hi = (D - R) / V
    t_lo = t_hi - L * (1.0 / V - 1.0 / C)
    assert t.min() >= t_lo - 1e-4 and t.max() <= t_hi + 1e-4
    ell = (t_hi - t) / (1.0 / V - 1.0 / C)
    mean_ell = L * math.exp(L / lam) / (math.exp(L / lam) - 1.0) - lam
    assert ell.mean() == pytest.approx(mean_ell, abs=4 * L / math.sqrt(12 * len(ell)))
    ref = O.propagate(geo, ice, src, seed=21, brute_force=True, lengths=[L])
    c = compare_hits(hits, ref.hits, n)
    assert c["frac_all"] >= 0.9999 and c["max_dt"] <= 1e-3, c


def test_segments_with_acceptance_and_bad_lengths():
    geo, ice = W.geometry_full(radius=1.0), W.ice_layered()
    src = W.sources_track(n_seg=40, n_casc=10)
    src.src[:, 7] = 2.0
    n = total_photons(src, ice)
    hits, st = run(geo, ice, src, 8, src.length, acceptance="weighted")
    ref = O.propagate(geo, ice, src, seed=8, acceptance_mode="weighted", acceptance_coef=W.ACCEPTANCE_COEF)
    assert st.photons_done == n and flights_agree(st.flights, ref.flights) and abs(st.photons_hit - ref.hit) <= 2
    c = compare_hits(hits, ref.hits, n)
    assert c["frac_all"] >= 0.999 and c["frac_hit"] >= 0.97, c
    with B.Propagator(geo, ice, seed=0) as p:
        for bad in (-1.0, float("nan"), float("inf")):
            with pytest.raises(B.PPError) as e:
                p.submit(src.src[:1], src.event_id[:1], src.source_id[:1], [bad])
            assert e.value.code == -1
        assert len(p.collect_all()) == 0


def test_effective_scattering_lengths():
    """NEXT-2, R-20: the scattering table given as lambda_e = lambda_s/(1-g) (PP_FLAG_EFFECTIVE_SCATTERING)."""
    geo = W.geometry_full(radius=1.0)
    ice = W.ice_layered()
    eff = W.ice_layered()
    eff.scat_len = (ice.scat_len.astype(np.float64) / (1.0 - float(np.float32(ice.g)))).astype(np.float32)
    eff.effective_scattering = True
    src = W.sources_c1().subset(slice(0, 30))
    src.src[:, 7] = 3.0
    n = total_photons(src, ice)
    hits, st = run(geo, eff, src, 10, None)
    ref = O.propagate(geo, eff, src, seed=10)
    assert st.photons_done == n == ref.photons and ref.hit > 500
    assert abs(st.flights - ref.flights) <= 2 and abs(st.photons_hit - ref.hit) <= 2
    c = compare_hits(hits, ref.hits, n)
    assert c["frac_all"] >= 0.999 and c["frac_hit"] >= 0.97, c
    # the same physics as the geometric table (lambda_e (1-g) rounds to lambda_s within an ulp): same statistics
    base, st_b = run(geo, ice, src, 10, None)
    assert abs(st.flights - st_b.flights) <= 1e-3 * st_b.flights and abs(len(base) - len(hits)) <= 6 * math.sqrt(len(base))


def test_longitudinal_profile():
    """NEXT-2, R-23: emission offsets drawn through a caller-supplied inverse-CDF table."""
    knots = np.sqrt(np.linspace(0.0, 1.0, 33)).astype(np.float32)
    geo, ice = W.geometry_full(radius=1.0), W.ice_layered()
    src = W.sources_track(n_seg=40, n_casc=10)
    src.src[:, 7] = 3.0
    n = total_photons(src, ice)

    def go(table, lengths):
        with B.Propagator(geo, ice, seed=29) as p:
            p.set_segment_profile(table)
            hits = sort_hits(p.run(src.src, src.event_id, src.source_id, lengths))
            return hits, p.stats()

    hits, st = go(knots, src.length)
    ref = O.propagate(geo, ice, src, seed=29, segment_profile=knots)
    assert st.photons_done == n == ref.photons and ref.hit > 800
    assert abs(st.flights - ref.flights) <= 3 and abs(st.photons_hit - ref.hit) <= 2
    c = compare_hits(hits, ref.hits, n)
    assert c["frac_all"] >= 0.999 and c["frac_hit"] >= 0.97, c
    uni, _ = go(None, src.length)
    assert not np.array_equal(uni, hits)
    # closed form on the GPU: beam from a 30 m segment at a DOM 40 m ahead, scattering off, density 2 l / L^2
    lam, L, D, m = 100.0, 30.0, 40.0, 400000
    R = float(np.float32(W.DOM_RADIUS))
    geo2 = W.Geometry(xyz=np.array([[0.0, 0.0, D]], np.float32), radius=W.DOM_RADIUS)
    ice2 = W.ice_homogeneous(scat_len=1.0e30, cos_cherenkov=1.0)
    beam = W.pencil_beam([0, 0, 0], [0, 0, 1], float(m))
    with B.Propagator(geo2, ice2, seed=5, flags=B.FLAG_BRUTE_FORCE_DOMS) as p:
        p.set_segment_profile(knots)
        h2 = p.run(beam.src, beam.event_id, beam.source_id, [L])
    k = knots.astype(np.float64)
    # hit fraction = E[exp(-(D - R - l)/lam)] over the table's piecewise-uniform offsets
    a, b = L * k[:-1], L * k[1:]
    seg = np.where(b > a, lam * (np.exp(b / lam) - np.exp(a / lam)) / np.maximum(b - a, 1e-12), np.exp(a / lam))
    frac = math.exp(-(D - R) / lam) * seg.mean()
    assert len(h2) / m == pytest.approx(frac, abs=4 * math.sqrt(frac * (1 - frac) / m))
    ref2 = O.propagate(geo2, ice2, beam, seed=5, brute_force=True, lengths=[L], segment_profile=knots)
    c2 = compare_hits(sort_hits(h2), ref2.hits, m)
    assert c2["frac_all"] >= 0.9999 and c2["max_dt"] <= 1e-3, c2
    with B.Propagator(geo, ice, seed=0) as p:
        for bad in ([0.5], [0.0, 0.6, 0.5], [0.0, 1.2], list(np.linspace(0, 1, 34))):
            with pytest.raises(B.PPError):
                p.set_segment_profile(bad)
