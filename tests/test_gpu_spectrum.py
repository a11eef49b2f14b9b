"""GPU parity of the wavelength bins (NEXT-2, R-21) against the oracle, through the C ABI."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import workloads as W

from gpu_util import compare_hits, sort_hits, total_photons

pytestmark = pytest.mark.gpu
C = W.C_VACUUM


def run(geo, ice, src, seed, spectrum, acceptance=None, lengths=None, **kw):
    with B.Propagator(geo, ice, seed=seed, **kw) as p:
        p.set_spectrum(spectrum)
        if acceptance:
            p.set_acceptance(acceptance, W.ACCEPTANCE_COEF)
        hits = sort_hits(p.run(src.src, src.event_id, src.source_id, lengths))
        st = p.stats()
    return hits, st


def test_layered_oversized_doms_per_photon():
    """8 stand-in wavelength bins, full detector with oversized DOMs, layered ice, several launches."""
    geo, ice, sp = W.geometry_full(radius=1.0), W.ice_layered(), W.spectrum_standin()
    src = W.sources_c1().subset(slice(0, 40))
    src.src[:, 7] = 4.0
    n = total_photons(src, ice)
    hits, st = run(geo, ice, src, 17, sp, launch_photons_target=500000)
    ref = O.propagate(geo, ice, src, seed=17, spectrum=sp)
    assert st.photons_done == n == ref.photons and st.launches >= 3 and ref.hit > 1000
    assert abs(st.flights - ref.flights) <= 3 and abs(st.photons_hit - ref.hit) <= 2
    c = compare_hits(hits, ref.hits, n)
    assert c["frac_all"] >= 0.999 and c["frac_hit"] >= 0.97, c
    # the bins matter, and switching them off again restores the monochromatic path bit for bit
    mono, _ = run(geo, ice, src, 17, None, launch_photons_target=500000)
    assert not np.array_equal(mono, hits)
    with B.Propagator(geo, ice, seed=17, launch_photons_target=500000) as p:
        p.set_spectrum(sp)
        p.set_spectrum(None)
        again = sort_hits(p.run(src.src, src.event_id, src.source_id))
    assert np.array_equal(again, mono)
    # one bin with unit scales is the monochromatic path too
    one = W.Spectrum(*(np.asarray(v, np.float32) for v in ([1.0], [1.0], [1.0], [ice.n_group], [1.0])))
    same, _ = run(geo, ice, src, 17, one, launch_photons_target=500000)
    assert np.array_equal(same, mono)


def test_closed_form_on_the_gpu():
    """The oracle's pin: a DOM on a pencil beam, scattering off, two bins: two arrival times (d-R) n_j / c with
    frequencies w_j exp(-(d-R) a_j)."""
    f = lambda v: np.asarray(v, np.float32)
    sp = W.Spectrum(f([0.25, 1.0]), f([2.0, 0.5]), f([1.0, 1.0]), f([1.30, 1.40]), f([1.0, 1.0]))
    dist, n = 40.0, 400000
    R = float(np.float32(W.DOM_RADIUS))
    geo = W.Geometry(xyz=np.array([[0.0, 0.0, dist]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous(scat_len=1.0e30, cos_cherenkov=1.0)
    src = W.pencil_beam([0, 0, 0], [0, 0, 1], float(n))
    hits, st = run(geo, ice, src, 15, sp, flags=B.FLAG_BRUTE_FORCE_DOMS)
    t = hits["time_ns"]
    t0, t1 = (dist - R) * float(np.float32(1.30)) / C, (dist - R) * float(np.float32(1.40)) / C
    e0, e1 = 0.25 * math.exp(-(dist - R) / 50.0), 0.75 * math.exp(-(dist - R) / 200.0)
    n0, n1 = int((np.abs(t - t0) < 1e-4).sum()), int((np.abs(t - t1) < 1e-4).sum())
    assert n0 + n1 == len(t) == st.photons_hit
    assert n0 / n == pytest.approx(e0, abs=4 * math.sqrt(e0 / n)) and n1 / n == pytest.approx(e1, abs=4 * math.sqrt(e1 / n))
    ref = O.propagate(geo, ice, src, seed=15, brute_force=True, spectrum=sp)
    c = compare_hits(hits, ref.hits, n)
    assert c["frac_all"] >= 0.9999 and c["max_dt"] <= 1e-3, c


def test_everything_together_and_bad_inputs():
    """Wavelength bins + weighted acceptance + track segments in one run; rejected spectra."""
    geo, ice, sp = W.geometry_full(radius=1.0), W.ice_layered(), W.spectrum_standin()
    src = W.sources_track(n_seg=40, n_casc=10)
    src.src[:, 7] = 3.0
    n = total_photons(src, ice)
    hits, st = run(geo, ice, src, 19, sp, acceptance="weighted", lengths=src.length)
    ref = O.propagate(geo, ice, src, seed=19, spectrum=sp, acceptance_mode="weighted", acceptance_coef=W.ACCEPTANCE_COEF)
    assert st.photons_done == n and abs(st.flights - ref.flights) <= 3 and abs(st.photons_hit - ref.hit) <= 2
    c = compare_hits(hits, ref.hits, n)
    assert c["frac_all"] >= 0.999 and c["frac_hit"] >= 0.97, c
    kr = {(int(a), int(b), int(c_)): float(w) for a, b, c_, w in
          zip(ref.hits["event_id"], ref.hits["source_id"], ref.hits["photon_idx"], ref.hits["weight"])}
    dw = [abs(float(h["weight"]) - kr[k]) for h in hits
          for k in [(int(h["event_id"]), int(h["source_id"]), int(h["photon_idx"]))] if k in kr]
    assert len(dw) >= 0.97 * len(hits) and max(dw) <= 3e-5
    f = lambda v: np.asarray(v, np.float32)
    with B.Propagator(geo, ice, seed=0) as p:
        for bad in (W.Spectrum(f([0.5, 0.4]), f([1, 1]), f([1, 1]), f([1.3, 1.3]), f([1, 1])),      # cdf decreasing
                    W.Spectrum(f([0.5, 1.0]), f([1, 0]), f([1, 1]), f([1.3, 1.3]), f([1, 1])),      # zero abs scale
                    W.Spectrum(f([0.5, 1.0]), f([1, 1]), f([1, 1]), f([0.9, 1.3]), f([1, 1])),      # n_group < 1
                    W.Spectrum(f([0.5, 1.0]), f([1, 1]), f([1, 1]), f([1.3, 1.3]), f([1, -1]))):    # negative acceptance
            with pytest.raises(B.PPError) as e:
                p.set_spectrum(bad)
            assert e.value.code == -1
        big = W.Spectrum(*(np.ones(33, np.float32) for _ in range(5)))
        with pytest.raises(B.PPError):
            p.set_spectrum(big)


def test_emission_smearing():
    """NEXT-2, R-22: emission axis deflected by an HG(g_axis) angle: per-photon parity, the closed form <cos> =
    g cos(theta_c) on the GPU, off == exact cone bit for bit."""
    geo, ice = W.geometry_full(radius=1.0), W.ice_layered()
    src = W.sources_c1().subset(slice(0, 40))
    src.src[:, 7] = 3.0
    n = total_photons(src, ice)

    def go(g_axis, **kw):
        with B.Propagator(geo, ice, seed=23, **kw) as p:
            if g_axis is not None:
                p.set_emission_smearing(g_axis)
            hits = sort_hits(p.run(src.src, src.event_id, src.source_id))
            return hits, p.stats()

    hits, st = go(0.8, launch_photons_target=400000)
    ref = O.propagate(geo, ice, src, seed=23, g_axis=0.8)
    assert st.photons_done == n == ref.photons and ref.hit > 800 and st.launches >= 3
    assert abs(st.flights - ref.flights) <= 3 and abs(st.photons_hit - ref.hit) <= 2
    c = compare_hits(hits, ref.hits, n)
    assert c["frac_all"] >= 0.999 and c["frac_hit"] >= 0.97, c
    plain, _ = go(None)
    off, _ = go(1.0)
    assert np.array_equal(plain, off) and not np.array_equal(plain, hits)
    # closed form: scattering off, a ring of huge "DOMs" is not needed -- use the fates of the resident path
    ice2 = W.ice_homogeneous(scat_len=1.0e30)
    geo2 = W.Geometry(xyz=np.array([[1.0e6, 0.0, 0.0]], np.float32), radius=W.DOM_RADIUS)
    beam = W.pencil_beam([1, 2, 3], [0.48, -0.6, 0.64], 200000.0)
    with B.Propagator(geo2, ice2, seed=31, flags=B.FLAG_BRUTE_FORCE_DOMS) as p:
        p.set_emission_smearing(0.6)
        d = p.upload(beam.src, beam.event_id, beam.source_id)
        ph, ms, f = p.run_resident(*d, want_fates=True, n_photons_hint=200000)
    dirs = np.stack([f["x"] - 1.0, f["y"] - 2.0, f["z"] - 3.0], axis=1).astype(np.float64) / f["path_m"][:, None]
    a = beam.src[0, 3:6].astype(np.float64)
    cosg = dirs @ (a / np.linalg.norm(a))
    cc, g = float(np.float32(ice2.cos_cherenkov)), float(np.float32(0.6))
    assert cosg.mean() == pytest.approx(g * cc, abs=4 * cosg.std() / math.sqrt(len(cosg)) + 1e-5)
    with B.Propagator(geo, ice, seed=0) as p:
        for bad in (0.0, 1.5, -1.0, float("nan")):
            with pytest.raises(B.PPError):
                p.set_emission_smearing(bad)
