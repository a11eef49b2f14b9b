"""Pins of the oracle's extended (track-segment) sources (NEXT-2, R-18; PAPER.md:29 continuous losses along
the muon, "photon emitting steps") against closed forms."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2405_05700_b200 import workloads as W

C = W.C_VACUUM
V = C / float(np.float32(W.N_GROUP))


def test_beam_from_a_segment_at_a_dom_ahead():
    # beam along the axis (cos_cherenkov = 1), scattering off, DOM centred on the axis at distance D > L:
    # a photon emitted at offset l survives D - R - l metres of absorption and arrives at l/c + (D - R - l)/v
    lam, L, D, n = 100.0, 20.0, 30.0, 400000
    R = float(np.float32(W.DOM_RADIUS))
    geo = W.Geometry(xyz=np.array([[0.0, 0.0, D]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous(scat_len=1.0e30, cos_cherenkov=1.0)
    src = W.pencil_beam([0, 0, 0], [0, 0, 1], float(n), t0=7.0)
    r = O.propagate(geo, ice, src, seed=21, brute_force=True, lengths=[L])
    frac = lam / L * math.exp(-(D - R) / lam) * (math.exp(L / lam) - 1.0)
    assert frac == pytest.approx(0.821, abs=2e-3)
    assert r.hit / n == pytest.approx(frac, abs=4 * math.sqrt(frac * (1 - frac) / n))
    t = r.hits["time_ns"] - 7.0
    t_hi = (D - R) / V
    t_lo = t_hi - L * (1.0 / V - 1.0 / C)
    assert t.min() >= t_lo - 1e-9 and t.max() <= t_hi + 1e-9
    assert t.min() < t_lo + 0.01 * (t_hi - t_lo) and t.max() > t_hi - 0.01 * (t_hi - t_lo)
    ell = (t_hi - t) / (1.0 / V - 1.0 / C)  # emission offset implied by each arrival time
    mean_ell = L * math.exp(L / lam) / (math.exp(L / lam) - 1.0) - lam  # density ~ exp(l / lambda) on [0, L]
    assert mean_ell == pytest.approx(10.332, abs=2e-3)
    assert ell.mean() == pytest.approx(mean_ell, abs=4 * L / math.sqrt(12 * len(ell)))
    # the same source with L = 0 is the pencil beam of test_oracle_propagate: exp(-(D-R)/lambda), one arrival time
    r0 = O.propagate(geo, ice, src, seed=21, brute_force=True, lengths=[0.0])
    e0 = math.exp(-(D - R) / lam)
    assert r0.hit / n == pytest.approx(e0, abs=4 * math.sqrt(e0 * (1 - e0) / n))
    assert np.allclose(r0.hits["time_ns"], 7.0 + t_hi, atol=1e-9)


def test_end_point_displacement_and_time_offset():
    # no DOM in reach, homogeneous ice: mean end-point displacement along the axis = L/2 + 1/(a + b(1-g)) (beam),
    # and end time - path/v = t0 + l/c is uniform on [t0, t0 + L/c]
    L, n = 50.0, 200000
    geo = W.Geometry(xyz=np.array([[1.0e5, 0.0, 0.0]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous(cos_cherenkov=1.0)
    src = W.pencil_beam([1, 2, 3], [0.6, 0.0, 0.8], float(n), t0=-5.0)
    r = O.propagate(geo, ice, src, seed=4, brute_force=True, want_fates=True, lengths=[L])
    f = r.fates
    assert r.hit == 0 and r.absorbed == n
    disp = (f["x"] - 1.0) * float(np.float32(0.6)) + (f["z"] - 3.0) * float(np.float32(0.8))
    expect = L / 2 + 1.0 / (0.01 + 0.04 * 0.1)
    assert expect == pytest.approx(96.4286, abs=1e-4)
    assert disp.mean() == pytest.approx(expect, abs=4 * disp.std() / math.sqrt(n))
    delay = f["time_ns"] - f["path_m"] / V + 5.0
    assert delay.min() >= -1e-9 and delay.max() <= L / C + 1e-9
    assert delay.mean() == pytest.approx(0.5 * L / C, abs=4 * (L / C) / math.sqrt(12 * n))
    assert np.var(delay) == pytest.approx((L / C) ** 2 / 12, rel=0.02)
    # Cherenkov cone about the axis is untouched by the offset: with cos_cherenkov = cos 41.2 deg the first flight
    # makes that angle with the axis -- checked through the unscattered photons' end points relative to their start
    ice2 = W.ice_homogeneous(scat_len=1.0e30)
    r2 = O.propagate(geo, ice2, src, seed=4, brute_force=True, want_fates=True, lengths=[L])
    g = r2.fates
    ell = (g["time_ns"] - g["path_m"] / V + 5.0) * C
    ax = np.array([float(np.float32(0.6)), 0.0, float(np.float32(0.8))])
    start = np.array([1.0, 2.0, 3.0])[None, :] + ell[:, None] * ax[None, :]
    end = np.stack([g["x"], g["y"], g["z"]], axis=1)
    cosang = ((end - start) @ ax) / g["path_m"]
    assert np.allclose(cosang, float(np.float32(ice2.cos_cherenkov)), atol=1e-6)


def test_zero_length_is_the_point_source_bit_for_bit_and_mixed_lists():
    geo, ice = W.geometry_full(radius=1.0), W.ice_layered()
    src = W.sources_track(n_seg=10, n_casc=5)
    src.src[:, 7] = 0.5
    a = O.propagate(geo, ice, src, seed=2, lengths=np.zeros(len(src), np.float32))
    b = O.propagate(geo, ice, src, seed=2, lengths=None if False else np.zeros(len(src), np.float32) * 0)
    pt = W.Sources(src.src, src.event_id, src.source_id)
    c = O.propagate(geo, ice, pt, seed=2)
    assert np.array_equal(a.hits, c.hits) and np.array_equal(b.hits, c.hits) and a.flights == c.flights
    d = O.propagate(geo, ice, src, seed=2)  # picks up src.length
    assert d.photons == c.photons and not np.array_equal(d.hits, c.hits)
    # the point cascades of the mixed list (length 0) are untouched by their neighbours' lengths
    is_pt = src.length == 0
    sid_pt = set(int(x) for x in src.source_id[is_pt])
    hd = d.hits[[int(s) in sid_pt for s in d.hits["source_id"]]]
    hc = c.hits[[int(s) in sid_pt for s in c.hits["source_id"]]]
    assert np.array_equal(hd, hc)


def test_longitudinal_profile_table():
    """NEXT-2, R-23: the emission offset is L F(u), F piecewise linear through a caller-supplied table."""
    tab = [0.0, 0.5, 0.7, 1.0]
    assert O.segment_fraction(tab, 0.0) == 0.0 and O.segment_fraction(tab, 1.0) == pytest.approx(1.0, abs=1e-7)
    assert O.segment_fraction(tab, 1 / 3) == pytest.approx(0.5, abs=1e-6)
    assert O.segment_fraction(tab, 0.5) == pytest.approx(0.6, abs=1e-6)       # halfway between knots 1 and 2
    assert O.segment_fraction(tab, 0.9) == pytest.approx(0.7 + 0.7 * 0.3, abs=1e-6)
    # F(u) = sqrt(u) sampled finely = density 2 l / L^2 (light piles up towards the end): mean 2L/3, variance L^2/18
    knots = np.sqrt(np.linspace(0.0, 1.0, 33)).astype(np.float32)
    L, n = 30.0, 200000
    geo = W.Geometry(xyz=np.array([[1.0e6, 0.0, 0.0]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous(scat_len=1.0e30, cos_cherenkov=1.0)
    src = W.pencil_beam([0, 0, 0], [0, 0, 1], float(n))
    r = O.propagate(geo, ice, src, seed=4, brute_force=True, want_fates=True, lengths=[L], segment_profile=knots)
    ell = (r.fates["time_ns"] - r.fates["path_m"] / V) * C          # emission delay x c
    # the table is the chord approximation of sqrt: its exact moments follow from the knots
    k = knots.astype(np.float64)
    m1 = L * np.mean((k[:-1] + k[1:]) / 2)
    m2 = L * L * np.mean((k[:-1] ** 2 + k[:-1] * k[1:] + k[1:] ** 2) / 3)
    assert m1 == pytest.approx(2 * L / 3, rel=5e-3)
    assert ell.mean() == pytest.approx(m1, abs=4 * ell.std() / math.sqrt(n))
    assert np.var(ell) == pytest.approx(m2 - m1 * m1, rel=0.02)
    assert ell.min() >= -1e-9 and ell.max() <= L + 1e-9
    # the identity table is the uniform segment of R-18 (to rounding)
    ident = np.linspace(0.0, 1.0, 9).astype(np.float32)
    a = O.propagate(geo, ice, src, seed=4, brute_force=True, want_fates=True, lengths=[L])
    b = O.propagate(geo, ice, src, seed=4, brute_force=True, want_fates=True, lengths=[L], segment_profile=ident)
    assert np.allclose(a.fates["z"], b.fates["z"], atol=1e-5) and np.allclose(a.fates["time_ns"], b.fates["time_ns"], atol=1e-5)
