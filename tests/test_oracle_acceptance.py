"""Pins of the oracle's DOM acceptance (NEXT-1, R-17; "creates a photoelectron with a
probability calculated from its position, direction, time, and wavelength": the hit carries a weight)
against hand values and closed forms."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2405_05700_b200 import workloads as W

COEF = W.ACCEPTANCE_COEF
C32 = [float(np.float32(c)) for c in COEF]


def p_hand(eta):
    return min(1.0, max(0.0, C32[0] + C32[1] * eta + C32[2] * eta * eta))


def test_polynomial_values_and_clamp():
    assert O.acceptance(COEF, 1.0) == pytest.approx(1.0, abs=1e-7)
    assert O.acceptance(COEF, -1.0) == pytest.approx(0.0, abs=1e-7)
    assert O.acceptance(COEF, 0.0) == pytest.approx(0.35, abs=1e-7)
    assert O.acceptance(COEF, 0.5) == pytest.approx(0.35 + 0.25 + 0.0375, abs=1e-7)
    assert O.acceptance([2.0, 1.0], 0.3) == 1.0 and O.acceptance([-1.0, 0.5], 0.3) == 0.0  # clamped to [0, 1]
    assert O.acceptance([0.25], -0.9) == 0.25  # constant
    # a term per power: 1 + 2x + 3x^2 + 4x^3 at x = 0.1, scaled to stay under 1
    assert O.acceptance([0.1, 0.2, 0.3, 0.4], 0.1) == pytest.approx(0.1 + 0.02 + 0.003 + 0.0004, abs=1e-8)


@pytest.mark.parametrize("axis_z", [1.0, -1.0])
def test_photons_started_inside_a_dom(axis_z):
    # A cascade inside a DOM with a vertical axis: every photon is emitted on the Cherenkov cone, so it meets the
    # DOM at distance 0 (R-5) with d_z = +-cos(theta_c) exactly: accepted fraction = p(+-cos theta_c), all weights equal.
    geo = W.Geometry(xyz=np.array([[0.0, 0.0, 0.0]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous()
    n = 200000
    src = W.pencil_beam([0.01, 0.0, 0.02], [0, 0, axis_z], float(n))
    eta = axis_z * float(np.float32(ice.cos_cherenkov))
    p = p_hand(eta)
    assert p == pytest.approx(0.8111 if axis_z > 0 else 0.0587, abs=2e-4)
    r1 = O.propagate(geo, ice, src, seed=3, brute_force=True, acceptance_mode="probabilistic", acceptance_coef=COEF)
    assert r1.photons == n and r1.hit + r1.rejected == n and r1.absorbed == 0 and r1.aborted == 0
    assert r1.hit / n == pytest.approx(p, abs=4 * math.sqrt(p * (1 - p) / n))
    assert np.all(r1.hits["weight"] == 1.0) and np.all(r1.hits["time_ns"] == 0.0)
    r2 = O.propagate(geo, ice, src, seed=3, brute_force=True, acceptance_mode="weighted", acceptance_coef=COEF)
    assert r2.hit == n and r2.rejected == 0
    assert np.allclose(r2.hits["weight"], p, rtol=0, atol=1e-12)
    r0 = O.propagate(geo, ice, src, seed=3, brute_force=True)
    assert r0.hit == n and np.all(r0.hits["weight"] == 1.0)


@pytest.mark.parametrize("direction,eta", [([1, 0, 0], 0.0), ([0, 0, 1], 1.0), ([0, 0.6, -0.8], -0.8)])
def test_pencil_beam_hit_fraction_is_survival_times_acceptance(direction, eta):
    # scattering off, beam aimed at a DOM centre at distance d: every surviving photon arrives with the beam's
    # direction, so the hit fraction is exp(-(d-R)/lambda_a) * p(d_z)
    dist, n = 20.0, 200000
    d = np.asarray(direction, float)
    geo = W.Geometry(xyz=np.array([dist * d], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous(scat_len=1.0e30, cos_cherenkov=1.0)
    src = W.pencil_beam([0, 0, 0], direction, float(n))
    surv = math.exp(-(dist - float(np.float32(W.DOM_RADIUS))) / 100.0)
    assert surv == pytest.approx(0.820084, abs=2e-6)
    p = p_hand(eta)
    r1 = O.propagate(geo, ice, src, seed=11, brute_force=True, acceptance_mode="probabilistic", acceptance_coef=COEF)
    e = surv * p
    assert r1.hit / n == pytest.approx(e, abs=4 * math.sqrt(e * (1 - e) / n) + 1e-9)
    assert (r1.hit + r1.rejected) / n == pytest.approx(surv, abs=4 * math.sqrt(surv * (1 - surv) / n))
    assert r1.photons == r1.absorbed + r1.hit + r1.aborted + r1.rejected
    r2 = O.propagate(geo, ice, src, seed=11, brute_force=True, acceptance_mode="weighted", acceptance_coef=COEF)
    if p > 0:
        assert r2.hit == r1.hit + r1.rejected  # the same photons intersect; none is dropped
        assert np.allclose(r2.hits["weight"], p, atol=1e-6)
        assert r2.hits["weight"].sum() / n == pytest.approx(e, abs=4 * math.sqrt(surv * (1 - surv) / n) * p + 1e-9)


def test_modes_agree_on_a_scattering_case_and_draw_is_keyed_by_the_hit_flight():
    # oversized DOMs in scattering ice: arrival directions vary.  The intersecting photons are the same in all modes;
    # the probabilistic mode keeps exactly those with u < p where u = word 0 of block (photon, source, event, 2^31 | k),
    # k = index of the flight that met the DOM; sum of weights ~ number accepted.
    geo = W.geometry_single_string(radius=2.0)
    ice = W.ice_homogeneous()
    src = W.sources_c0(seed=0, n_photons=400000.0, toward_string=True)
    seed = 9
    r0 = O.propagate(geo, ice, src, seed=seed, want_fates=True)
    r1 = O.propagate(geo, ice, src, seed=seed, acceptance_mode="probabilistic", acceptance_coef=COEF)
    r2 = O.propagate(geo, ice, src, seed=seed, acceptance_mode="weighted", acceptance_coef=COEF)
    assert r0.hit > 1500
    assert r1.hit + r1.rejected == r0.hit == r2.hit + r2.rejected
    assert r1.flights == r0.flights == r2.flights and r1.absorbed == r0.absorbed
    w2 = {int(h["photon_idx"]): float(h["weight"]) for h in r2.hits}
    kept = set(int(i) for i in r1.hits["photon_idx"])
    assert kept <= set(int(i) for i in r0.hits["photon_idx"])
    ev, sid = int(src.event_id[0]), int(src.source_id[0])
    n_chk = 0
    for h in r0.hits[:400]:
        i = int(h["photon_idx"])
        k = int(r0.fates["n_flights"][i]) - 1
        u = O.uniform(O.philox4x32_10((i, sid, ev, 0x80000000 | k), (seed, 0))[0])
        p = w2.get(i, 0.0)
        assert (i in kept) == (u < p)
        n_chk += 1
    assert n_chk == 400
    # times and DOMs of the kept hits are those of the acceptance-free run
    m0 = {int(h["photon_idx"]): (int(h["dom_id"]), float(h["time_ns"])) for h in r0.hits}
    for h in r1.hits[:500]:
        assert m0[int(h["photon_idx"])] == (int(h["dom_id"]), float(h["time_ns"]))
    s2 = float(r2.hits["weight"].sum())
    var = float((r2.hits["weight"] * (1 - r2.hits["weight"])).sum())
    assert abs(r1.hit - s2) <= 4.5 * math.sqrt(var)
