"""Pins for the oracle's Henyey-Greenstein sampler (R-1) and rotation (R-9)."""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle import oracle as O


def hg_pdf(mu, g):
    """Henyey & Greenstein (1941) phase function in mu = cos(theta), normalised on [-1, 1]."""
    return (1.0 - g * g) / (2.0 * (1.0 + g * g - 2.0 * g * mu) ** 1.5)


@pytest.mark.parametrize("g", [0.9, 0.5, -0.3, 0.99])
def test_hg_inverse_cdf_matches_integrated_pdf(g):
    # u = CDF(mu) with CDF obtained by numerical quadrature of the textbook pdf: independent of
    # the oracle's closed-form inverse.  u -> 1 is forward (mu -> 1).
    for u in (0.001, 0.1, 0.37, 0.5, 0.9, 0.999):
        mu = O.hg_cos(g, u)
        cdf, _ = integrate.quad(hg_pdf, -1.0, mu, args=(g,), epsabs=1e-12, epsrel=1e-12, limit=200)
        assert cdf == pytest.approx(u, abs=2e-9)


@pytest.mark.parametrize("g", [0.9, 0.3])
def test_hg_moments(g):
    # <cos> = g and <cos^2> = (1 + 2 g^2)/3 (Legendre moments of HG: <P_l> = g^l)
    n = 200001
    u = (np.arange(n) + 0.5) / n
    mu = np.array([O.hg_cos(g, x) for x in u])
    assert mu.mean() == pytest.approx(g, abs=2e-6)
    assert (mu * mu).mean() == pytest.approx((1.0 + 2.0 * g * g) / 3.0, abs=2e-6)
    assert mu.min() >= -1.0 and mu.max() <= 1.0
    assert np.all(np.diff(mu) > 0)  # monotone: forward for u -> 1


def test_hg_isotropic_limit():
    for u in (0.0, 0.25, 0.5, 1.0):
        assert O.hg_cos(0.0, u) == 2.0 * u - 1.0
    # continuity g -> 0
    assert O.hg_cos(1e-9, 0.3) == pytest.approx(2 * 0.3 - 1, abs=1e-6)


def _rand_unit(rng):
    v = rng.normal(size=3)
    return v / np.linalg.norm(v)


def test_rotate_unit_and_polar_angle():
    rng = np.random.default_rng(7)
    for _ in range(300):
        d = _rand_unit(rng)
        ct = rng.uniform(-1, 1)
        phi = rng.uniform(0, 2 * math.pi)
        n = O.rotate(d, ct, phi)
        assert np.linalg.norm(n) == pytest.approx(1.0, abs=1e-14)
        assert float(n @ d) == pytest.approx(ct, abs=1e-12)


def test_rotate_azimuth_reference():
    # R-9: for a direction in the xz-plane the azimuth is measured from the "downward-tilted"
    # meridian: phi = 0 moves the direction toward -z (for d_z != +-1), phi = pi/2 toward
    # the vector z x d / |z x d| (counter-clockwise seen from above).
    d = np.array([1.0, 0.0, 0.0])
    st, ct = math.sin(0.3), math.cos(0.3)
    assert np.allclose(O.rotate(d, ct, 0.0), [ct, 0.0, -st], atol=1e-15)
    assert np.allclose(O.rotate(d, ct, math.pi / 2), [ct, st, 0.0], atol=1e-15)
    assert np.allclose(O.rotate(d, ct, math.pi), [ct, 0.0, st], atol=1e-15)
    # general d: the phi = 0 image lies in the plane spanned by d and z, the phi = pi/2 image
    # keeps the z component d_z cos(theta)
    rng = np.random.default_rng(3)
    for _ in range(50):
        d = _rand_unit(rng)
        n0 = O.rotate(d, ct, 0.0)
        assert abs(np.linalg.det(np.stack([d, [0, 0, 1.0], n0]))) < 1e-12
        assert n0[2] < d[2] * ct + 1e-15
        n90 = O.rotate(d, ct, math.pi / 2)
        assert n90[2] == pytest.approx(d[2] * ct, abs=1e-14)
        # right-handedness: (d, n0_perp, n90_perp) is a right-handed triad
        e0 = n0 - ct * d
        e90 = n90 - ct * d
        assert float(np.cross(e0, e90) @ d) > 0


def test_rotate_azimuth_uniform_and_composition():
    # phi -> phi + delta rotates the image about d by delta
    rng = np.random.default_rng(11)
    d = _rand_unit(rng)
    ct = 0.4
    ref = O.rotate(d, ct, 0.0) - ct * d
    ref /= np.linalg.norm(ref)
    ref2 = np.cross(d, ref)
    for phi in np.linspace(0, 2 * math.pi, 17):
        n = O.rotate(d, ct, phi)
        e = n - ct * d
        ang = math.atan2(float(e @ ref2), float(e @ ref))
        assert math.isclose(math.cos(ang), math.cos(phi), abs_tol=1e-12)
        assert math.isclose(math.sin(ang), math.sin(phi), abs_tol=1e-12)


def test_rotate_pole_branch_is_the_limit_of_the_general_branch():
    ct, phi = 0.8, 1.1
    st = math.sqrt(1 - ct * ct)
    for sign in (1.0, -1.0):
        pole = O.rotate([0.0, 0.0, sign], ct, phi)
        assert np.allclose(pole, [st * math.cos(phi), st * math.sin(phi), sign * ct], atol=1e-15)
        assert np.linalg.norm(pole) == pytest.approx(1.0, abs=1e-15)
    # general branch approaching +z along the x meridian: d = (eps, 0, 1): image -> (st cos(phi), st sin(phi), ct)
    eps = 1e-4
    d = np.array([eps, 0.0, math.sqrt(1 - eps * eps)])
    assert np.allclose(O.rotate(d, ct, phi), O.rotate([0, 0, 1.0], ct, phi), atol=3e-4)
    # approaching -z along the x meridian: image -> (-st cos(phi), st sin(phi), -ct) for the general branch
    d = np.array([eps, 0.0, -math.sqrt(1 - eps * eps)])
    g = O.rotate(d, ct, phi)
    assert np.allclose(g, [-st * math.cos(phi), st * math.sin(phi), -ct], atol=3e-4)
