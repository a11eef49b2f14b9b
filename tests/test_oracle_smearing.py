"""Pins of the oracle's angular smearing of the emission axis (NEXT-2, R-22) against closed forms."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2405_05700_b200 import workloads as W

V = W.C_VACUUM / float(np.float32(W.N_GROUP))


def first_flight_directions(g_axis, axis, n=200000, seed=31):
    # scattering off, no DOM in reach: every photon flies straight from the source to where it is absorbed
    geo = W.Geometry(xyz=np.array([[1.0e6, 0.0, 0.0]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous(scat_len=1.0e30)
    src = W.pencil_beam([1, 2, 3], axis, float(n))
    r = O.propagate(geo, ice, src, seed=seed, brute_force=True, want_fates=True, g_axis=g_axis)
    f = r.fates
    d = np.stack([f["x"] - 1.0, f["y"] - 2.0, f["z"] - 3.0], axis=1) / f["path_m"][:, None]
    return d, float(np.float32(ice.cos_cherenkov)), r


@pytest.mark.parametrize("g_axis", [0.95, 0.6])
def test_legendre_moments_multiply(g_axis):
    axis = np.array([0.48, -0.6, 0.64])
    d, cc, _ = first_flight_directions(g_axis, axis)
    a32 = (axis / np.linalg.norm(axis)).astype(np.float32).astype(np.float64)
    a32 /= np.linalg.norm(a32)
    c = d @ a32
    g = float(np.float32(g_axis))
    n = len(c)
    assert c.mean() == pytest.approx(g * cc, abs=4 * c.std() / math.sqrt(n))
    p2 = 0.5 * (3 * c * c - 1)
    assert p2.mean() == pytest.approx(g * g * 0.5 * (3 * cc * cc - 1), abs=4 * p2.std() / math.sqrt(n))
    # azimuthal symmetry about the axis: the transverse part averages to zero
    t = d - c[:, None] * a32[None, :]
    assert np.all(np.abs(t.mean(axis=0)) < 4 * t.std(axis=0) / math.sqrt(n))
    assert np.allclose(np.linalg.norm(d, axis=1), 1.0, atol=1e-9)


def test_off_is_the_exact_cone_bit_for_bit():
    axis = np.array([0.0, 0.6, -0.8])
    d1, cc, r1 = first_flight_directions(1.0, axis, n=50000)
    a32 = axis.astype(np.float32).astype(np.float64)
    assert np.allclose(d1 @ (a32 / np.linalg.norm(a32)), cc, atol=1e-6)
    geo, ice = W.geometry_full(radius=1.0), W.ice_layered()
    src = W.sources_c1().subset(slice(0, 10))
    src.src[:, 7] = 1.0
    a = O.propagate(geo, ice, src, seed=1)
    b = O.propagate(geo, ice, src, seed=1, g_axis=1.0)
    c = O.propagate(geo, ice, src, seed=1, g_axis=0.9)
    assert np.array_equal(a.hits, b.hits) and not np.array_equal(a.hits, c.hits) and c.photons == a.photons
