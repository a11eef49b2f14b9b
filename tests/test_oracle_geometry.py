"""Pins for the oracle's DOM intersection ("intersects a detector"; R-5, R-8, R-11)."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2405_05700_b200 import workloads as W


def one_dom(c=(3.0, -2.0, 7.0), radius=0.5):
    return W.Geometry(xyz=np.array([c], np.float32), radius=radius)


def test_geometry_recipe():
    g = W.geometry_full()
    assert g.n_dom == 5160
    z = g.xyz[:60, 2]
    assert z[0] == 500.0 and z[59] == 500.0 - 17.0 * 59  # depths 1450 ... 2453 m
    assert np.all(np.diff(z) == -17.0)
    xy = W.hex_string_xy(86)
    r = np.hypot(xy[:, 0], xy[:, 1])
    assert r[0] == 0.0 and np.all(np.diff(np.round(r, 6)) >= 0)
    assert r[85] == pytest.approx(625.0) and xy[85, 0] == pytest.approx(-312.5)  # SURVEY R-11: 86th = (0,-5)
    # nearest-neighbour distance is the 125 m pitch for every string
    d = np.hypot(xy[:, None, 0] - xy[None, :, 0], xy[:, None, 1] - xy[None, :, 1]) + 1e9 * np.eye(86)
    assert np.allclose(d.min(axis=1), 125.0)
    # shells 1,6,6,6,12,6,6,12,6,12,12 = 85 points inside 125*sqrt(21)
    assert int((r < 125.0 * math.sqrt(21) + 1e-6).sum()) == 85


def test_head_on_chord():
    g = one_dom()
    c = np.array([3.0, -2.0, 7.0])
    d = np.array([0.6, 0.0, 0.8])
    p = c - 10.0 * d
    j, t = O.intersect(g, p, d, 20.0)
    assert j == 0 and t == pytest.approx(9.5, abs=1e-12)
    # flight too short to reach the sphere: entry at 9.5
    assert O.intersect(g, p, d, 9.4999)[0] == -1
    assert O.intersect(g, p, d, 9.5000001)[0] == 0
    # moving away
    assert O.intersect(g, p, -d, 100.0)[0] == -1


def test_offset_chord_and_tangent():
    g = one_dom((0, 0, 0), 0.5)
    # ray along +x at impact parameter b: entry at x = -sqrt(R^2 - b^2)
    for b in (0.0, 0.1, 0.3, 0.49, 0.5):
        j, t = O.intersect(g, [-5.0, b, 0.0], [1.0, 0.0, 0.0], 10.0)
        assert j == 0
        assert t == pytest.approx(5.0 - math.sqrt(0.25 - b * b), abs=1e-9)
    assert O.intersect(g, [-5.0, 0.5000001, 0.0], [1.0, 0.0, 0.0], 10.0)[0] == -1


def test_start_inside_is_hit_at_zero():
    g = one_dom((0, 0, 0), 0.5)
    j, t = O.intersect(g, [0.1, 0.2, -0.1], [0.0, 0.0, 1.0], 3.0)
    assert j == 0 and t == 0.0
    j, t = O.intersect(g, [0.1, 0.2, -0.1], [0.0, 0.0, 1.0], 0.0)  # zero-length flight
    assert j == 0 and t == 0.0


def test_nearest_dom_wins():
    g = W.Geometry(xyz=np.array([[0, 0, 10], [0, 0, 5], [0, 0, 20]], np.float32), radius=0.5)
    j, t = O.intersect(g, [0, 0, 0], [0, 0, 1.0], 100.0)
    assert j == 1 and t == pytest.approx(4.5)
    j, t = O.intersect(g, [0, 0, 7.0], [0, 0, 1.0], 100.0)
    assert j == 0 and t == pytest.approx(2.5)
    j, t = O.intersect(g, [0, 0, 30.0], [0, 0, -1.0], 100.0)
    assert j == 2 and t == pytest.approx(9.5)


def test_line_prefilter_identical_to_brute_force():
    g = W.geometry_full()
    rng = np.random.default_rng(21)
    n_hit = 0
    for i in range(1500):
        # aim near a random DOM so that a good fraction of rays hit something
        j = rng.integers(0, g.n_dom)
        c = g.xyz[j].astype(np.float64)
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        if i % 5 == 0:
            d = np.array([0.0, 0.0, 1.0 if i % 2 else -1.0])  # along a string: many DOMs in line
        off = rng.normal(size=3) * 0.15
        dist = rng.uniform(0.0, 80.0)
        p = c + off - dist * d
        s = rng.uniform(0.0, 160.0)
        jb, tb = O.intersect(g, p, d, s, brute=True)
        jl, tl = O.intersect(g, p, d, s, brute=False)
        assert jb == jl
        if jb >= 0:
            n_hit += 1
            assert tb == tl
            q = p + tb * d
            assert np.linalg.norm(q - g.xyz[jb]) <= g.radius * (1 + 1e-6) + 1e-9
    assert n_hit > 300
