"""Pins for the oracle's layer walk (PAPER.md:31 10 m layers; readings R-6, R-7)."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2405_05700_b200 import workloads as W


def three_layers():
    # layer 0: z in (20, 30]  len 10 ; layer 1: (10, 20] len 5 ; layer 2: (0, 10] len 20; ends infinite
    return W.Ice(abs_len=np.array([40.0, 8.0, 100.0], np.float32), scat_len=np.array([10.0, 5.0, 20.0], np.float32),
                 z_top=30.0, dz=10.0)


def test_layer_index_and_infinite_end_layers():
    ice = three_layers()
    assert O.layer_of(ice, 29.0) == 0
    assert O.layer_of(ice, 1e6) == 0  # above the table: first layer extends to +inf
    assert O.layer_of(ice, 15.0) == 1
    assert O.layer_of(ice, 5.0) == 2
    assert O.layer_of(ice, -1e6) == 2  # below: last layer extends to -inf
    lay = W.ice_layered()
    assert O.layer_of(lay, 499.0) == 0 and O.layer_of(lay, -499.0) == 99
    # depth 2050 m (z = -100) is layer 60 (depth 2050-2060)
    assert O.layer_of(lay, -100.5) == 60


def test_walk_hand_computed_downward():
    ice = three_layers()
    # start z=25 going straight down (dir_z=-1), scattering table: c = 0.1, 0.2, 0.05 per metre
    # optical depth to z=20: 0.5 ; to z=10: 0.5 + 2.0 = 2.5 ; below: 0.05/m for ever
    assert O.walk(ice, "scat", 25.0, -1.0, 0.3) == pytest.approx(3.0, abs=1e-12)
    assert O.walk(ice, "scat", 25.0, -1.0, 0.5) == pytest.approx(5.0, abs=1e-12)
    assert O.walk(ice, "scat", 25.0, -1.0, 1.5) == pytest.approx(5.0 + 5.0, abs=1e-12)
    assert O.walk(ice, "scat", 25.0, -1.0, 2.5 + 1.0) == pytest.approx(15.0 + 20.0, abs=1e-12)
    assert O.walk(ice, "scat", 25.0, -1.0, 2.5 + 50.0) == pytest.approx(15.0 + 1000.0, abs=1e-9)  # infinite last layer
    # absorption table is selected by "abs": c = 1/40 in layer 0
    assert O.walk(ice, "abs", 25.0, -1.0, 0.05) == pytest.approx(2.0, abs=1e-12)


def test_walk_hand_computed_upward_and_oblique():
    ice = three_layers()
    # start z=5 going up with dir_z = 0.5: path lengths double: 10 m to z=10 (tau 0.5), 20 m to z=20 (tau 4.0), then 0.1/m
    assert O.walk(ice, "scat", 5.0, 0.5, 0.25) == pytest.approx(5.0, abs=1e-12)
    assert O.walk(ice, "scat", 5.0, 0.5, 0.5 + 2.0) == pytest.approx(10.0 + 10.0, abs=1e-12)
    assert O.walk(ice, "scat", 5.0, 0.5, 4.5 + 3.0) == pytest.approx(30.0 + 30.0, abs=1e-12)
    # horizontal ray never leaves its layer
    assert O.walk(ice, "scat", 15.0, 0.0, 7.0) == pytest.approx(35.0, abs=1e-12)


def test_depth_is_inverse_of_walk():
    ice = W.ice_layered()
    rng = np.random.default_rng(5)
    for _ in range(400):
        z = rng.uniform(-700, 700)
        dz = rng.uniform(-1, 1)
        tau = rng.exponential(1.0) + 1e-3
        which = "abs" if rng.uniform() < 0.5 else "scat"
        s = O.walk(ice, which, z, dz, tau)
        assert s > 0
        assert O.depth(ice, which, z, dz, s) == pytest.approx(tau, rel=1e-12)


def test_depth_against_numerical_integration_of_the_table():
    # independent check: integrate c(z(s)) with a fine midpoint rule using only the table definition
    ice = W.ice_layered()
    z0, dz, s = 123.0, -0.37, 400.0
    n = 400000
    ss = (np.arange(n) + 0.5) * (s / n)
    zz = z0 + dz * ss
    idx = np.clip(np.floor((ice.z_top - zz) / ice.dz), 0, ice.n_layers - 1).astype(int)
    tau = (1.0 / ice.abs_len.astype(np.float64)[idx]).sum() * (s / n)
    assert O.depth(ice, "abs", z0, dz, s) == pytest.approx(tau, rel=2e-5)


def test_homogeneous_single_layer_is_infinite():
    ice = W.ice_homogeneous()
    for z, dz in ((0.0, 1.0), (1e5, -1.0), (-1e5, 0.3)):
        assert O.walk(ice, "scat", z, dz, 2.0) == pytest.approx(50.0, rel=1e-14)
        assert O.walk(ice, "abs", z, dz, 2.0) == pytest.approx(200.0, rel=1e-14)


def test_layered_table_recipe():
    ice = W.ice_layered()
    assert ice.n_layers == 100 and ice.dz == 10.0 and ice.z_top == 500.0
    a, b = ice.abs_len.astype(np.float64), ice.scat_len.astype(np.float64)
    dust = np.arange(100)[(np.arange(100) >= 55) & (np.arange(100) < 65)]  # depth 2000-2100
    clean = np.setdiff1d(np.arange(100), dust)
    assert a[clean].min() >= 20.0 - 1e-4 and a[clean].max() <= 250.0 + 1e-4
    assert b[clean].min() >= 5.0 - 1e-4 and b[clean].max() <= 60.0 + 1e-4
    # one profile drives both: (a-20)/230 == (b-5)/55 outside the dust layer, and 5x both inside
    assert np.allclose((a[clean] - 20) / 230, (b[clean] - 5) / 55, atol=1e-5)
    assert np.allclose((5 * a[dust] - 20) / 230, (5 * b[dust] - 5) / 55, atol=1e-5)
