"""Pins of the oracle's effective-scattering option (NEXT-2, R-20): the scattering table may hold
lambda_e = lambda_s / (1 - g), the convention of measured ice tables (PAPER.md:9, :31 say only that the optical
properties vary with depth and are tabulated in 10 m layers)."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2405_05700_b200 import workloads as W


def test_effective_table_equals_geometric_table_bit_for_bit():
    # g = 0.875 and lambda_e = 200 m: lambda_s = 25 m exactly and the factor 1 - g = 1/8 is a power of two, so every
    # intermediate of the walk is the same number: the two runs must agree bit for bit
    geo = W.geometry_single_string(radius=2.0)
    src = W.sources_c0(seed=0, n_photons=100000.0, toward_string=True)
    geom = W.ice_homogeneous(scat_len=25.0, g=0.875)
    eff = W.ice_homogeneous(scat_len=200.0, g=0.875)
    eff.effective_scattering = True
    a = O.propagate(geo, geom, src, seed=3, want_fates=True)
    b = O.propagate(geo, eff, src, seed=3, want_fates=True)
    assert a.hit > 300 and np.array_equal(a.hits, b.hits) and np.array_equal(a.fates, b.fates)
    # without the flag the same 200 m table means eight times fewer scatters
    c = O.propagate(geo, W.ice_homogeneous(scat_len=200.0, g=0.875), src, seed=3)
    assert c.flights < 0.4 * a.flights


def test_closed_forms_with_effective_lengths():
    # lambda_e = 250 m, g = 0.9, lambda_a = 100 m: scatters per photon geometric with mean lambda_a/lambda_s = 4
    # (lambda_s = 25 m), mean displacement along the start direction 1/(a + 1/lambda_e) = 71.4286 m
    n = 200000
    geo = W.Geometry(xyz=np.array([[1.0e5, 0.0, 0.0]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous(scat_len=250.0, cos_cherenkov=1.0)
    ice.effective_scattering = True
    src = W.pencil_beam([0, 0, 0], [0, 0, 1], float(n))
    r = O.propagate(geo, ice, src, seed=8, brute_force=True, want_fates=True)
    lam_s = 250.0 * (1.0 - float(np.float32(0.9)))
    assert r.flights / n == pytest.approx(1.0 + 100.0 / lam_s, rel=0.01)
    expect = 1.0 / (0.01 + 1.0 / 250.0)
    assert expect == pytest.approx(71.4286, abs=1e-4)
    z = r.fates["z"]
    assert z.mean() == pytest.approx(expect, abs=4 * z.std() / math.sqrt(n))
    # layered: the first-scatter depth CDF of a vertical beam with absorption off is 1 - exp(-sum (1-g)^-1 dz/lambda_e)
    lay = W.ice_layered()
    lay.effective_scattering = True
    tau = 1.3
    s = O.walk(lay, "scat", 100.0, -1.0, tau * (1.0 - float(np.float32(lay.g))))
    # numerical integral of dz / lambda_e down to the end point reproduces tau (1 - g)
    zs = np.linspace(100.0, 100.0 - s, 200001)
    lam = np.array([lay.scat_len[O.layer_of(lay, float(zz))] for zz in zs[::200]])
    integral = np.trapezoid(1.0 / np.repeat(lam, 200)[: len(zs) - 1], dx=s / (len(zs) - 1))
    assert integral == pytest.approx(tau * (1.0 - float(np.float32(lay.g))), rel=2e-3)
