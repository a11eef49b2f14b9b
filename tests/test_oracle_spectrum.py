"""Pins of the oracle's wavelength bins (NEXT-2, R-21; PAPER.md:33 names the wavelength among the things
the photoelectron probability depends on) against closed forms."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2405_05700_b200 import workloads as W

C = W.C_VACUUM


def two_bins(w0=0.25, sa=(2.0, 0.5), sb=(1.0, 1.0), ng=(1.30, 1.40), acc=(1.0, 1.0)):
    f = lambda v: np.asarray(v, np.float32)
    return W.Spectrum(f([w0, 1.0]), f(sa), f(sb), f(ng), f(acc))


def test_one_bin_with_unit_scales_is_the_monochromatic_path_bit_for_bit():
    geo, ice = W.geometry_full(radius=1.0), W.ice_layered()
    src = W.sources_c1().subset(slice(0, 10))
    src.src[:, 7] = 1.0
    one = W.Spectrum(*(np.asarray(v, np.float32) for v in ([1.0], [1.0], [1.0], [ice.n_group], [1.0])))
    a = O.propagate(geo, ice, src, seed=1, want_fates=True)
    b = O.propagate(geo, ice, src, seed=1, want_fates=True, spectrum=one)
    assert a.hit > 50 and np.array_equal(a.hits, b.hits) and np.array_equal(a.fates, b.fates)


def test_absorption_and_bin_frequencies():
    # scattering off, no DOM in reach: a photon of bin j travels Exp(lambda_a / abs_scale_j); bins drawn with w = (1/4, 3/4)
    n = 400000
    geo = W.Geometry(xyz=np.array([[1.0e6, 0.0, 0.0]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous(scat_len=1.0e30, cos_cherenkov=1.0)
    src = W.pencil_beam([0, 0, 0], [0, 0, 1], float(n))
    r = O.propagate(geo, ice, src, seed=13, brute_force=True, want_fates=True, spectrum=two_bins())
    path = r.fates["path_m"]
    expect = 0.25 * 50.0 + 0.75 * 200.0
    assert path.mean() == pytest.approx(expect, abs=4 * path.std() / math.sqrt(n))
    # the speed tells the bin: time = path n_j / c
    ng = r.fates["time_ns"] * C / path
    is0 = np.abs(ng - float(np.float32(1.30))) < 1e-6
    is1 = np.abs(ng - float(np.float32(1.40))) < 1e-6
    assert np.all(is0 | is1)
    assert is0.mean() == pytest.approx(0.25, abs=4 * math.sqrt(0.25 * 0.75 / n))
    assert path[is0].mean() == pytest.approx(50.0, rel=0.01) and path[is1].mean() == pytest.approx(200.0, rel=0.01)
    # the bin is the uniform made of the low 9 bits of words 0, 1, 2 of block 0, against the cdf
    assert O.spectrum_word((0x1FF, 0, 0, 0)) == 0xFF800000 and O.spectrum_word((0xFFFFFE00, 0x101, 0xFFFFFFFF, 7)) == \
        (0x101 << 14) | (0x1FF << 5)
    for i in range(200):
        w = O.philox4x32_10((i, 0, 0, 0), (13, 0))
        x = ((w[0] & 0x1FF) << 23) | ((w[1] & 0x1FF) << 14) | ((w[2] & 0x1FF) << 5)
        assert x == O.spectrum_word(w)
        assert bool(is0[i]) == (O.uniform(x) < 0.25)
    # ... and is independent of the uniforms that share the block (they use the top 23 bits of each word)
    az = np.array([O.uniform(O.philox4x32_10((i, 0, 0, 0), (13, 0))[0]) for i in range(4000)])
    assert abs(np.corrcoef(az, is0[:4000].astype(float))[0, 1]) < 0.06


def test_wavelength_uniform_is_independent_of_the_blocks_other_uniforms():
    """R-21 takes the wavelength uniform from the low 9 bits of words 0, 1, 2 of Philox block 0; the four uniforms of
    R-3 use the top 23 bits of a word.  (a) The two bit sets are disjoint, exactly: changing one never changes the
    other.  (b) Jointly uniform: chi-square of the 8 x 8 table of (wavelength uniform, each of the four uniforms) over
    1e5 blocks, and of the wavelength uniform alone."""
    rng = np.random.default_rng(5)
    for _ in range(200):
        w = [int(x) for x in rng.integers(0, 2 ** 32, 4)]
        low = [int(x) for x in rng.integers(0, 512, 4)]
        w_low = [(a & 0xFFFFFE00) | b for a, b in zip(w, low)]         # other low bits: the four uniforms stay
        assert [O.uniform(a) for a in w] == [O.uniform(a) for a in w_low]
        high = [int(x) << 9 for x in rng.integers(0, 2 ** 23, 4)]
        w_high = [(a & 0x1FF) | b for a, b in zip(w, high)]            # other high bits: the wavelength word stays
        assert O.spectrum_word(w) == O.spectrum_word(w_high)
        assert O.spectrum_word(w) == O.spectrum_word((w[0], w[1], w[2], w[3] ^ 0xFFFFFFFF))  # word 3 takes no part
    n = 100000
    lam = np.empty(n)
    u4 = np.empty((n, 4))
    for i in range(n):
        w = O.philox4x32_10((i, 3, 7, 0), (21, 0))
        lam[i] = O.uniform(O.spectrum_word(w))
        u4[i] = [O.uniform(x) for x in w]
    from scipy import stats
    bl = np.minimum((lam * 8).astype(int), 7)
    assert stats.chisquare(np.bincount(bl, minlength=8)).pvalue > 1e-3
    for k in range(4):
        bu = np.minimum((u4[:, k] * 8).astype(int), 7)
        table = np.zeros((8, 8))
        np.add.at(table, (bl, bu), 1)
        chi2, p, _, _ = stats.chi2_contingency(table)
        assert p > 1e-3, (k, chi2, p)
        assert abs(np.corrcoef(lam, u4[:, k])[0, 1]) < 4.0 / math.sqrt(n)


def test_scattering_scale_and_arrival_times():
    # scattering scaled by (2, 0.5): flights per photon 1 + lambda_a_j / lambda_s_j with lambda_s_j = 25 / scat_scale_j
    n = 200000
    geo = W.Geometry(xyz=np.array([[1.0e6, 0.0, 0.0]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous(cos_cherenkov=1.0)
    src = W.pencil_beam([0, 0, 0], [0, 0, 1], float(n))
    sp = two_bins(w0=0.5, sa=(1.0, 1.0), sb=(2.0, 0.5))
    r = O.propagate(geo, ice, src, seed=14, brute_force=True, want_fates=True, spectrum=sp)
    ng = r.fates["time_ns"] * C / r.fates["path_m"]
    is0 = np.abs(ng - float(np.float32(1.30))) < 1e-6
    nf = r.fates["n_flights"].astype(float)
    assert nf[is0].mean() == pytest.approx(1 + 100.0 / 12.5, rel=0.02)
    assert nf[~is0].mean() == pytest.approx(1 + 100.0 / 50.0, rel=0.02)
    # a DOM on a pencil beam, scattering off: two arrival times (d-R) n_j / c, frequencies ~ w_j exp(-(d-R) a_j)
    dist = 40.0
    R = float(np.float32(W.DOM_RADIUS))
    geo2 = W.Geometry(xyz=np.array([[0.0, 0.0, dist]], np.float32), radius=W.DOM_RADIUS)
    ice2 = W.ice_homogeneous(scat_len=1.0e30, cos_cherenkov=1.0)
    r2 = O.propagate(geo2, ice2, src, seed=15, brute_force=True, spectrum=two_bins())
    t = r2.hits["time_ns"]
    t0, t1 = (dist - R) * float(np.float32(1.30)) / C, (dist - R) * float(np.float32(1.40)) / C
    e0, e1 = 0.25 * math.exp(-(dist - R) / 50.0), 0.75 * math.exp(-(dist - R) / 200.0)
    n0, n1 = int((np.abs(t - t0) < 1e-6).sum()), int((np.abs(t - t1) < 1e-6).sum())
    assert n0 + n1 == len(t)
    assert n0 / n == pytest.approx(e0, abs=4 * math.sqrt(e0 / n)) and n1 / n == pytest.approx(e1, abs=4 * math.sqrt(e1 / n))


def test_acceptance_scale():
    # photons born inside a DOM (axis +z): accepted fraction = sum_j w_j min(1, p(cos theta_c) acc_scale_j)
    n = 200000
    geo = W.Geometry(xyz=np.array([[0.0, 0.0, 0.0]], np.float32), radius=W.DOM_RADIUS)
    ice = W.ice_homogeneous()
    src = W.pencil_beam([0.01, 0.0, 0.02], [0, 0, 1], float(n))
    sp = two_bins(w0=0.25, sa=(1.0, 1.0), acc=(0.5, 2.0))
    eta = float(np.float32(ice.cos_cherenkov))
    c = [float(np.float32(x)) for x in W.ACCEPTANCE_COEF]
    p = c[0] + c[1] * eta + c[2] * eta * eta
    expect = 0.25 * min(1.0, 0.5 * p) + 0.75 * min(1.0, 2.0 * p)
    r = O.propagate(geo, ice, src, seed=16, brute_force=True, acceptance_mode="probabilistic",
                    acceptance_coef=W.ACCEPTANCE_COEF, spectrum=sp)
    assert r.hit / n == pytest.approx(expect, abs=4 * math.sqrt(expect * (1 - expect) / n))
    r2 = O.propagate(geo, ice, src, seed=16, brute_force=True, acceptance_mode="weighted",
                     acceptance_coef=W.ACCEPTANCE_COEF, spectrum=sp)
    w = r2.hits["weight"]
    assert set(np.round(w, 6)) == {round(min(1.0, 0.5 * p), 6), 1.0}
    assert w.mean() == pytest.approx(expect, abs=4 * w.std() / math.sqrt(n))
