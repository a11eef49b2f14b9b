"""Pins for the whole oracle propagation loop against closed forms (BASELINE.json north_star:
unscattered survival, mean free path, HG mean cosine, arrival time >= d n/c, photon-count
conservation, brute force on a single string)."""
import math

import numpy as np
import pytest
from scipy import stats

from oracle import oracle as O
from paper_2405_05700_b200 import workloads as W

V = W.C_VACUUM / float(np.float32(W.N_GROUP))  # group velocity m/ns
FAR = W.Geometry(xyz=np.array([[1.0e7, 0.0, 0.0]], np.float32), radius=0.1651)  # no DOM in reach


@pytest.fixture(scope="module")
def homog_run():
    ice = W.ice_homogeneous(cos_cherenkov=1.0)  # pencil beam along the source axis
    axis = np.array([0.3, -0.5, 0.81])
    src = W.pencil_beam([1.0, 2.0, 3.0], axis, 4.0e5, t0=12.5)
    r = O.propagate(FAR, ice, src, seed=17, want_fates=True, brute_force=True)
    return ice, src, r


def test_conservation_and_no_aborts(homog_run):
    _, _, r = homog_run
    assert r.photons == 400000
    assert r.photons == r.absorbed + r.hit + r.aborted
    assert r.aborted == 0 and r.hit == 0
    assert r.flights == int(r.fates["n_flights"].sum())


def test_flights_per_photon_geometric(homog_run):
    # scatters per photon geometric with success prob p = (1/la)/(1/la + 1/ls) = 0.2: mean flights 5
    _, _, r = homog_run
    n = r.fates["n_flights"].astype(np.int64)
    assert n.mean() == pytest.approx(5.0, abs=4 * math.sqrt(20.0 / len(n)))
    kmax = 40
    obs = np.bincount(np.minimum(n, kmax), minlength=kmax + 1)[1:]
    p = 0.2 * 0.8 ** np.arange(kmax)
    p[-1] = 0.8 ** (kmax - 1)  # tail pooled
    chi2 = ((obs - len(n) * p) ** 2 / (len(n) * p)).sum()
    assert stats.chi2.sf(chi2, kmax - 1) > 1e-3


def test_total_path_exponential_with_absorption_length(homog_run):
    _, _, r = homog_run
    path = r.fates["path_m"]
    assert path.mean() == pytest.approx(100.0, abs=4 * 100.0 / math.sqrt(len(path)))
    assert stats.kstest(path, "expon", args=(0, 100.0)).pvalue > 1e-3


def test_time_is_path_over_group_velocity(homog_run):
    _, _, r = homog_run
    assert np.allclose(r.fates["time_ns"], 12.5 + r.fates["path_m"] / V, rtol=0, atol=1e-8)


def test_mean_displacement_along_initial_direction(homog_run):
    # <displacement . d0> = 1 / (a + b (1 - g)) = 1 / (0.01 + 0.04 * 0.1) = 71.4286 m
    _, src, r = homog_run
    d0 = src.src[0, 3:6].astype(np.float64)
    d0 /= np.linalg.norm(d0)
    disp = np.stack([r.fates["x"] - 1.0, r.fates["y"] - 2.0, r.fates["z"] - 3.0], axis=1)
    along = disp @ d0
    assert along.mean() == pytest.approx(1.0 / (0.01 + 0.04 * (1 - 0.9)), abs=4 * along.std() / math.sqrt(len(along)))
    # no preferred transverse direction
    e1 = np.cross(d0, [0, 0, 1.0])
    e1 /= np.linalg.norm(e1)
    e2 = np.cross(d0, e1)
    for e in (e1, e2):
        t = disp @ e
        assert abs(t.mean()) < 4 * t.std() / math.sqrt(len(t))


def test_scattering_length_is_the_mean_free_path():
    # absorption (almost) off: first flight length = total path of photons that are absorbed in
    # flight 1 is awkward, so instead make absorption strong and scattering the test subject:
    # P(n_flights = 1) = a/(a+b); with la = 10, ls = 40: 0.8; mean flights 1.25
    ice = W.ice_homogeneous(abs_len=10.0, scat_len=40.0, cos_cherenkov=1.0)
    r = O.propagate(FAR, ice, W.pencil_beam([0, 0, 0], [0, 0, 1], 2.0e5), seed=3, want_fates=True, brute_force=True)
    n = r.fates["n_flights"]
    assert (n == 1).mean() == pytest.approx(0.8, abs=4 * math.sqrt(0.8 * 0.2 / len(n)))
    assert r.fates["path_m"].mean() == pytest.approx(10.0, abs=4 * 10 / math.sqrt(len(n)))


@pytest.mark.parametrize("dist,frac,frac_noscat,t_ns", [(20.0, 0.370929, 0.820084, 89.3188),
                                                       (50.0, 0.082765, 0.607533, 224.4123)])
def test_unscattered_survival_to_a_sphere(dist, frac, frac_noscat, t_ns):
    # pencil beam aimed at a DOM centre at distance d: fraction of photons that hit
    # with zero scatters = exp(-(d-R)(1/la + 1/ls)); they arrive at exactly (d-R)/v.
    R = 0.1651
    geo = W.Geometry(xyz=np.array([[dist, 0.0, 0.0]], np.float32), radius=R)
    src = W.pencil_beam([0, 0, 0], [1, 0, 0], 2.0e5)
    ice = W.ice_homogeneous(cos_cherenkov=1.0)
    r = O.propagate(geo, ice, src, seed=5, want_fates=True, brute_force=True)
    f = r.fates
    direct = (f["fate"] == O.FATE_HIT) & (f["n_flights"] == 1)
    n = len(f)
    Rf = float(np.float32(R))
    expect = math.exp(-(dist - Rf) * (1 / 100.0 + 1 / 25.0))
    assert expect == pytest.approx(frac, abs=2e-6)
    assert direct.mean() == pytest.approx(expect, abs=4 * math.sqrt(expect * (1 - expect) / n))
    assert np.allclose(f["time_ns"][direct], (dist - Rf) / V, atol=1e-9)
    assert (dist - Rf) / V == pytest.approx(t_ns, abs=2e-4)
    assert np.all(f["dom"][direct] == 0)
    assert len(r.hits) == int((f["fate"] == O.FATE_HIT).sum()) == r.hit
    # scattering off: every surviving photon hits: exp(-(d-R)/la)
    ice2 = W.ice_homogeneous(scat_len=1.0e30, cos_cherenkov=1.0)
    r2 = O.propagate(geo, ice2, src, seed=6, want_fates=True, brute_force=True)
    e2 = math.exp(-(dist - Rf) / 100.0)
    assert e2 == pytest.approx(frac_noscat, abs=2e-6)
    assert r2.hit / r2.photons == pytest.approx(e2, abs=4 * math.sqrt(e2 * (1 - e2) / n))
    assert np.all(r2.fates["n_flights"] == 1)
    assert np.allclose(r2.hits["time_ns"], (dist - Rf) / V, atol=1e-9)


def test_cherenkov_cone_emission_and_azimuth_uniformity():
    # cos_cherenkov = 0: photons leave in the plane perpendicular to the axis, uniform in azimuth.
    # A DOM in that plane at distance d subtends |alpha| <= asin(R/d); unscattered hit fraction =
    # (1/2pi) int exp(-t(alpha)(a+b)) d alpha, t(alpha) = d cos(alpha) - sqrt(R^2 - d^2 sin^2(alpha)).
    d, R = 5.0, 0.5
    ice = W.ice_homogeneous(cos_cherenkov=0.0)
    src = W.pencil_beam([0, 0, 0], [0, 0, 1], 4.0e5)
    from scipy import integrate
    am = math.asin(R / d)
    k = 1 / 100.0 + 1 / 25.0
    expect = integrate.quad(lambda a: math.exp(-k * (d * math.cos(a) - math.sqrt(max(0.0, R * R - (d * math.sin(a)) ** 2)))),
                            -am, am)[0] / (2 * math.pi)
    tot = 0
    for ang in (0.0, 2.0, 4.5):  # three DOM azimuths: the emission azimuth must be uniform
        geo = W.Geometry(xyz=np.array([[d * math.cos(ang), d * math.sin(ang), 0.0]], np.float32), radius=R)
        r = O.propagate(geo, ice, src, seed=9, want_fates=True, brute_force=True)
        f = r.fates
        direct = ((f["fate"] == O.FATE_HIT) & (f["n_flights"] == 1)).mean()
        assert direct == pytest.approx(expect, abs=4.5 * math.sqrt(expect / len(f)))
        tot += direct
    # Cherenkov angle proper: with cos_c = cos(41.2 deg) the first flight makes 41.2 deg with the axis
    ice = W.ice_homogeneous(abs_len=1e-3, scat_len=1e30)  # absorbed at once: end point = p0 + d * s
    r = O.propagate(FAR, ice, W.pencil_beam([0, 0, 0], [0, 0, 1], 2.0e4), seed=1, want_fates=True, brute_force=True)
    f = r.fates
    cosang = f["z"] / np.sqrt(f["x"] ** 2 + f["y"] ** 2 + f["z"] ** 2)
    assert np.allclose(cosang, math.cos(math.radians(41.2)), atol=2e-7)
    phi = np.arctan2(f["y"], f["x"])
    assert stats.kstest((phi + math.pi) / (2 * math.pi), "uniform").pvalue > 1e-3


def test_layered_vertical_beam_absorption_depth_cdf():
    # scattering off, vertical pencil beam downwards from z = 495: absorbed-depth CDF is
    # 1 - exp(-sum a_i dz_i), piecewise (SURVEY 8(c) "Layer walk" pin).  CDF built here from the table only.
    ice = W.ice_layered(cos_cherenkov=1.0)
    ice.scat_len = np.full(100, 1.0e30, np.float32)
    z0 = 495.0
    r = O.propagate(FAR, ice, W.pencil_beam([0, 0, z0], [0, 0, -1], 2.0e5), seed=2, want_fates=True, brute_force=True)
    path = z0 - r.fates["z"]
    assert np.allclose(path, r.fates["path_m"], atol=1e-9)
    a = 1.0 / ice.abs_len.astype(np.float64)
    edges = np.concatenate([[0.0], 5.0 + 10.0 * np.arange(100)])  # path length at which each boundary is crossed
    tau_edges = np.concatenate([[0.0], np.cumsum(a[:100] * np.diff(np.concatenate([edges, [1e9]]))[:100])])

    def cdf(s, cosz=1.0):  # s = vertical drop; optical depth along the ray is tau_vertical / |cos|
        s = np.asarray(s, dtype=np.float64)
        i = np.clip(np.searchsorted(edges, s, side="right") - 1, 0, 99)
        tau = tau_edges[i] + a[i] * (s - edges[i])
        return 1.0 - np.exp(-tau / cosz)

    assert stats.kstest(path, cdf).pvalue > 1e-3
    # oblique beam: same with path = drop / |cos|
    dz = -0.6
    r = O.propagate(FAR, ice, W.pencil_beam([0, 0, z0], [0.8, 0, dz], 2.0e5), seed=4, want_fates=True, brute_force=True)
    assert stats.kstest(r.fates["path_m"] * abs(dz), lambda x: cdf(x, abs(dz))).pvalue > 1e-3


def _vertical_tau_cdf(ice, z0):
    """CDF of the vertical drop at which a downward beam from z0 = 495 is absorbed, from the table only."""
    a = 1.0 / ice.abs_len.astype(np.float64)
    edges = np.concatenate([[0.0], 5.0 + 10.0 * np.arange(100)])
    tau_edges = np.concatenate([[0.0], np.cumsum(a[:100] * np.diff(np.concatenate([edges, [1e9]]))[:100])])

    def cdf(s):
        s = np.asarray(s, dtype=np.float64)
        i = np.clip(np.searchsorted(edges, s, side="right") - 1, 0, 99)
        return 1.0 - np.exp(-(tau_edges[i] + a[i] * (s - edges[i])))

    return cdf


def test_layered_absorption_budget_across_many_flights_forward_peaked():
    # Step 8's bookkeeping (tau_a -= optical depth of the stretch just flown) in LAYERED ice with scattering ON
    # (PAPER.md:31 layers with their own coefficients + PAPER.md:33 "repeated until ... absorbed").  With
    # g = 0.999999 every scatter leaves the direction unchanged to ~1e-3 rad, so the photon flies straight down in
    # many flights (mean free path 5-60 m) and the total path must still follow 1 - exp(-sum a_i dz_i), a CDF built
    # from the table only.  Charging the budget for the wrong stretch of ice (e.g. evaluating the optical depth
    # after the position advance) fails this with p = 0.
    ice = W.ice_layered(cos_cherenkov=1.0, g=0.999999)
    z0 = 495.0
    r = O.propagate(FAR, ice, W.pencil_beam([0, 0, z0], [0, 0, -1], 2.0e5), seed=11, want_fates=True, brute_force=True)
    f = r.fates
    assert f["n_flights"].mean() > 3.0  # the budget really is carried over several flights
    # straight down: the Henyey-Greenstein tail leaves a few 1e-5 of the photons with one sizeable deflection
    assert np.quantile(np.abs(f["path_m"] - (z0 - f["z"])), 0.999) < 1e-3
    assert stats.kstest(f["path_m"], _vertical_tau_cdf(ice, z0)).pvalue > 1e-3


def test_layered_proportional_tables_flights_geometric_whatever_the_path():
    # If abs_len = 4 scat_len in EVERY layer, each interaction is an absorption with probability
    # a/(a+b) = 1/5 wherever it happens and whatever the direction: flights per photon are geometric with mean
    # exactly 5 in any layered ice.  Only correct carry-over of the absorption budget between flights and across
    # layer boundaries gives that (a mis-ordered step 8 gives 4.56).  C1's cascades, the real Cherenkov cone, g = 0.9.
    ice = W.ice_layered()
    ice.abs_len = (4.0 * ice.scat_len.astype(np.float64)).astype(np.float32)
    assert np.array_equal(ice.abs_len.astype(np.float64), 4.0 * ice.scat_len.astype(np.float64))  # x4 is exact in fp32
    src = W.sources_c1().subset(slice(0, 40))
    src.src[:, 7] = 0.5  # GeV: 5000 photons per cascade
    r = O.propagate(FAR, ice, src, seed=13, want_fates=True, brute_force=True)
    n = r.fates["n_flights"].astype(np.int64)
    assert len(n) == 40 * 5000 and r.aborted == 0 and r.hit == 0
    assert n.mean() == pytest.approx(5.0, abs=4 * math.sqrt(20.0 / len(n)))
    kmax = 40
    obs = np.bincount(np.minimum(n, kmax), minlength=kmax + 1)[1:]
    p = 0.2 * 0.8 ** np.arange(kmax)
    p[-1] = 0.8 ** (kmax - 1)
    chi2 = ((obs - len(n) * p) ** 2 / (len(n) * p)).sum()
    assert stats.chi2.sf(chi2, kmax - 1) > 1e-3
    # and the layers are really visited: the photons end in many different layers
    assert len(np.unique(np.floor((500.0 - r.fates["z"]) / 10.0))) > 30


def test_causality_and_brute_force_on_single_string():
    # C0 geometry with oversized DOMs (1.5 m) so that there are enough hits to look at
    geo, ice = W.geometry_single_string(radius=1.5), W.ice_homogeneous()
    src = W.sources_c0(seed=0, n_photons=3.0e5, toward_string=True)
    rb = O.propagate(geo, ice, src, seed=0, brute_force=True)
    rl = O.propagate(geo, ice, src, seed=0, brute_force=False)
    assert rb.hit > 20
    assert np.array_equal(rb.hits, rl.hits)  # exact pre-filter == brute-force enumeration
    p = src.src[0, :3].astype(np.float64)
    c = geo.xyz[rb.hits["dom_id"]].astype(np.float64)
    dmin = np.linalg.norm(c - p, axis=1) - float(np.float32(geo.radius))
    assert np.all(rb.hits["time_ns"] - src.src[0, 6] >= dmin / V - 1e-9)  # arrival time >= d n_group / c
    assert rb.photons == rb.absorbed + rb.hit and rb.aborted == 0


def test_prefilter_identical_on_layered_full_detector_subsample():
    geo, ice = W.geometry_full(), W.ice_layered()
    src = W.sources_c1().subset(slice(0, 8))
    cnt = np.minimum(np.array([O.photon_count(e) for e in src.src[:, 7]], np.uint64), 3000)
    rb = O.propagate(geo, ice, src, seed=0, count=cnt, brute_force=True, want_fates=True)
    rl = O.propagate(geo, ice, src, seed=0, count=cnt, brute_force=False, want_fates=True)
    assert np.array_equal(rb.hits, rl.hits)
    assert np.array_equal(rb.fates, rl.fates)


def test_selection_replay_and_thread_invariance():
    # counter-based streams: any subset of photons replays bit-identically
    geo, ice = W.geometry_single_string(), W.ice_homogeneous()
    src = W.sources_c0(seed=0, n_photons=2.0e4, toward_string=True)
    full = O.propagate(geo, ice, src, seed=3, want_fates=True, n_threads=8)
    one = O.propagate(geo, ice, src, seed=3, want_fates=True, n_threads=1)
    assert np.array_equal(full.fates, one.fates) and np.array_equal(full.hits, one.hits)
    sub = O.propagate(geo, ice, src, seed=3, want_fates=True, stride=7, offset=3)
    assert np.array_equal(sub.fates, full.fates[3::7])
    win = O.propagate(geo, ice, src, seed=3, want_fates=True, first=[1000], count=[500])
    assert np.array_equal(win.fates, full.fates[1000:1500])
    other = O.propagate(geo, ice, src, seed=4, want_fates=True)
    assert not np.array_equal(other.fates["x"], full.fates["x"])


def test_hit_probability_scale_inside_array():
    # optically-thin estimate n pi R^2 lambda_abs ~ 4e-5 hits per photon: order of magnitude only
    geo, ice = W.geometry_full(), W.ice_layered()
    src = W.sources_c1()
    r = O.propagate(geo, ice, src, seed=0, stride=4096)
    rate = r.hit / r.photons
    assert 4e-6 < rate < 4e-4
    assert r.aborted == 0
