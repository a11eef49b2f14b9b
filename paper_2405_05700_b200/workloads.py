"""Seeded synthetic input generators shared by the CUDA path, the oracle and the tests.

This module holds NO method arithmetic (no Philox, no photon counting, no
propagation): it only draws geometry, ice tables and light-source lists with
``numpy.random.default_rng(seed)``.  Everything it returns is float32 / uint32
so that the CUDA library and the fp64 oracle consume bit-identical inputs.

Stand-ins, not data: the paper's real inputs (IceCube geometry file, measured
ice tables, Corsika/Proposal output) are not available.
Shapes and distributions follow BASELINE.json configs[0..4] (named C0..C4) and
the readings listed in DESIGN.md section 3 (SURVEY.md section 8(c)/(d),
PR-11, PR-12 and the C2/C4 normalisation).

Conventions: metres, nanoseconds, GeV; z up; origin at 1950 m depth, so
``depth = 1950 - z`` (PAPER.md:9 gives 1450-2450 m).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

C_VACUUM = 0.299792458  # m/ns
DOM_RADIUS = 0.1651  # m, BASELINE.json configs[0]
N_GROUP = 1.35  # BASELINE.json configs[0]
HG_G = 0.9  # BASELINE.json configs[0]
CHERENKOV_DEG = 41.2  # BASELINE.json configs[0]
PHOTONS_PER_GEV = 1.0e4  # BASELINE.json configs[1]
DEPTH_ORIGIN = 1950.0  # m
STRING_PITCH = 125.0  # m, BASELINE.json configs[1]
DOM_PITCH = 17.0  # m
DOMS_PER_STRING = 60
# Stand-in angular acceptance (R-17; the real DOM acceptance curves are not available): coefficients of
# p(eta) = 0.35 + 0.5 eta + 0.15 eta^2, eta = cosine between the photon's travel direction and +z; p(-1) = 0 (photon
# arriving on the back of the down-looking PMT), p(+1) = 1, monotone in between.
ACCEPTANCE_COEF = (0.35, 0.5, 0.15)


@dataclass
class Geometry:
    """DOM positions; ``dom_id`` is the row index of ``xyz``."""

    xyz: np.ndarray  # float32 [n_dom, 3]
    radius: float = DOM_RADIUS

    @property
    def n_dom(self) -> int:
        return int(self.xyz.shape[0])


@dataclass
class Ice:
    """Layered ice table.  Layer i spans z in (z_top-(i+1)dz, z_top-i*dz]; the first and
    last layer extend to +-infinity (reading R-6)."""

    abs_len: np.ndarray  # float32 [n_layers], metres
    scat_len: np.ndarray  # float32 [n_layers], metres (geometric, reading R-7)
    z_top: float = 500.0
    dz: float = 10.0
    g: float = HG_G
    n_group: float = N_GROUP
    cos_cherenkov: float = float(np.float32(math.cos(math.radians(CHERENKOV_DEG))))
    photons_per_GeV: float = PHOTONS_PER_GEV
    effective_scattering: bool = False  # scat_len holds lambda_e = lambda_s / (1 - g) (R-20)

    @property
    def n_layers(self) -> int:
        return int(self.abs_len.shape[0])


@dataclass
class Spectrum:
    """Wavelength bins (R-21): per bin the cumulative probability, the factors on the absorption and
    scattering coefficients, the group index and the factor on the acceptance.  A stand-in: the real Cherenkov
    spectrum, ice dispersion and DOM efficiency curves are not available."""

    cdf: np.ndarray  # float32 [n], non-decreasing, last = 1
    abs_scale: np.ndarray
    scat_scale: np.ndarray
    n_group: np.ndarray
    acc_scale: np.ndarray


def spectrum_standin(n_bins: int = 8) -> Spectrum:
    """8 bins from blue to red: bluer light is drawn more often (1/lambda^2-like weights), scatters more and is
    absorbed less in the blue-green, travels a little slower; the acceptance falls off towards both ends."""
    x = (np.arange(n_bins) + 0.5) / n_bins  # 0 = blue end, 1 = red end
    w = 1.0 / (1.0 + x) ** 2
    cdf = np.cumsum(w) / w.sum()
    cdf[-1] = 1.0
    return Spectrum(cdf.astype(np.float32), (0.6 + 1.6 * x ** 2).astype(np.float32), (1.25 - 0.5 * x).astype(np.float32),
                    (1.38 - 0.05 * x).astype(np.float32), (1.0 - 1.6 * (x - 0.4) ** 2).astype(np.float32))


@dataclass
class Sources:
    """A list of light sources.  ``src`` rows are (x, y, z, dx, dy, dz, t_ns, E_GeV)."""

    src: np.ndarray  # float32 [n, 8]
    event_id: np.ndarray  # uint32 [n]
    source_id: np.ndarray  # uint32 [n]  (index of the source within its event)
    meta: dict = field(default_factory=dict)
    length: np.ndarray | None = None  # float32 [n] metres: track segments (R-18); None = point sources

    def __len__(self) -> int:
        return int(self.src.shape[0])

    def subset(self, sel) -> "Sources":
        return Sources(np.ascontiguousarray(self.src[sel]), np.ascontiguousarray(self.event_id[sel]),
                       np.ascontiguousarray(self.source_id[sel]), dict(self.meta),
                       None if self.length is None else np.ascontiguousarray(self.length[sel]))


# --------------------------------------------------------------------------------------
# geometry
# --------------------------------------------------------------------------------------
def _string_z() -> np.ndarray:
    """DOM k of a string sits at depth 1450 + 17k m (k = 0..59)."""
    depth = 1450.0 + DOM_PITCH * np.arange(DOMS_PER_STRING, dtype=np.float64)
    return DEPTH_ORIGIN - depth


def hex_string_xy(n_strings: int = 86, pitch: float = STRING_PITCH) -> np.ndarray:
    """First ``n_strings`` points of a triangular lattice, sorted by the integer key
    (q^2+qr+r^2, r, q) (reading R-11)."""
    pts = []
    m = 12
    for q in range(-m, m + 1):
        for r in range(-m, m + 1):
            pts.append((q * q + q * r + r * r, r, q))
    pts.sort()
    pts = pts[:n_strings]
    xy = np.empty((n_strings, 2), dtype=np.float64)
    for i, (_, r, q) in enumerate(pts):
        xy[i, 0] = pitch * (q + 0.5 * r)
        xy[i, 1] = pitch * (math.sqrt(3.0) / 2.0) * r
    return xy


def geometry_strings(xy: np.ndarray, radius: float = DOM_RADIUS) -> Geometry:
    z = _string_z()
    n_s = xy.shape[0]
    xyz = np.empty((n_s * DOMS_PER_STRING, 3), dtype=np.float32)
    for s in range(n_s):
        sl = slice(s * DOMS_PER_STRING, (s + 1) * DOMS_PER_STRING)
        xyz[sl, 0] = np.float32(xy[s, 0])
        xyz[sl, 1] = np.float32(xy[s, 1])
        xyz[sl, 2] = z.astype(np.float32)
    return Geometry(xyz=xyz, radius=radius)


def geometry_single_string(radius: float = DOM_RADIUS) -> Geometry:
    """C0: one vertical string of 60 DOMs at x = y = 0."""
    return geometry_strings(np.zeros((1, 2)), radius)


def geometry_full(radius: float = DOM_RADIUS) -> Geometry:
    """C1..C4: 86 strings x 60 DOMs = 5160 DOMs; dom_id = 60*string + k."""
    return geometry_strings(hex_string_xy(86), radius)


# --------------------------------------------------------------------------------------
# ice
# --------------------------------------------------------------------------------------
def ice_homogeneous(abs_len: float = 100.0, scat_len: float = 25.0, g: float = HG_G, **kw) -> Ice:
    """C0: a single layer, which by R-6 extends to +-infinity."""
    return Ice(abs_len=np.array([abs_len], dtype=np.float32), scat_len=np.array([scat_len], dtype=np.float32),
               g=g, **kw)


def ice_layered(seed: int = 2405, n_layers: int = 100, **kw) -> Ice:
    """C1 profile (reading R-12): one smooth seeded profile drives both lengths; absorption
    20-250 m, scattering 5-60 m; dust layer at depth [2000, 2100) divides both by 5."""
    rng = np.random.default_rng(seed)
    periods = np.array([1000.0, 500.0, 250.0, 125.0])
    phases = rng.uniform(0.0, 2.0 * math.pi, size=4)
    depth_c = 1450.0 + 10.0 * (np.arange(n_layers) + 0.5)
    s = np.zeros(n_layers)
    for k in range(4):
        s += (1.0 / (k + 1)) * np.sin(2.0 * math.pi * depth_c / periods[k] + phases[k])
    s = (s - s.min()) / (s.max() - s.min())
    lam_a = 20.0 + 230.0 * s
    lam_s = 5.0 + 55.0 * s
    dust = (depth_c >= 2000.0) & (depth_c < 2100.0)
    lam_a[dust] /= 5.0
    lam_s[dust] /= 5.0
    return Ice(abs_len=lam_a.astype(np.float32), scat_len=lam_s.astype(np.float32),
               z_top=DEPTH_ORIGIN - 1450.0, dz=10.0, **kw)


# --------------------------------------------------------------------------------------
# sources
# --------------------------------------------------------------------------------------
def _unit(v: np.ndarray) -> np.ndarray:
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _f32_unit(d: np.ndarray) -> np.ndarray:
    """Round to float32 and renormalise once more in float32 so the stored vector is as
    close to unit length as float32 allows."""
    d32 = d.astype(np.float32)
    n = np.sqrt((d32.astype(np.float64) ** 2).sum(axis=-1, keepdims=True))
    return (d32.astype(np.float64) / n).astype(np.float32)


def _pack(pos, dirs, t, e, event_id, source_id, meta=None) -> Sources:
    n = len(e)
    src = np.empty((n, 8), dtype=np.float32)
    src[:, 0:3] = np.asarray(pos, dtype=np.float64).reshape(n, 3)
    src[:, 3:6] = _f32_unit(np.asarray(dirs, dtype=np.float64).reshape(n, 3))
    src[:, 6] = t
    src[:, 7] = e
    return Sources(src, np.asarray(event_id, dtype=np.uint32), np.asarray(source_id, dtype=np.uint32), meta or {})


def travel_direction(zenith: float, azimuth: float) -> np.ndarray:
    """Zenith/azimuth name the direction the particle comes FROM (reading R-11b)."""
    return -np.array([math.sin(zenith) * math.cos(azimuth), math.sin(zenith) * math.sin(azimuth), math.cos(zenith)])


def sources_c0(seed: int = 0, n_photons: float = 1.0e5, toward_string: bool = False) -> Sources:
    """C0: one point cascade 20 m from the string at 1950 m depth, axis uniform on the sphere."""
    rng = np.random.default_rng(seed)
    cos_t = 2.0 * rng.uniform() - 1.0
    phi = 2.0 * math.pi * rng.uniform()
    sin_t = math.sqrt(1.0 - cos_t * cos_t)
    axis = np.array([sin_t * math.cos(phi), sin_t * math.sin(phi), cos_t])
    if toward_string:  # supplementary "C0-big" variant: fixed axis pointing at the string
        axis = np.array([-1.0, 0.0, 0.0])
    e = n_photons / PHOTONS_PER_GEV
    return _pack([[20.0, 0.0, 0.0]], [axis], [0.0], [e], [0], [0], {"config": "C0", "gen_seed": seed})


def _track_cascades(rng, point, direction, n_casc, half_len=500.0):
    """Cascade positions uniform along a 2*half_len segment centred on ``point``; the muon
    moves at c and reaches the start of the segment at t = 0."""
    dist = rng.uniform(-half_len, half_len, size=n_casc)
    pos = point[None, :] + dist[:, None] * direction[None, :]
    t = (dist + half_len) / C_VACUUM
    return pos, t


def sources_c1(seed: int = 1, n_casc: int = 200) -> Sources:
    """C1: one 1 km muon through the array centre, zenith 30 deg, seeded azimuth, 200
    cascades with dN/dE ~ 1/E on [1, 1e4] GeV."""
    rng = np.random.default_rng(seed)
    azimuth = 2.0 * math.pi * rng.uniform()
    d = travel_direction(math.radians(30.0), azimuth)
    pos, t = _track_cascades(rng, np.zeros(3), d, n_casc)
    e = np.exp(rng.uniform(math.log(1.0), math.log(1.0e4), size=n_casc))
    dirs = np.repeat(d[None, :], n_casc, axis=0)
    return _pack(pos, dirs, t, e, np.zeros(n_casc), np.arange(n_casc), {"config": "C1", "gen_seed": seed})


def sources_track(seed: int = 5, n_seg: int = 100, seg_len: float = 10.0, gev_per_m: float = 0.03,
                  n_casc: int = 20) -> Sources:
    """NEXT-2 stand-in (R-18): a muon through the array centre (zenith 30 deg, seeded azimuth) whose own
    Cherenkov light comes from ``n_seg`` contiguous track segments of ``seg_len`` metres (light-equivalent energy
    ``gev_per_m`` per metre), plus ``n_casc`` point cascades (length 0) with dN/dE ~ 1/E on [1, 100] GeV."""
    rng = np.random.default_rng(seed)
    azimuth = 2.0 * math.pi * rng.uniform()
    d = travel_direction(math.radians(30.0), azimuth)
    half = 0.5 * n_seg * seg_len
    start = -half + seg_len * np.arange(n_seg)
    pos = start[:, None] * d[None, :]
    t = (start + half) / C_VACUUM
    e = np.full(n_seg, gev_per_m * seg_len)
    cpos, ct = _track_cascades(rng, np.zeros(3), d, n_casc, half_len=half)
    ce = np.exp(rng.uniform(math.log(1.0), math.log(100.0), size=n_casc))
    n = n_seg + n_casc
    out = _pack(np.concatenate([pos, cpos]), np.repeat(d[None, :], n, axis=0), np.concatenate([t, ct]),
                np.concatenate([e, ce]), np.zeros(n), np.arange(n), {"config": "track", "gen_seed": seed})
    out.length = np.concatenate([np.full(n_seg, seg_len), np.zeros(n_casc)]).astype(np.float32)
    return out


def _power_law(rng, gamma, e0, e1, size=None):
    a = 1.0 - gamma
    u = rng.uniform(size=size)
    return (e0 ** a + u * (e1 ** a - e0 ** a)) ** (1.0 / a)


def _perp_basis(d):
    h = np.array([1.0, 0.0, 0.0]) if abs(d[0]) < 0.9 else np.array([0.0, 1.0, 0.0])
    e1 = _unit(np.cross(d, h))
    e2 = np.cross(d, e1)
    return e1, e2


def _bundle(rng, event_id, n_muons, light_fraction_gev, first_source_id=0):
    """One muon bundle: parallel muons within a 20 m disc through a point uniform in a
    cylinder r=600 m, h=1100 m; 50-500 cascades per muon; cascade energies log-uniform over
    four decades, rescaled so that they sum to ``light_fraction_gev`` (None: not rescaled)."""
    cos_z = rng.uniform(0.0, 1.0)
    az = 2.0 * math.pi * rng.uniform()
    d = travel_direction(math.acos(cos_z), az)
    r = 600.0 * math.sqrt(rng.uniform())
    a = 2.0 * math.pi * rng.uniform()
    point = np.array([r * math.cos(a), r * math.sin(a), rng.uniform(-550.0, 550.0)])
    e1, e2 = _perp_basis(d)
    pos_l, t_l, e_l = [], [], []
    for _ in range(n_muons):
        rr = 20.0 * math.sqrt(rng.uniform())
        aa = 2.0 * math.pi * rng.uniform()
        p0 = point + rr * (math.cos(aa) * e1 + math.sin(aa) * e2)
        n_casc = int(rng.integers(50, 501))
        pos, t = _track_cascades(rng, p0, d, n_casc)
        pos_l.append(pos)
        t_l.append(t)
        e_l.append(np.exp(rng.uniform(math.log(1.0), math.log(1.0e4), size=n_casc)))
    pos = np.concatenate(pos_l)
    t = np.concatenate(t_l)
    e = np.concatenate(e_l)
    if light_fraction_gev is not None:
        e *= light_fraction_gev / e.sum()
    n = len(e)
    dirs = np.repeat(d[None, :], n, axis=0)
    return pos, dirs, t, e, np.full(n, event_id), first_source_id + np.arange(n)


LIGHT_FRACTION = 0.005  # sum(E_cascade) = 0.005 * E_primary: the one normalisation that makes C4 ~5e9 photons


def sources_c2(seed: int = 2, n_events: int = 1000, literal: bool = False) -> Sources:
    """C2: 1000 muon-bundle events, E_prim ~ E^-2.7 on [1e3, 1e8] GeV, multiplicity
    floor(1 + (E/1e4)^0.8).  With ``literal=False`` (default, reading R-C2) cascade
    energies are rescaled per event to 0.005*E_prim; ``literal=True`` keeps the raw
    log-uniform [1, 1e4] GeV energies (~3e12 photons: throughput only)."""
    rng = np.random.default_rng(seed)
    parts = []
    e_prim = _power_law(rng, 2.7, 1.0e3, 1.0e8, size=n_events)
    for ev in range(n_events):
        mult = int(math.floor(1.0 + (e_prim[ev] / 1.0e4) ** 0.8))
        parts.append(_bundle(rng, ev, mult, None if literal else LIGHT_FRACTION * e_prim[ev]))
    pos, dirs, t, e, evid, sid = (np.concatenate([p[i] for p in parts]) for i in range(6))
    return _pack(pos, dirs, t, e, evid, sid, {"config": "C2", "gen_seed": seed, "e_prim": e_prim, "literal": literal})


def sources_c3(n_photons: float, seed: int = 3) -> Sources:
    """C3: cascades uniform in the instrumented volume (cylinder r=575 m, z in [-503, 500]),
    isotropic axes, E log-uniform on [1, 100] TeV; the list is cut where the expected photon
    total (E * 1e4/GeV) reaches ``n_photons`` by reducing the last cascade's energy."""
    rng = np.random.default_rng(seed)
    pos_l, dir_l, e_l = [], [], []
    total = 0.0
    while total < n_photons:
        r = 575.0 * math.sqrt(rng.uniform())
        a = 2.0 * math.pi * rng.uniform()
        z = rng.uniform(-503.0, 500.0)
        cos_t = 2.0 * rng.uniform() - 1.0
        phi = 2.0 * math.pi * rng.uniform()
        sin_t = math.sqrt(1.0 - cos_t * cos_t)
        e = math.exp(rng.uniform(math.log(1.0e3), math.log(1.0e5)))
        if total + e * PHOTONS_PER_GEV > n_photons:
            e = (n_photons - total) / PHOTONS_PER_GEV
        total += e * PHOTONS_PER_GEV
        pos_l.append([r * math.cos(a), r * math.sin(a), z])
        dir_l.append([sin_t * math.cos(phi), sin_t * math.sin(phi), cos_t])
        e_l.append(e)
    n = len(e_l)
    return _pack(pos_l, dir_l, np.zeros(n), e_l, np.arange(n), np.zeros(n),
                 {"config": "C3", "gen_seed": seed, "target_photons": n_photons})


def sources_c4(seed: int = 4, n_muons: int = 500, n_photons: float = 5.0e9) -> Sources:
    """C4: one 1e8 GeV bundle of 500 parallel muons, normalised to ~5e9 photons."""
    rng = np.random.default_rng(seed)
    pos, dirs, t, e, evid, sid = _bundle(rng, 0, n_muons, n_photons / PHOTONS_PER_GEV)
    return _pack(pos, dirs, t, e, evid, sid, {"config": "C4", "gen_seed": seed})


def pencil_beam(origin, direction, n_photons: float, t0: float = 0.0, event_id: int = 0) -> Sources:
    """A single source used by the closed-form tests (with ``cos_cherenkov = 1`` it is a
    pencil beam along ``direction``)."""
    d = _unit(np.asarray(direction, dtype=np.float64))
    return _pack([origin], [d], [t0], [n_photons / PHOTONS_PER_GEV], [event_id], [0], {"config": "pencil"})
