"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes front end of the CPU oracle (oracle.hpp / oracle_capi.cpp): a plain fp64 restatement of
the photon-propagation path of arXiv:2405.05700 that shares no code with the
CUDA library.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.

Build: ``python -m oracle.oracle`` (or :func:`build`) compiles ``liboracle.so`` with g++ -O2,
no fast-math, no FMA contraction.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import sys
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboracle.so")
_SRCS = [os.path.join(_HERE, "oracle_capi.cpp")]
_DEPS = _SRCS + [os.path.join(_HERE, "oracle.hpp")]


def build(force: bool = False) -> str:
    """Compile liboracle.so if it is missing or older than its sources."""
    if not force and os.path.exists(_LIB_PATH):
        if all(os.path.getmtime(_LIB_PATH) >= os.path.getmtime(s) for s in _DEPS):
            return _LIB_PATH
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-ffp-contract=off", "-fno-fast-math",
           "-Wall", "-o", _LIB_PATH] + _SRCS
    subprocess.check_call(cmd)
    return _LIB_PATH


class _Ice(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("z_top", C.c_double), ("dz", C.c_double),
                ("abs_len", C.POINTER(C.c_float)), ("scat_len", C.POINTER(C.c_float)),
                ("g", C.c_double), ("n_group", C.c_double), ("cos_cherenkov", C.c_double),
                ("photons_per_gev", C.c_double), ("effective_scattering", C.c_int32), ("pad", C.c_int32)]


class _Geo(C.Structure):
    _fields_ = [("n_dom", C.c_int32), ("xyz", C.POINTER(C.c_float)), ("radius", C.c_double)]


HIT_DTYPE = np.dtype([("event_id", "<u4"), ("source_id", "<u4"), ("photon_idx", "<u4"), ("dom_id", "<u4"),
                      ("time_ns", "<f8"), ("weight", "<f8")])
FATE_DTYPE = np.dtype([("fate", "<i4"), ("dom", "<i4"), ("n_flights", "<u4"), ("pad", "<u4"),
                       ("x", "<f8"), ("y", "<f8"), ("z", "<f8"), ("time_ns", "<f8"), ("path_m", "<f8"),
                       ("dx", "<f8"), ("dy", "<f8"), ("dz", "<f8")])
FATE_ABSORBED, FATE_HIT, FATE_ABORTED, FATE_REJECTED = 0, 1, 2, 3


class _Stats(C.Structure):
    _fields_ = [("photons", C.c_uint64), ("absorbed", C.c_uint64), ("hit", C.c_uint64), ("aborted", C.c_uint64),
                ("flights", C.c_uint64), ("rejected", C.c_uint64)]


class _Job(C.Structure):
    _fields_ = [("geo", _Geo), ("ice", _Ice), ("seed", C.c_uint64), ("n_sources", C.c_uint64),
                ("src", C.POINTER(C.c_float)), ("event_id", C.POINTER(C.c_uint32)),
                ("source_id", C.POINTER(C.c_uint32)), ("first", C.POINTER(C.c_uint64)),
                ("count", C.POINTER(C.c_uint64)), ("stride", C.c_uint64), ("offset", C.c_uint64),
                ("brute_force", C.c_int32), ("real_type", C.c_int32), ("n_threads", C.c_int32), ("pad", C.c_int32),
                ("hits", C.c_void_p), ("hit_cap", C.c_uint64), ("fates", C.c_void_p), ("fate_cap", C.c_uint64),
                ("acc_mode", C.c_int32), ("acc_n_coef", C.c_int32), ("acc_coef", C.c_double * 8),
                ("length", C.POINTER(C.c_float)), ("spec_n", C.c_int32), ("pad2", C.c_int32),
                ("spec_cdf", C.POINTER(C.c_float)), ("spec_abs_scale", C.POINTER(C.c_float)),
                ("spec_scat_scale", C.POINTER(C.c_float)), ("spec_n_group", C.POINTER(C.c_float)),
                ("spec_acc_scale", C.POINTER(C.c_float)), ("g_axis", C.c_double),
                ("prof_n", C.c_int32), ("pad3", C.c_int32), ("prof_f", C.POINTER(C.c_float))]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB_PATH)
        L.orc_uniform.restype = C.c_double
        L.orc_uniform.argtypes = [C.c_uint32]
        L.orc_photon_count.restype = C.c_uint64
        L.orc_photon_count.argtypes = [C.c_float, C.c_float]
        L.orc_hg_cos.restype = C.c_double
        L.orc_hg_cos.argtypes = [C.c_double, C.c_double]
        L.orc_segment_fraction.restype = C.c_double
        L.orc_segment_fraction.argtypes = [C.POINTER(C.c_float), C.c_int32, C.c_double]
        L.orc_spectrum_word.restype = C.c_uint32
        L.orc_spectrum_word.argtypes = [C.POINTER(C.c_uint32)]
        L.orc_acceptance.restype = C.c_double
        L.orc_acceptance.argtypes = [C.POINTER(C.c_double), C.c_int32, C.c_double]
        L.orc_rotate.restype = None
        L.orc_rotate.argtypes = [C.POINTER(C.c_double), C.c_double, C.c_double, C.POINTER(C.c_double)]
        L.orc_philox4x32_10.restype = None
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.orc_layer_of.restype = C.c_int32
        L.orc_layer_of.argtypes = [C.POINTER(_Ice), C.c_double]
        L.orc_walk.restype = C.c_double
        L.orc_walk.argtypes = [C.POINTER(_Ice), C.c_int32, C.c_double, C.c_double, C.c_double]
        L.orc_depth.restype = C.c_double
        L.orc_depth.argtypes = [C.POINTER(_Ice), C.c_int32, C.c_double, C.c_double, C.c_double]
        L.orc_intersect.restype = C.c_int32
        L.orc_intersect.argtypes = [C.POINTER(_Geo), C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double),
                                    C.c_double, C.POINTER(C.c_double)]
        L.orc_propagate.restype = C.c_int64
        L.orc_propagate.argtypes = [C.POINTER(_Job), C.POINTER(_Stats)]
        _lib = L
    return _lib


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _mk_ice(ice):
    a = np.ascontiguousarray(ice.abs_len, dtype=np.float32)
    s = np.ascontiguousarray(ice.scat_len, dtype=np.float32)
    st = _Ice(int(a.shape[0]), float(ice.z_top), float(ice.dz), _fp(a), _fp(s), float(np.float32(ice.g)),
              float(np.float32(ice.n_group)), float(np.float32(ice.cos_cherenkov)),
              float(np.float32(ice.photons_per_GeV)), 1 if getattr(ice, "effective_scattering", False) else 0, 0)
    return st, (a, s)


def _mk_geo(geo):
    x = np.ascontiguousarray(geo.xyz, dtype=np.float32)
    return _Geo(int(x.shape[0]), _fp(x), float(np.float32(geo.radius))), (x,)


# ---- component functions (each pinned in tests/test_oracle_*.py) ---------------------------
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def uniform(word: int) -> float:
    return lib().orc_uniform(int(word) & 0xFFFFFFFF)


def photon_count(energy_gev, photons_per_gev=1.0e4) -> int:
    return int(lib().orc_photon_count(float(np.float32(energy_gev)), float(np.float32(photons_per_gev))))


def hg_cos(g: float, u: float) -> float:
    return lib().orc_hg_cos(float(g), float(u))


def segment_fraction(table, u: float) -> float:
    """F(u) of DESIGN.md R-23: the piecewise-linear inverse cumulative distribution of the emission offset."""
    t = np.ascontiguousarray(table, dtype=np.float32)
    return lib().orc_segment_fraction(_fp(t), int(t.shape[0]), float(u))


def spectrum_word(words) -> int:
    """The word of the wavelength uniform, from the four words of a photon's Philox block 0 (R-21)."""
    w = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in words])
    return int(lib().orc_spectrum_word(w))


def acceptance(coef, eta: float) -> float:
    """p(eta) of DESIGN.md R-17: the clamped polynomial in the arrival direction cosine."""
    c = (C.c_double * len(coef))(*[float(np.float32(x)) for x in coef])
    return lib().orc_acceptance(c, len(coef), float(eta))


ACCEPTANCE_MODES = {"off": 0, "probabilistic": 1, "weighted": 2}


def rotate(d, cos_t: float, phi: float) -> np.ndarray:
    a = (C.c_double * 3)(*[float(x) for x in d])
    o = (C.c_double * 3)()
    lib().orc_rotate(a, float(cos_t), float(phi), o)
    return np.array(list(o))


def layer_of(ice, z: float) -> int:
    st, keep = _mk_ice(ice)
    return int(lib().orc_layer_of(C.byref(st), float(z)))


def walk(ice, which: str, z: float, dir_z: float, tau: float) -> float:
    st, keep = _mk_ice(ice)
    return lib().orc_walk(C.byref(st), 1 if which == "abs" else 0, float(z), float(dir_z), float(tau))


def depth(ice, which: str, z: float, dir_z: float, s: float) -> float:
    st, keep = _mk_ice(ice)
    return lib().orc_depth(C.byref(st), 1 if which == "abs" else 0, float(z), float(dir_z), float(s))


def intersect(geo, p, d, s: float, brute: bool = True):
    st, keep = _mk_geo(geo)
    pp = (C.c_double * 3)(*[float(x) for x in p])
    dd = (C.c_double * 3)(*[float(x) for x in d])
    t = C.c_double(0.0)
    j = lib().orc_intersect(C.byref(st), 1 if brute else 0, pp, dd, float(s), C.byref(t))
    return int(j), (t.value if j >= 0 else float("inf"))


@dataclass
class Result:
    hits: np.ndarray  # HIT_DTYPE, sorted by (event_id, source_id, photon_idx)
    fates: np.ndarray | None  # FATE_DTYPE in (source order, photon_idx) order, if requested
    photons: int
    absorbed: int
    hit: int
    aborted: int
    flights: int
    rejected: int = 0


def propagate(geo, ice, sources, seed: int = 0, *, stride: int = 1, offset: int = 0, first=None, count=None,
              brute_force: bool = False, real_type: str = "f64", n_threads: int = 0, want_fates: bool = False,
              hit_cap: int | None = None, acceptance_mode: str = "off", acceptance_coef=(), lengths=None, spectrum=None, g_axis: float = 1.0, segment_profile=None) -> Result:
    """Run the selected photons (``first <= i < first+count`` and ``i % stride == offset``) of
    every source through the oracle.  Hits come back sorted by (event, source, photon)."""
    L = lib()
    g_st, g_keep = _mk_geo(geo)
    i_st, i_keep = _mk_ice(ice)
    src = np.ascontiguousarray(sources.src, dtype=np.float32)
    ev = np.ascontiguousarray(sources.event_id, dtype=np.uint32)
    sid = np.ascontiguousarray(sources.source_id, dtype=np.uint32)
    n = src.shape[0]
    counts = np.array([photon_count(e, ice.photons_per_GeV) for e in src[:, 7]], dtype=np.uint64) if n else \
        np.zeros(0, np.uint64)
    f_arr = None if first is None else np.ascontiguousarray(first, dtype=np.uint64)
    c_arr = None if count is None else np.ascontiguousarray(count, dtype=np.uint64)
    lo = np.zeros(n, np.uint64) if f_arr is None else f_arr
    hi = counts if c_arr is None else np.minimum(counts, lo + c_arr)
    n_sel = int(sum(len(range(int(a) + ((offset - int(a)) % stride), int(b), stride)) for a, b in zip(lo, hi) if b > a))
    if hit_cap is None:
        hit_cap = max(n_sel, 1)
    hits = np.zeros(hit_cap, dtype=HIT_DTYPE)
    fates = np.zeros(n_sel if want_fates else 0, dtype=FATE_DTYPE)
    job = _Job()
    job.geo, job.ice = g_st, i_st
    job.seed = int(seed)
    job.n_sources = n
    job.src = _fp(src)
    job.event_id = ev.ctypes.data_as(C.POINTER(C.c_uint32))
    job.source_id = sid.ctypes.data_as(C.POINTER(C.c_uint32))
    job.first = None if f_arr is None else f_arr.ctypes.data_as(C.POINTER(C.c_uint64))
    job.count = None if c_arr is None else c_arr.ctypes.data_as(C.POINTER(C.c_uint64))
    job.stride, job.offset = int(stride), int(offset)
    job.brute_force = 1 if brute_force else 0
    job.real_type = {"f64": 0, "f32": 1}[real_type]
    job.n_threads = int(n_threads)
    job.hits = hits.ctypes.data
    job.hit_cap = hit_cap
    job.fates = fates.ctypes.data if want_fates and n_sel else None
    job.fate_cap = n_sel if want_fates else 0
    if lengths is None:
        lengths = getattr(sources, "length", None)
    len_arr = None if lengths is None else np.ascontiguousarray(lengths, dtype=np.float32)
    assert len_arr is None or len_arr.shape[0] == n
    job.length = None if len_arr is None else _fp(len_arr)
    job.g_axis = float(np.float32(g_axis))
    prof_arr = None if segment_profile is None else np.ascontiguousarray(segment_profile, dtype=np.float32)
    job.prof_n = 0 if prof_arr is None else int(prof_arr.shape[0])
    job.prof_f = None if prof_arr is None else _fp(prof_arr)
    spec_keep = []
    job.spec_n = 0
    if spectrum is not None:  # anything with cdf, abs_scale, scat_scale, n_group, acc_scale (workloads.Spectrum)
        for name in ("cdf", "abs_scale", "scat_scale", "n_group", "acc_scale"):
            a = np.ascontiguousarray(getattr(spectrum, name), dtype=np.float32)
            spec_keep.append(a)
            setattr(job, "spec_" + name, _fp(a))
        job.spec_n = int(spec_keep[0].shape[0])
        assert all(a.shape[0] == job.spec_n for a in spec_keep)
    job.acc_mode = ACCEPTANCE_MODES[acceptance_mode]
    job.acc_n_coef = len(acceptance_coef)
    for k, c in enumerate(acceptance_coef):
        job.acc_coef[k] = float(np.float32(c))  # the same fp32 coefficients the CUDA library receives
    st = _Stats()
    nh = L.orc_propagate(C.byref(job), C.byref(st))
    if nh < 0:
        raise ValueError("oracle: bad job")
    if nh > hit_cap:
        raise RuntimeError(f"oracle: {nh} hits exceed hit_cap {hit_cap}")
    return Result(hits[:nh].copy(), fates if want_fates else None, int(st.photons), int(st.absorbed), int(st.hit),
                  int(st.aborted), int(st.flights), int(st.rejected))


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
