"""Thin ctypes binding of the C ABI in ``include/pp.h`` (argument marshalling only).

PyTorch is used for exactly three things here: device memory (the workspace and the resident
input arrays), pinned host memory, and the two CUDA streams.  Every step of the hot path runs in
the library's own kernels; there is no CPU or PyTorch fallback: if ``libpp.so`` is missing or
no CUDA device is present, construction fails loudly.
"""
from __future__ import annotations

import ctypes as C
import os
import threading
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# (developer knob: PP_LIB names another build of the library, e.g. the tests' guard build -- never a fallback)
LIB_PATH = os.environ.get("PP_LIB") or os.path.join(_HERE, "libpp.so")

PP_OK = 0
ERRORS = {-1: "PP_E_INVAL", -2: "PP_E_NOMEM", -3: "PP_E_CUDA", -4: "PP_E_OVERFLOW", -5: "PP_E_WOULDBLOCK",
          -6: "PP_E_UNSUPPORTED", -7: "PP_E_STATE"}
FLAG_BRUTE_FORCE_DOMS = 1
FLAG_NONBLOCKING_SUBMIT = 2
FLAG_EFFECTIVE_SCATTERING = 4
FLAG_DEVICE_ORDINAL = 8
ACCEPTANCE_MODES = {"off": 0, "probabilistic": 1, "weighted": 2}

SOURCE_DTYPE = np.dtype([("x", "<f4"), ("y", "<f4"), ("z", "<f4"), ("dx", "<f4"), ("dy", "<f4"), ("dz", "<f4"),
                         ("t_ns", "<f4"), ("energy_GeV", "<f4")])
HIT_DTYPE = np.dtype([("event_id", "<u4"), ("source_id", "<u4"), ("photon_idx", "<u4"), ("dom_id", "<u4"),
                      ("time_ns", "<f8"), ("weight", "<f4"), ("n_scatter", "<u4")])
FATE_DTYPE = np.dtype([("x", "<f4"), ("y", "<f4"), ("z", "<f4"), ("path_m", "<f4"), ("time_ns", "<f8"),
                       ("n_flights", "<u4"), ("dom", "<i4"), ("fate", "<u4"), ("photon_idx", "<u4")])
assert SOURCE_DTYPE.itemsize == 32 and HIT_DTYPE.itemsize == 32 and FATE_DTYPE.itemsize == 40


class PPError(RuntimeError):
    def __init__(self, code: int, msg: str = ""):
        self.code = code
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")


class _Geometry(C.Structure):
    _fields_ = [("n_dom", C.c_uint32), ("xyz", C.POINTER(C.c_float)), ("radius", C.c_float)]


class _Ice(C.Structure):
    _fields_ = [("n_layers", C.c_uint32), ("z_top", C.c_float), ("dz", C.c_float),
                ("abs_len", C.POINTER(C.c_float)), ("scat_len", C.POINTER(C.c_float)), ("g", C.c_float),
                ("n_group", C.c_float), ("cos_cherenkov", C.c_float), ("photons_per_GeV", C.c_float)]


class _Config(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("launch_photons_target", C.c_uint64), ("hit_ring_bytes", C.c_uint64),
                ("source_ring_bytes", C.c_uint64), ("device_workspace", C.c_void_p),
                ("device_workspace_bytes", C.c_uint64), ("pinned_workspace", C.c_void_p),
                ("pinned_workspace_bytes", C.c_uint64), ("stream0", C.c_void_p), ("stream1", C.c_void_p),
                ("flags", C.c_uint32), ("max_flights", C.c_uint32), ("device", C.c_int32), ("reserved", C.c_uint32)]


class _Stats(C.Structure):
    _fields_ = [("sources_submitted", C.c_uint64), ("photons_submitted", C.c_uint64), ("photons_done", C.c_uint64),
                ("photons_absorbed", C.c_uint64), ("photons_hit", C.c_uint64), ("photons_aborted", C.c_uint64),
                ("flights", C.c_uint64), ("launches", C.c_uint64), ("relaunches", C.c_uint64),
                ("hits_collected", C.c_uint64), ("kernel_busy_ms", C.c_double), ("wall_ms", C.c_double),
                ("source_ring_high_water", C.c_uint64), ("hit_ring_high_water", C.c_uint64),
                ("photons_rejected", C.c_uint64), ("sources_completed", C.c_uint64)]


EXPORTS = ["pp_workspace_size", "pp_create", "pp_submit", "pp_flush", "pp_collect", "pp_stats", "pp_last_error",
           "pp_destroy", "pp_run_resident", "pp_version", "pp_kernel_launch_count", "pp_check_inputs",
           "pp_photon_count", "pp_debug_plan_launches", "pp_set_acceptance", "pp_submit_segments", "pp_set_spectrum",
           "pp_set_emission_smearing", "pp_set_segment_profile", "pp_submit_packed", "pp_run_resident_noalloc"]
NOALLOC_MAX_SOURCES = 4096        # PP_NOALLOC_MAX_SOURCES
NOALLOC_MAX_PHOTONS = 1 << 22     # PP_NOALLOC_MAX_PHOTONS


class _LaunchPlan(C.Structure):
    _fields_ = [("first_source", C.c_uint64), ("n_sources", C.c_uint64), ("g_begin", C.c_uint64),
                ("g_end", C.c_uint64)]

_lib = None


def load_library(path: str = LIB_PATH):
    """Loads libpp.so and declares the prototypes of every symbol include/pp.h declares."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} is missing: build it with `python -m paper_2405_05700_b200.build` "
                                "(there is no CPU fallback)")
    L = C.CDLL(path)
    vp, u32p = C.c_void_p, C.POINTER(C.c_uint32)
    L.pp_workspace_size.restype = C.c_int
    L.pp_workspace_size.argtypes = [C.POINTER(_Geometry), C.POINTER(_Ice), C.POINTER(_Config),
                                    C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.pp_create.restype = C.c_int
    L.pp_create.argtypes = [C.POINTER(_Geometry), C.POINTER(_Ice), C.POINTER(_Config), C.POINTER(vp)]
    L.pp_submit.restype = C.c_int
    L.pp_submit.argtypes = [vp, vp, vp, vp, C.c_size_t]
    L.pp_submit_segments.restype = C.c_int
    L.pp_submit_segments.argtypes = [vp, vp, vp, vp, vp, C.c_size_t]
    L.pp_submit_packed.restype = C.c_int
    L.pp_submit_packed.argtypes = [vp, vp, C.c_size_t, C.POINTER(C.c_uint64)]
    L.pp_flush.restype = C.c_int
    L.pp_flush.argtypes = [vp]
    L.pp_collect.restype = C.c_int
    L.pp_collect.argtypes = [vp, vp, C.c_size_t, C.POINTER(C.c_size_t), C.c_int]
    L.pp_set_acceptance.restype = C.c_int
    L.pp_set_acceptance.argtypes = [vp, C.c_uint32, C.POINTER(C.c_float), C.c_uint32]
    L.pp_set_emission_smearing.restype = C.c_int
    L.pp_set_emission_smearing.argtypes = [vp, C.c_float]
    L.pp_set_segment_profile.restype = C.c_int
    L.pp_set_segment_profile.argtypes = [vp, C.c_uint32, C.POINTER(C.c_float)]
    L.pp_set_spectrum.restype = C.c_int
    L.pp_set_spectrum.argtypes = [vp, C.c_uint32] + [C.POINTER(C.c_float)] * 5
    L.pp_stats.restype = C.c_int
    L.pp_stats.argtypes = [vp, C.POINTER(_Stats)]
    L.pp_last_error.restype = C.c_char_p
    L.pp_last_error.argtypes = [vp]
    L.pp_destroy.restype = None
    L.pp_destroy.argtypes = [vp]
    L.pp_run_resident.restype = C.c_int
    L.pp_run_resident.argtypes = [vp, vp, vp, vp, C.c_size_t, vp, C.POINTER(C.c_uint64), C.POINTER(C.c_double)]
    L.pp_run_resident_noalloc.restype = C.c_int
    L.pp_run_resident_noalloc.argtypes = [vp, vp, vp, vp, C.c_size_t, vp, C.c_size_t, C.POINTER(C.c_size_t),
                                          C.POINTER(C.c_uint64), vp]
    L.pp_version.restype = C.c_char_p
    L.pp_kernel_launch_count.restype = C.c_uint64
    L.pp_check_inputs.restype = C.c_int
    L.pp_check_inputs.argtypes = [C.POINTER(_Geometry), C.POINTER(_Ice), C.c_uint32]
    L.pp_photon_count.restype = C.c_int
    L.pp_photon_count.argtypes = [C.c_float, C.c_float, C.POINTER(C.c_uint64)]
    L.pp_debug_plan_launches.restype = C.c_int
    L.pp_debug_plan_launches.argtypes = [u32p, C.c_size_t, C.c_uint64, C.POINTER(_LaunchPlan), C.c_size_t,
                                         C.POINTER(C.c_size_t)]
    _lib = L
    return L


def kernel_launch_count() -> int:
    return int(load_library().pp_kernel_launch_count())


def version() -> str:
    return load_library().pp_version().decode()


def _marshal_inputs(geometry, ice):
    fp = C.POINTER(C.c_float)
    xyz = np.ascontiguousarray(geometry.xyz, dtype=np.float32).reshape(-1, 3)
    a = np.ascontiguousarray(ice.abs_len, dtype=np.float32)
    s = np.ascontiguousarray(ice.scat_len, dtype=np.float32)
    geo = _Geometry(xyz.shape[0], xyz.ctypes.data_as(fp), float(geometry.radius))
    ic = _Ice(a.shape[0], float(ice.z_top), float(ice.dz), a.ctypes.data_as(fp), s.ctypes.data_as(fp), float(ice.g),
              float(ice.n_group), float(ice.cos_cherenkov), float(ice.photons_per_GeV))
    return geo, ic, (xyz, a, s)


def check_inputs(geometry, ice, flags: int = 0) -> int:
    """pp_check_inputs: host-only validation; returns the status code (0 = OK)."""
    geo, ic, keep = _marshal_inputs(geometry, ice)
    return int(load_library().pp_check_inputs(C.byref(geo), C.byref(ic), int(flags)))


def photon_count(energy_gev: float, photons_per_gev: float = 1.0e4) -> int:
    n = C.c_uint64(0)
    rc = load_library().pp_photon_count(float(np.float32(energy_gev)), float(np.float32(photons_per_gev)), C.byref(n))
    if rc != PP_OK:
        raise PPError(rc, "pp_photon_count")
    return int(n.value)


def plan_launches(photon_counts, target: int):
    """pp_debug_plan_launches: list of (first_source, n_sources, g_begin, g_end)."""
    cnt = np.ascontiguousarray(photon_counts, dtype=np.uint32)
    L = load_library()
    n_out = C.c_size_t(0)
    cap = 64
    while True:
        buf = (_LaunchPlan * cap)()
        rc = L.pp_debug_plan_launches(cnt.ctypes.data_as(C.POINTER(C.c_uint32)), cnt.shape[0], int(target), buf, cap,
                                      C.byref(n_out))
        if rc == -2:
            cap = int(n_out.value)
            continue
        if rc != PP_OK:
            raise PPError(rc, "pp_debug_plan_launches")
        return [(int(b.first_source), int(b.n_sources), int(b.g_begin), int(b.g_end)) for b in buf[: n_out.value]]


# pp_packed_source (include/pp.h): a source with its length and ids as one 48-byte record
PACKED_DTYPE = np.dtype([("src", np.float32, (8,)), ("length_m", np.float32), ("event_id", np.uint32),
                         ("source_id", np.uint32), ("reserved", np.uint32)])
assert PACKED_DTYPE.itemsize == 48


def pack_records(sources, event_ids, source_ids, lengths=None) -> np.ndarray:
    """float32 [n, 8] rows + ids (+ lengths) -> pp_packed_source records."""
    a = np.ascontiguousarray(sources, dtype=np.float32).reshape(-1, 8)
    out = np.zeros(a.shape[0], PACKED_DTYPE)
    out["src"] = a
    out["event_id"] = event_ids
    out["source_id"] = source_ids
    if lengths is not None:
        out["length_m"] = lengths
    return out


def pack_sources(src: np.ndarray) -> np.ndarray:
    """float32 [n, 8] rows (x,y,z,dx,dy,dz,t,E) -> pp_source records (a view when possible)."""
    a = np.ascontiguousarray(src, dtype=np.float32).reshape(-1, 8)
    return a.view(SOURCE_DTYPE).reshape(-1)


@dataclass
class Stats:
    sources_submitted: int
    photons_submitted: int
    photons_done: int
    photons_absorbed: int
    photons_hit: int
    photons_aborted: int
    flights: int
    launches: int
    relaunches: int
    hits_collected: int
    kernel_busy_ms: float
    wall_ms: float
    source_ring_high_water: int
    hit_ring_high_water: int
    photons_rejected: int = 0
    sources_completed: int = 0


class Propagator:
    """pp_create / pp_submit / pp_flush / pp_collect / pp_run_resident over one handle.

    ``geometry`` and ``ice`` are the dataclasses of :mod:`.workloads` (or anything with the same
    attributes)."""

    def __init__(self, geometry, ice, *, seed: int = 0, launch_photons_target: int = 0, hit_ring_bytes: int = 0,
                 source_ring_bytes: int = 0, flags: int = 0, max_flights: int = 0, device: int | None = None,
                 use_torch_memory: bool = True):
        """``device``: a CUDA device ordinal (0 is device 0), or None for torch's current device."""
        import torch  # device memory, pinned memory and streams only

        if not torch.cuda.is_available():
            raise PPError(-3, "no CUDA device: the photon propagator has no CPU fallback")
        self._torch = torch
        self._L = load_library()
        self._geo, self._ice, self._inputs_keep = _marshal_inputs(geometry, ice)
        cfg = _Config()
        cfg.seed = int(seed)
        cfg.launch_photons_target = int(launch_photons_target)
        cfg.hit_ring_bytes = int(hit_ring_bytes)
        cfg.source_ring_bytes = int(source_ring_bytes)
        cfg.flags = int(flags) | (FLAG_EFFECTIVE_SCATTERING if getattr(ice, "effective_scattering", False) else 0)
        cfg.max_flights = int(max_flights)
        if device is None:
            device = torch.cuda.current_device()
        cfg.device = int(device)
        cfg.flags |= FLAG_DEVICE_ORDINAL
        self.device = torch.device("cuda", int(device))
        self._keep = []
        if use_torch_memory:
            dev_b, pin_b = C.c_uint64(0), C.c_uint64(0)
            with torch.cuda.device(self.device):
                self._check(self._L.pp_workspace_size(C.byref(self._geo), C.byref(self._ice), C.byref(cfg),
                                                      C.byref(dev_b), C.byref(pin_b)), None)
                ws = torch.empty(int(dev_b.value), dtype=torch.uint8, device=self.device)
                pin = torch.empty(int(pin_b.value), dtype=torch.uint8, pin_memory=True)
                self.streams = (torch.cuda.Stream(device=self.device), torch.cuda.Stream(device=self.device))
            self._keep += [ws, pin]
            cfg.device_workspace, cfg.device_workspace_bytes = ws.data_ptr(), ws.numel()
            cfg.pinned_workspace, cfg.pinned_workspace_bytes = pin.data_ptr(), pin.numel()
            cfg.stream0, cfg.stream1 = self.streams[0].cuda_stream, self.streams[1].cuda_stream
            self.device_workspace_bytes, self.pinned_workspace_bytes = ws.numel(), pin.numel()
        self._cfg = cfg
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            self._check(self._L.pp_create(C.byref(self._geo), C.byref(self._ice), C.byref(cfg), C.byref(h)), None)
        self._h = h

    # ---- plumbing ----
    def _check(self, rc: int, h):
        if rc != PP_OK:
            msg = self._L.pp_last_error(h).decode() if h else ""
            raise PPError(rc, msg)

    def close(self):
        if getattr(self, "_h", None):
            self._L.pp_destroy(self._h)
            self._h = None
            self._keep = []  # give the torch workspace back

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass

    # ---- the paper's calls ----
    def submit(self, sources, event_ids, source_ids=None, lengths=None):
        """pp_submit (pp_submit_segments when ``lengths`` [n] metres is given): ``sources`` float32 [n, 8] (or
        SOURCE_DTYPE [n]); host buffers; thread-safe."""
        rec = pack_sources(sources) if sources.dtype != SOURCE_DTYPE else np.ascontiguousarray(sources)
        ev = np.ascontiguousarray(event_ids, dtype=np.uint32)
        sid = None if source_ids is None else np.ascontiguousarray(source_ids, dtype=np.uint32)
        assert ev.shape[0] == rec.shape[0] and (sid is None or sid.shape[0] == rec.shape[0])
        if lengths is None:
            rc = self._L.pp_submit(self._h, rec.ctypes.data, ev.ctypes.data, None if sid is None else sid.ctypes.data,
                                   rec.shape[0])
        else:
            ln = np.ascontiguousarray(lengths, dtype=np.float32)
            assert ln.shape[0] == rec.shape[0]
            rc = self._L.pp_submit_segments(self._h, rec.ctypes.data, ln.ctypes.data, ev.ctypes.data,
                                            None if sid is None else sid.ctypes.data, rec.shape[0])
        self._check(rc, self._h)

    def submit_packed(self, records):
        """pp_submit_packed: PACKED_DTYPE [n] records (see pack_records); host buffer; thread-safe."""
        rec = np.ascontiguousarray(records, dtype=PACKED_DTYPE)
        end = C.c_uint64(0)
        self._check(self._L.pp_submit_packed(self._h, rec.ctypes.data, rec.shape[0], C.byref(end)), self._h)
        return int(end.value)  # sources submitted to the handle up to and including this call's last one

    def set_acceptance(self, mode: str = "off", coef=()):
        """pp_set_acceptance: ``mode`` in ACCEPTANCE_MODES; ``coef`` = polynomial coefficients in d_z."""
        c = np.ascontiguousarray(coef, dtype=np.float32)
        rc = self._L.pp_set_acceptance(self._h, ACCEPTANCE_MODES[mode], c.ctypes.data_as(C.POINTER(C.c_float)),
                                       c.shape[0])
        self._check(rc, self._h)

    def set_emission_smearing(self, g_axis: float = 1.0):
        """pp_set_emission_smearing: HG parameter of the emission-axis deflection (1 = exact cone)."""
        self._check(self._L.pp_set_emission_smearing(self._h, float(g_axis)), self._h)

    def set_segment_profile(self, cum_fraction=None):
        """pp_set_segment_profile: knots of the inverse CDF of the emission offset (None: uniform)."""
        if cum_fraction is None:
            rc = self._L.pp_set_segment_profile(self._h, 0, None)
        else:
            t = np.ascontiguousarray(cum_fraction, dtype=np.float32)
            rc = self._L.pp_set_segment_profile(self._h, t.shape[0], t.ctypes.data_as(C.POINTER(C.c_float)))
        self._check(rc, self._h)

    def set_spectrum(self, spectrum=None):
        """pp_set_spectrum: ``spectrum`` has cdf, abs_scale, scat_scale, n_group, acc_scale arrays (None: off)."""
        fp = C.POINTER(C.c_float)
        if spectrum is None:
            rc = self._L.pp_set_spectrum(self._h, 0, None, None, None, None, None)
        else:
            arrs = [np.ascontiguousarray(getattr(spectrum, k), dtype=np.float32)
                    for k in ("cdf", "abs_scale", "scat_scale", "n_group", "acc_scale")]
            assert all(a.shape == arrs[0].shape for a in arrs)
            rc = self._L.pp_set_spectrum(self._h, arrs[0].shape[0], *[a.ctypes.data_as(fp) for a in arrs])
        self._check(rc, self._h)

    def flush(self):
        self._check(self._L.pp_flush(self._h), self._h)

    def collect(self, cap: int = 1 << 20, block: bool = True) -> np.ndarray:
        """pp_collect: up to ``cap`` hits; an empty array from a blocking call means drained."""
        # one landing buffer per calling thread, not a fresh 32 MB allocation per call: that alone was a tenth of the
        # wall time of a 1e5-photon launch
        tls = self.__dict__.setdefault("_collect_tls", threading.local())
        buf = getattr(tls, "buf", None)
        if buf is None or buf.shape[0] < cap:
            buf = tls.buf = np.empty(cap, dtype=HIT_DTYPE)
        n = C.c_size_t(0)
        self._check(self._L.pp_collect(self._h, buf.ctypes.data, cap, C.byref(n), 1 if block else 0), self._h)
        return buf[: n.value].copy()

    def collect_all(self, chunk: int = 1 << 20) -> np.ndarray:
        """flush, then collect until drained."""
        self.flush()
        parts = []
        while True:
            h = self.collect(chunk, block=True)
            if len(h) == 0:
                break
            parts.append(h)
        return np.concatenate(parts) if parts else np.empty(0, dtype=HIT_DTYPE)

    def run(self, sources, event_ids, source_ids=None, lengths=None) -> np.ndarray:
        """End-to-end convenience: submit + flush + collect everything (host buffers in and out)."""
        self.submit(sources, event_ids, source_ids, lengths)
        return self.collect_all()

    def stats(self) -> Stats:
        s = _Stats()
        self._check(self._L.pp_stats(self._h, C.byref(s)), self._h)
        return Stats(**{f[0]: getattr(s, f[0]) for f in _Stats._fields_})

    # ---- device-resident path ----
    def upload(self, sources, event_ids, source_ids=None):
        """Copies a source list into HBM (torch tensors) for :meth:`run_resident`."""
        torch = self._torch
        rec = pack_sources(sources) if sources.dtype != SOURCE_DTYPE else np.ascontiguousarray(sources)
        d_src = torch.from_numpy(rec.view(np.float32).reshape(-1, 8).copy()).to(self.device)
        d_ev = torch.from_numpy(np.ascontiguousarray(event_ids, dtype=np.uint32).view(np.int32).copy()).to(self.device)
        d_sid = None if source_ids is None else \
            torch.from_numpy(np.ascontiguousarray(source_ids, dtype=np.uint32).view(np.int32).copy()).to(self.device)
        torch.cuda.synchronize(self.device)
        return d_src, d_ev, d_sid

    def run_resident(self, d_src, d_ev, d_sid=None, want_fates: bool = False, n_photons_hint: int | None = None):
        """pp_run_resident on tensors from :meth:`upload`.  Returns (photons, device_ms, fates|None);
        hits are fetched with :meth:`collect` afterwards."""
        torch = self._torch
        n = int(d_src.shape[0])
        fates_t = None
        if want_fates:
            assert n_photons_hint is not None, "want_fates needs the total photon count"
            fates_t = torch.zeros(int(n_photons_hint) * FATE_DTYPE.itemsize, dtype=torch.uint8, device=self.device)
        ph, ms = C.c_uint64(0), C.c_double(0.0)
        rc = self._L.pp_run_resident(self._h, d_src.data_ptr(), d_ev.data_ptr(), None if d_sid is None else d_sid.data_ptr(),
                                     n, None if fates_t is None else fates_t.data_ptr(), C.byref(ph), C.byref(ms))
        self._check(rc, self._h)
        fates = None
        if want_fates:
            fates = fates_t.cpu().numpy().view(FATE_DTYPE)[: ph.value]
        return int(ph.value), float(ms.value), fates

    def run_resident_noalloc(self, d_src, d_ev, d_sid, d_hits):
        """pp_run_resident_noalloc on tensors from :meth:`upload` (source ids required) and a caller-made uint8 CUDA
        tensor ``d_hits`` of a multiple of 32 bytes that receives the hits.  The library allocates nothing for this
        call: its scratch is a fixed 512 KiB array inside libpp.so, shared by all calls on the device -- at most
        NOALLOC_MAX_SOURCES sources / NOALLOC_MAX_PHOTONS photons per call, and never two calls at once.  Runs on
        torch's current stream and returns after synchronising it: (number of hits now in ``d_hits``, photons)."""
        torch = self._torch
        assert d_sid is not None and d_hits.dtype == torch.uint8 and d_hits.is_cuda and d_hits.is_contiguous()
        n_hits, ph = C.c_size_t(0), C.c_uint64(0)
        rc = self._L.pp_run_resident_noalloc(self._h, d_src.data_ptr(), d_ev.data_ptr(), d_sid.data_ptr(),
                                             int(d_src.shape[0]), d_hits.data_ptr(),
                                             d_hits.numel() // HIT_DTYPE.itemsize, C.byref(n_hits), C.byref(ph),
                                             torch.cuda.current_stream(self.device).cuda_stream)
        self._check(rc, self._h)
        return int(n_hits.value), int(ph.value)

    def drain(self, chunk: int = 1 << 20) -> np.ndarray:
        """Collect whatever is ready without flushing (after run_resident)."""
        parts = []
        while True:
            h = self.collect(chunk, block=False)
            if len(h) == 0:
                break
            parts.append(h)
        return np.concatenate(parts) if parts else np.empty(0, dtype=HIT_DTYPE)
