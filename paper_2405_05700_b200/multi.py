"""Thin ctypes binding of ``include/pp_multi.h``: several devices behind one photon server (
PAPER.md:33 "embarrassingly parallel").  Argument marshalling only.
"""
from __future__ import annotations

import ctypes as C
import threading

import numpy as np

from .binding import HIT_DTYPE, PP_OK, PPError, Propagator, load_library, pack_sources, SOURCE_DTYPE

EXPORTS = ["pp_multi_create", "pp_multi_create_backends", "pp_multi_destroy", "pp_multi_submit", "pp_multi_flush",
           "pp_multi_collect", "pp_multi_get_stats", "pp_multi_backend"]


class _MultiConfig(C.Structure):
    _fields_ = [("deal_photons", C.c_uint64), ("photons_per_GeV", C.c_float), ("reserved", C.c_uint32)]


class _MultiStats(C.Structure):
    _fields_ = [("n_devices", C.c_uint32), ("reserved", C.c_uint32), ("sources_submitted", C.c_uint64),
                ("photons_submitted", C.c_uint64), ("sources_staged", C.c_uint64), ("sources_completed", C.c_uint64),
                ("batches", C.c_uint64 * 64), ("photons", C.c_uint64 * 64), ("photons_outstanding", C.c_uint64 * 64)]


class Backend(C.Structure):
    """pp_ipc_backend (include/pp_ipc.h)."""
    _fields_ = [("ctx", C.c_void_p), ("submit", C.c_void_p), ("flush", C.c_void_p), ("collect", C.c_void_p),
                ("completed", C.c_void_p), ("submit_packed", C.c_void_p)]


_declared = False


def _lib():
    global _declared
    L = load_library()
    if not _declared:
        vp = C.c_void_p
        L.pp_multi_create.restype = C.c_int
        L.pp_multi_create.argtypes = [C.POINTER(vp), C.c_uint32, C.POINTER(_MultiConfig), C.POINTER(vp)]
        L.pp_multi_create_backends.restype = C.c_int
        L.pp_multi_create_backends.argtypes = [C.POINTER(Backend), C.c_uint32, C.POINTER(_MultiConfig), C.POINTER(vp)]
        L.pp_multi_destroy.restype = None
        L.pp_multi_destroy.argtypes = [vp]
        L.pp_multi_submit.restype = C.c_int
        L.pp_multi_submit.argtypes = [vp, vp, vp, vp, vp, C.c_size_t]
        L.pp_multi_flush.restype = C.c_int
        L.pp_multi_flush.argtypes = [vp]
        L.pp_multi_collect.restype = C.c_int
        L.pp_multi_collect.argtypes = [vp, vp, C.c_size_t, C.POINTER(C.c_size_t), C.c_int]
        L.pp_multi_get_stats.restype = C.c_int
        L.pp_multi_get_stats.argtypes = [vp, C.POINTER(_MultiStats)]
        L.pp_multi_backend.restype = C.c_int
        L.pp_multi_backend.argtypes = [vp, C.POINTER(Backend)]
        _declared = True
    return L


class MultiFront:
    """pp_multi_create over Propagators (one per device), or pp_multi_create_backends over ``backends`` (addresses of
    ``pp_ipc_backend`` structs; the CPU tests pass host-only ones)."""

    def __init__(self, propagators=None, *, photons_per_GeV: float, deal_photons: int = 0, backends=None):
        self._L = _lib()
        cfg = _MultiConfig(int(deal_photons), float(photons_per_GeV), 0)
        m = C.c_void_p()
        if backends is not None:
            arr = (Backend * len(backends))()
            for i, b in enumerate(backends):
                C.memmove(C.byref(arr[i]), C.c_void_p(b), C.sizeof(Backend))
            rc = self._L.pp_multi_create_backends(arr, len(backends), C.byref(cfg), C.byref(m))
        else:
            self._props = list(propagators)  # keep the handles alive
            arr = (C.c_void_p * len(self._props))(*[p._h for p in self._props])
            rc = self._L.pp_multi_create(arr, len(self._props), C.byref(cfg), C.byref(m))
        if rc != PP_OK:
            raise PPError(rc, "pp_multi_create")
        self._m = m
        self._be = None

    @classmethod
    def over_devices(cls, geometry, ice, devices, *, deal_photons: int = 0, **kw):
        """One Propagator per CUDA device ordinal in ``devices`` (same geometry, ice, seed, options), one front."""
        props = [Propagator(geometry, ice, device=int(d), **kw) for d in devices]
        return cls(props, photons_per_GeV=float(ice.photons_per_GeV), deal_photons=deal_photons)

    def _check(self, rc, what):
        if rc != PP_OK:
            raise PPError(rc, what)

    def submit(self, sources, event_ids, source_ids=None, lengths=None):
        rec = pack_sources(sources) if sources.dtype != SOURCE_DTYPE else np.ascontiguousarray(sources)
        ev = np.ascontiguousarray(event_ids, dtype=np.uint32)
        sid = None if source_ids is None else np.ascontiguousarray(source_ids, dtype=np.uint32)
        ln = None if lengths is None else np.ascontiguousarray(lengths, dtype=np.float32)
        assert ev.shape[0] == rec.shape[0]
        self._check(self._L.pp_multi_submit(self._m, rec.ctypes.data, None if ln is None else ln.ctypes.data,
                                            ev.ctypes.data, None if sid is None else sid.ctypes.data, rec.shape[0]),
                    "pp_multi_submit")

    def flush(self):
        self._check(self._L.pp_multi_flush(self._m), "pp_multi_flush")

    def collect(self, cap: int = 1 << 20, block: bool = True) -> np.ndarray:
        tls = self.__dict__.setdefault("_collect_tls", threading.local())  # one landing buffer per calling thread
        out = getattr(tls, "buf", None)
        if out is None or out.shape[0] < cap:
            out = tls.buf = np.empty(cap, dtype=HIT_DTYPE)
        n = C.c_size_t(0)
        self._check(self._L.pp_multi_collect(self._m, out.ctypes.data, cap, C.byref(n), 1 if block else 0),
                    "pp_multi_collect")
        return out[: n.value].copy()

    def collect_all(self) -> np.ndarray:
        self.flush()
        parts = []
        while True:
            h = self.collect(block=True)
            if len(h) == 0:
                break
            parts.append(h)
        return np.concatenate(parts) if parts else np.empty(0, dtype=HIT_DTYPE)

    def run(self, sources, event_ids, source_ids=None, lengths=None) -> np.ndarray:
        self.submit(sources, event_ids, source_ids, lengths)
        return self.collect_all()

    def stats(self) -> dict:
        st = _MultiStats()
        self._check(self._L.pp_multi_get_stats(self._m, C.byref(st)), "pp_multi_get_stats")
        n = int(st.n_devices)
        return {"n_devices": n, "sources_submitted": int(st.sources_submitted),
                "photons_submitted": int(st.photons_submitted), "sources_staged": int(st.sources_staged),
                "sources_completed": int(st.sources_completed), "batches": [int(x) for x in st.batches[:n]],
                "photons": [int(x) for x in st.photons[:n]],
                "photons_outstanding": [int(x) for x in st.photons_outstanding[:n]]}

    def backend_address(self) -> int:
        """Address of a pp_ipc_backend that drives this front (for ipc.IpcServer(..., backend=...))."""
        if self._be is None:
            self._be = Backend()
            self._check(self._L.pp_multi_backend(self._m, C.byref(self._be)), "pp_multi_backend")
        return C.addressof(self._be)

    def close(self, close_propagators: bool = True):
        if getattr(self, "_m", None):
            self._L.pp_multi_destroy(self._m)
            self._m = None
        if close_propagators:
            for p in getattr(self, "_props", []):
                p.close()
            self._props = []

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()
