"""Thin ctypes binding of ``include/pp_ipc.h``: the multi-process front end.

``IpcServer`` runs in the process that owns the :class:`~.binding.Propagator` (and the GPU); ``IpcClient`` runs in
any other process and needs neither CUDA nor torch.  Argument marshalling only.
"""
from __future__ import annotations

import ctypes as C
import threading

import numpy as np

from .binding import HIT_DTYPE, PP_OK, PPError, load_library, pack_sources, SOURCE_DTYPE

EXPORTS = ["pp_ipc_server_create", "pp_ipc_server_create_backend", "pp_ipc_server_destroy", "pp_ipc_server_get_stats",
           "pp_ipc_client_open", "pp_ipc_submit", "pp_ipc_flush", "pp_ipc_collect",
           "pp_ipc_client_close"]


class _IpcConfig(C.Structure):
    _fields_ = [("max_clients", C.c_uint32), ("ingest_threads", C.c_uint32), ("source_ring_bytes", C.c_uint64),
                ("hit_ring_bytes", C.c_uint64)]


class _IpcStats(C.Structure):
    _fields_ = [("clients_attached", C.c_uint64), ("blocks_ingested", C.c_uint64), ("sources_ingested", C.c_uint64),
                ("hits_routed", C.c_uint64), ("hits_unrouted", C.c_uint64), ("hits_dropped", C.c_uint64),
                ("clients_dropped", C.c_uint64), ("events_tracked", C.c_uint64), ("clients_failed", C.c_uint64)]


_declared = False


def _lib():
    global _declared
    L = load_library()
    if not _declared:
        vp = C.c_void_p
        L.pp_ipc_server_create.restype = C.c_int
        L.pp_ipc_server_create.argtypes = [vp, C.c_char_p, C.POINTER(_IpcConfig), C.POINTER(vp)]
        L.pp_ipc_server_create_backend.restype = C.c_int
        L.pp_ipc_server_create_backend.argtypes = [vp, C.c_char_p, C.POINTER(_IpcConfig), C.POINTER(vp)]
        L.pp_ipc_server_destroy.restype = None
        L.pp_ipc_server_destroy.argtypes = [vp]
        L.pp_ipc_server_get_stats.restype = C.c_int
        L.pp_ipc_server_get_stats.argtypes = [vp, C.POINTER(_IpcStats)]
        L.pp_ipc_client_open.restype = C.c_int
        L.pp_ipc_client_open.argtypes = [C.c_char_p, C.POINTER(vp)]
        L.pp_ipc_submit.restype = C.c_int
        L.pp_ipc_submit.argtypes = [vp, vp, vp, vp, vp, C.c_size_t]
        L.pp_ipc_flush.restype = C.c_int
        L.pp_ipc_flush.argtypes = [vp]
        L.pp_ipc_collect.restype = C.c_int
        L.pp_ipc_collect.argtypes = [vp, vp, C.c_size_t, C.POINTER(C.c_size_t), C.c_int]
        L.pp_ipc_client_close.restype = None
        L.pp_ipc_client_close.argtypes = [vp]
        _declared = True
    return L


class IpcServer:
    """pp_ipc_server_create over a Propagator, or pp_ipc_server_create_backend over ``backend`` (the address of a
    ``pp_ipc_backend`` struct that outlives the server; the CPU tests pass their host-only echo back end)."""

    def __init__(self, propagator, name: str, *, max_clients: int = 16, source_ring_bytes: int = 0,
                 hit_ring_bytes: int = 0, backend=None, ingest_threads: int = 0):
        self._L = _lib()
        cfg = _IpcConfig(int(max_clients), int(ingest_threads), int(source_ring_bytes), int(hit_ring_bytes))
        s = C.c_void_p()
        if backend is not None:
            rc = self._L.pp_ipc_server_create_backend(C.c_void_p(backend), name.encode(), C.byref(cfg), C.byref(s))
        else:
            self._prop = propagator  # keep the handle alive
            rc = self._L.pp_ipc_server_create(propagator._h, name.encode(), C.byref(cfg), C.byref(s))
        if rc != PP_OK:
            raise PPError(rc, f"pp_ipc_server_create({name})")
        self._s = s
        self.name = name

    def stats(self) -> dict:
        st = _IpcStats()
        rc = self._L.pp_ipc_server_get_stats(self._s, C.byref(st))
        d = {f[0]: int(getattr(st, f[0])) for f in _IpcStats._fields_}
        d["error"] = rc
        return d

    def close(self):
        if getattr(self, "_s", None):
            self._L.pp_ipc_server_destroy(self._s)
            self._s = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


class IpcClient:
    """pp_ipc_client_open / pp_ipc_submit / pp_ipc_flush / pp_ipc_collect."""

    def __init__(self, name: str):
        self._L = _lib()
        c = C.c_void_p()
        rc = self._L.pp_ipc_client_open(name.encode(), C.byref(c))
        if rc != PP_OK:
            raise PPError(rc, f"pp_ipc_client_open({name})")
        self._c = c

    def _check(self, rc, what):
        if rc != PP_OK:
            raise PPError(rc, what)

    def submit(self, sources, event_ids, source_ids=None, lengths=None):
        rec = pack_sources(sources) if sources.dtype != SOURCE_DTYPE else np.ascontiguousarray(sources)
        ev = np.ascontiguousarray(event_ids, dtype=np.uint32)
        sid = None if source_ids is None else np.ascontiguousarray(source_ids, dtype=np.uint32)
        ln = None if lengths is None else np.ascontiguousarray(lengths, dtype=np.float32)
        assert ev.shape[0] == rec.shape[0]
        self._check(self._L.pp_ipc_submit(self._c, rec.ctypes.data, None if ln is None else ln.ctypes.data, ev.ctypes.data,
                                          None if sid is None else sid.ctypes.data, rec.shape[0]), "pp_ipc_submit")

    def flush(self):
        self._check(self._L.pp_ipc_flush(self._c), "pp_ipc_flush")

    def collect(self, cap: int = 1 << 16, block: bool = True) -> np.ndarray:
        tls = self.__dict__.setdefault("_collect_tls", threading.local())  # one landing buffer per calling thread
        out = getattr(tls, "buf", None)
        if out is None or out.shape[0] < cap:
            out = tls.buf = np.empty(cap, dtype=HIT_DTYPE)
        n = C.c_size_t(0)
        self._check(self._L.pp_ipc_collect(self._c, out.ctypes.data, cap, C.byref(n), 1 if block else 0), "pp_ipc_collect")
        return out[: n.value].copy()

    def collect_all(self) -> np.ndarray:
        """flush, then collect until this client's work is drained."""
        self.flush()
        parts = []
        while True:
            h = self.collect(block=True)
            if len(h) == 0:
                break
            parts.append(h)
        return np.concatenate(parts) if parts else np.empty(0, dtype=HIT_DTYPE)

    def close(self):
        if getattr(self, "_c", None):
            self._L.pp_ipc_client_close(self._c)
            self._c = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()
