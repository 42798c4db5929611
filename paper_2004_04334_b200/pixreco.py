"""Thin ctypes binding of ``include/pixreco.h`` — argument marshalling only.

Every step of the hot path runs inside ``libpixreco.so`` (CUDA, sm_100a).  There is no CPU
fallback: if the library cannot be built/loaded, importing callers get an exception, and if no
CUDA device is present ``pr_create`` returns ``PR_ERR_CUDA``.  This module imports nothing from
``oracle/``.

Two layers:
  * the raw ``pr_*`` functions with the same names as the C ABI (``lib()`` returns the CDLL);
  * :class:`PixReco` / :class:`EventSlot`, small conveniences that fill the C structs from numpy
    arrays / torch tensors and wrap the returned views as torch tensors (device) or numpy arrays
    (pinned host mirrors).  PyTorch is used only for device memory and streams.
"""
from __future__ import annotations

import ctypes
from ctypes import POINTER, c_char_p, c_float, c_int, c_int32, c_size_t, c_uint16, c_uint32, c_uint64, c_void_p

import numpy as np

from . import _build

PR_OK, PR_NOT_READY = 0, 1
PR_ERR_INVALID_ARG, PR_ERR_BAD_STATE, PR_ERR_CAPACITY, PR_ERR_INPUT_ORDER = -1, -2, -3, -4
PR_ERR_BAD_CALIB, PR_ERR_OOM, PR_ERR_CUDA = -5, -6, -7
PR_MEM_HOST_PINNED, PR_MEM_DEVICE = 1, 2
PR_WANT_DIGIS, PR_WANT_CHARGE, PR_WANT_LABELS, PR_WANT_CLUSTERS, PR_WANT_ERRORS, PR_WANT_HITS = 1, 2, 4, 8, 16, 32
PR_WANT_ALL = 63
PR_STATUS_INPUT_ORDER, PR_STATUS_CAPACITY = 1, 2
PR_POOL_DEVICE, PR_POOL_PINNED, PR_POOL_FAKE = 0, 1, 2
PR_INVALID_LABEL = 0xFFFFFFFF
PR_FLAG_KERNEL_TIMING, PR_FLAG_NO_GRAPH, PR_FLAG_UNPACK_OVERSUBSCRIBE, PR_FLAG_UNORDERED_INPUT = 1, 2, 4, 8

pr_done_fn = ctypes.CFUNCTYPE(None, c_void_p, c_int)


class pr_config(ctypes.Structure):
    _fields_ = [("struct_size", c_uint32), ("device", c_int32), ("n_modules", c_uint32),
                ("n_rows", c_uint16), ("n_cols", c_uint16), ("gain", c_void_p), ("pedestal", c_void_p),
                ("pixel_threshold_e", c_float), ("cluster_threshold_e", c_float),
                ("max_words_hint", c_uint32), ("max_events_in_flight", c_uint32),
                ("max_cached_bytes_device", c_uint64), ("max_cached_bytes_host", c_uint64), ("flags", c_uint32),
                ("pitch_row_um", c_float), ("pitch_col_um", c_float)]


class pr_input(ctypes.Structure):
    _fields_ = [("words", c_void_p), ("adc", c_void_p), ("n_words", c_uint32), ("mem_kind", c_uint32),
                ("want", c_uint32), ("event_id", c_uint64), ("done", pr_done_fn), ("user", c_void_p)]


_VIEWS = ["module", "row", "col", "adc", "word_idx", "charge", "label", "clus", "mod_digi_start",
          "mod_clus_start", "cl_label", "cl_size", "cl_module", "cl_charge", "cl_row", "cl_col",
          "err_word", "err_idx", "ht_x", "ht_y", "ht_xerr", "ht_yerr", "ht_rows", "ht_cols", "ht_flags"]
# name -> (numpy dtype, which counter gives the length)
VIEW_SPEC = {
    "module": (np.uint16, "n_digis"), "row": (np.uint16, "n_digis"), "col": (np.uint16, "n_digis"),
    "adc": (np.uint16, "n_digis"), "word_idx": (np.uint32, "n_digis"), "charge": (np.float32, "n_digis"),
    "label": (np.uint32, "n_digis"), "clus": (np.int32, "n_digis"),
    "mod_digi_start": (np.uint32, "n_modules+1"), "mod_clus_start": (np.uint32, "n_modules+1"),
    "cl_label": (np.uint32, "n_clusters"), "cl_size": (np.uint32, "n_clusters"),
    "cl_module": (np.uint16, "n_clusters"), "cl_charge": (np.float32, "n_clusters"),
    "cl_row": (np.float32, "n_clusters"), "cl_col": (np.float32, "n_clusters"),
    "err_word": (np.uint32, "n_errors"), "err_idx": (np.uint32, "n_errors"),
    "ht_x": (np.float32, "n_clusters"), "ht_y": (np.float32, "n_clusters"), "ht_xerr": (np.float32, "n_clusters"),
    "ht_yerr": (np.float32, "n_clusters"), "ht_rows": (np.uint32, "n_clusters"), "ht_cols": (np.uint32, "n_clusters"),
    "ht_flags": (np.uint16, "n_clusters"),
}


class pr_output(ctypes.Structure):
    _fields_ = ([("event_id", c_uint64)] +
                [(n, c_uint32) for n in ("n_words", "n_digis", "n_errors", "n_kept_digis", "n_clusters_all",
                                         "n_clusters", "status_bits", "n_modules")] +
                [("t_start_ns", c_uint64), ("t_end_ns", c_uint64)] +
                [("d_" + n, c_void_p) for n in _VIEWS] + [("h_" + n, c_void_p) for n in _VIEWS])


class pr_pool_stats(ctypes.Structure):
    _fields_ = [(n, c_uint64) for n in ("hits", "misses", "backend_allocs", "backend_frees", "bytes_live",
                                        "bytes_cached", "bytes_peak", "cross_stream_reuses")]


class pr_stats(ctypes.Structure):
    _fields_ = ([(n, c_uint64) for n in ("events_acquired", "events_produced", "words", "digis", "clusters",
                                         "kernel_launches", "memcpy_calls", "callbacks_fired")] +
                [("events_in_flight", c_uint32), ("max_events_in_flight", c_uint32),
                 ("device_pool", pr_pool_stats), ("host_pool", pr_pool_stats), ("timed_acquires", c_uint64),
                 ("unpack_ms", ctypes.c_double), ("cluster_ms", ctypes.c_double), ("finalize_ms", ctypes.c_double),
                 ("export_ms", ctypes.c_double)])


PR_STATIC_MAX_WORDS = 1 << 24
DIGIS_OUT_FIELDS = ("d_module", "d_row", "d_col", "d_adc", "d_word_idx", "d_charge", "d_err_word", "d_err_idx",
                    "d_mod_digi_start", "d_counters")


class pr_digis_out(ctypes.Structure):
    _fields_ = [(n, c_void_p) for n in DIGIS_OUT_FIELDS]


# every symbol include/pixreco.h declares: name -> (restype, argtypes)
SIGNATURES = {
    "pr_create": (c_int, [POINTER(pr_config), POINTER(c_void_p)]),
    "pr_destroy": (c_int, [c_void_p]),
    "pr_event_create": (c_int, [c_void_p, POINTER(c_void_p)]),
    "pr_event_destroy": (c_int, [c_void_p]),
    "pr_acquire": (c_int, [c_void_p, POINTER(pr_input), c_void_p]),
    "pr_acquire_batch": (c_int, [c_void_p, POINTER(pr_input), c_uint32, c_void_p]),
    "pr_query": (c_int, [c_void_p]),
    "pr_produce": (c_int, [c_void_p, POINTER(pr_output)]),
    "pr_produce_batch": (c_int, [c_void_p, POINTER(pr_output), c_uint32]),
    "pr_release": (c_int, [c_void_p]),
    "pr_release_on": (c_int, [c_void_p, c_void_p]),
    "pr_event_cuda_event": (c_void_p, [c_void_p]),
    "pr_stream_wait_event": (c_int, [c_void_p, c_void_p]),
    "pr_host_alloc": (c_void_p, [c_void_p, c_size_t]),
    "pr_host_free": (c_int, [c_void_p, c_void_p]),
    "pr_get_stats": (c_int, [c_void_p, POINTER(pr_stats)]),
    "pr_strerror": (c_char_p, [c_int]),
    "pr_last_cuda_error": (c_char_p, [c_void_p]),
    "pr_abi_version": (c_int, []),
    "pr_transfer": (c_int, [c_void_p, c_uint32, c_void_p, pr_done_fn, c_void_p]),
    "pr_digis_acquire": (c_int, [c_void_p, POINTER(pr_input), c_void_p]),
    "pr_digis_product": (c_int, [c_void_p, POINTER(c_void_p)]),
    "pr_product_info": (c_int, [c_void_p, POINTER(c_int32), POINTER(c_void_p), POINTER(c_void_p)]),
    "pr_clusters_acquire": (c_int, [c_void_p, c_void_p, c_uint32, c_void_p, POINTER(c_void_p), pr_done_fn, c_void_p]),
    "pr_occupancy_acquire": (c_int, [c_void_p, c_void_p, c_void_p, POINTER(c_void_p), pr_done_fn, c_void_p]),
    "pr_occupancy_produce": (c_int, [c_void_p, POINTER(c_void_p), POINTER(c_void_p), POINTER(c_void_p), POINTER(c_void_p)]),
    "pr_static_scratch_bytes": (c_size_t, []),
    "pr_static_setup": (c_int, [c_void_p]),
    "pr_unpack_static": (c_int, [c_void_p, c_void_p, c_void_p, c_uint32, POINTER(pr_digis_out), c_void_p]),
    "pr_pool_create": (c_int, [c_int, c_int, c_uint64, POINTER(c_void_p)]),
    "pr_pool_alloc": (c_void_p, [c_void_p, c_size_t, c_void_p]),
    "pr_pool_free": (c_int, [c_void_p, c_void_p, c_void_p, c_int]),
    "pr_pool_trim": (c_int, [c_void_p, c_uint64]),
    "pr_pool_get_stats": (c_int, [c_void_p, POINTER(pr_pool_stats)]),
    "pr_pool_destroy": (c_int, [c_void_p]),
    "pr_pool_fake_complete": (c_int, [c_void_p, c_void_p]),
    "pr_pool_bin_bytes": (c_uint64, [c_uint64]),
}

_lib = None


def lib() -> ctypes.CDLL:
    """Load (building in-tree if needed) libpixreco.so.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        cdll = ctypes.CDLL(_build.build())
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(cdll, name)          # AttributeError if the .so lacks a declared symbol
            fn.restype, fn.argtypes = res, args
        _lib = cdll
    return _lib


def __getattr__(name):          # pr_* functions as module attributes, same names as the C ABI
    if name in SIGNATURES:
        return getattr(lib(), name)
    raise AttributeError(name)


class prd_result(ctypes.Structure):
    _fields_ = [("wall_s", ctypes.c_double), ("acquire_us_median", ctypes.c_double), ("acquire_us_mean", ctypes.c_double),
                ("acquire_us_p99", ctypes.c_double), ("events", c_uint64), ("digis", c_uint64), ("clusters", c_uint64),
                ("produce_polls", c_uint64), ("status", c_int32), ("threads", c_uint32)]


class prd_event_record(ctypes.Structure):
    _fields_ = [("event_id", c_uint64), ("n_digis", c_uint32), ("n_errors", c_uint32), ("n_kept_digis", c_uint32),
                ("n_clusters_all", c_uint32), ("n_clusters", c_uint32), ("status_bits", c_uint32), ("thread", c_uint32),
                ("pad", c_uint32), ("hash_label", c_uint64), ("hash_cl_label", c_uint64)]


class prd_cluster_aos(ctypes.Structure):
    _fields_ = [("label", c_uint32), ("size", c_uint32), ("module", ctypes.c_uint16), ("flags", ctypes.c_uint16),
                ("charge", c_float), ("row", c_float), ("col", c_float), ("x_um", c_float), ("y_um", c_float),
                ("xerr_um", c_float), ("yerr_um", c_float), ("row_min", ctypes.c_uint16), ("row_max", ctypes.c_uint16),
                ("col_min", ctypes.c_uint16), ("col_max", ctypes.c_uint16)]


AOS_DTYPE = np.dtype([("label", "<u4"), ("size", "<u4"), ("module", "<u2"), ("flags", "<u2"), ("charge", "<f4"), ("row", "<f4"),
                      ("col", "<f4"), ("x_um", "<f4"), ("y_um", "<f4"), ("xerr_um", "<f4"), ("yerr_um", "<f4"),
                      ("row_min", "<u2"), ("row_max", "<u2"), ("col_min", "<u2"), ("col_max", "<u2")])


DRIVER_SIGNATURES = {
    "prd_clusters_to_aos": (c_int, [POINTER(pr_output), c_void_p, c_uint32]),
    "prd_run_streams": (c_int, [POINTER(c_void_p), POINTER(c_void_p), c_uint32, POINTER(pr_input), c_uint32, c_uint32, c_uint32,
                                c_uint32, c_void_p, c_void_p, POINTER(prd_result)]),
    "prd_run_streams_rec": (c_int, [POINTER(c_void_p), POINTER(c_void_p), c_uint32, POINTER(pr_input), c_uint32, c_uint32,
                                    c_uint32, c_uint32, c_void_p, c_void_p, POINTER(prd_event_record), POINTER(prd_result)]),
}
_driver = None


def driver() -> ctypes.CDLL:
    """libpixreco_driver.so: the multi-threaded C++ client of the C ABI (include/pixreco_driver.h)."""
    global _driver
    if _driver is None:
        lib()                                   # libpixreco.so first (the driver links against it)
        cdll = ctypes.CDLL(_build.build_driver())
        for name, (res, args) in DRIVER_SIGNATURES.items():
            fn = getattr(cdll, name)
            fn.restype, fn.argtypes = res, args
        _driver = cdll
    return _driver


def fnv1a32(words) -> int:
    """The fingerprint of prd_event_record (FNV-1a, 64 bit, over 32-bit words) of a numpy u32 array."""
    h = 1469598103934665603
    for v in np.asarray(words, dtype=np.uint32).tolist():
        h = ((h ^ v) * 1099511628211) & 0xFFFFFFFFFFFFFFFF
    return h


def run_streams(slots, streams, inputs, n_events, n_threads=1, first=0, spans=False, records=False):
    """One pr_acquire per event on its own stream (slot = stream = e mod len(slots)), issued from ``n_threads`` C++
    host threads.  ``inputs``: a ctypes array of pr_input.  Returns a dict of the prd_result fields (+ spans, + one
    prd_event_record per event under "records")."""
    n = len(slots)
    sl = (c_void_p * n)(*[s.ptr for s in slots])
    st = (c_void_p * n)(*[getattr(s, "cuda_stream", s) for s in streams])
    t0 = np.zeros(n_events, np.uint64) if spans else None
    t1 = np.zeros(n_events, np.uint64) if spans else None
    res = prd_result()
    rec = (prd_event_record * n_events)() if records else None
    rc = driver().prd_run_streams_rec(sl, st, n, inputs, len(inputs), first, n_events, n_threads,
                                      t0.ctypes.data if spans else None, t1.ctypes.data if spans else None, rec, ctypes.byref(res))
    if rc != 0:
        raise PixRecoError(rc, "prd_run_streams")
    out = {k: getattr(res, k) for k, _ in prd_result._fields_}
    if spans:
        out["t_start_ns"], out["t_end_ns"] = t0, t1
    if records:
        out["records"] = rec
    return out


def clusters_to_aos(out: "Output") -> np.ndarray:
    """The legacy consumer of the transfer stage: one record per cluster (numpy structured array, AOS_DTYPE) from the
    pinned-host mirrors of a produced event (prd_clusters_to_aos)."""
    n = out.n_clusters
    dst = np.zeros(n, AOS_DTYPE)
    assert dst.itemsize == ctypes.sizeof(prd_cluster_aos)
    rc = driver().prd_clusters_to_aos(ctypes.byref(out.raw), dst.ctypes.data if n else None, n)
    if rc < 0:
        raise PixRecoError(rc, "prd_clusters_to_aos")
    return dst[:rc]


class PixRecoError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        msg = lib().pr_strerror(code).decode()
        super().__init__(f"{where}: {msg} ({code})" + (f": {detail}" if detail else ""))


def _check(code: int, where: str, h=None):
    if code < 0:
        detail = lib().pr_last_cuda_error(h).decode() if (h and code == PR_ERR_CUDA) else ""
        raise PixRecoError(code, where, detail)
    return code


def _ptr(x) -> int:
    """Address of a numpy array or a torch tensor (CPU pinned or CUDA)."""
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()


class Output:
    """Counters + lazily wrapped views of one produced event."""

    def __init__(self, raw: pr_output, device: int):
        self.raw, self._device = raw, device
        for n, _ in pr_output._fields_[:11]:                  # event_id, eight counters, t_start_ns, t_end_ns
            setattr(self, n, int(getattr(raw, n)))

    def _len(self, name):
        key = VIEW_SPEC[name][1]
        return self.n_modules + 1 if key == "n_modules+1" else getattr(self, key)

    def host(self, name) -> np.ndarray | None:
        """Pinned-host mirror as a numpy view (None if not requested in ``want``)."""
        p = getattr(self.raw, "h_" + name)
        if not p:
            return None
        dt = np.dtype(VIEW_SPEC[name][0])
        n = self._len(name)
        buf = (ctypes.c_char * (n * dt.itemsize)).from_address(p)
        return np.frombuffer(buf, dtype=dt, count=n)

    def _device_bytes(self, name):
        import torch
        dt = np.dtype(VIEW_SPEC[name][0])
        nbytes = self._len(name) * dt.itemsize
        if nbytes == 0:
            return torch.empty(0, dtype=torch.uint8, device=f"cuda:{self._device}")

        class _Cai:
            pass
        holder = _Cai()
        holder.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "version": 2, "strides": None,
                                           "data": (int(getattr(self.raw, "d_" + name)), False)}
        return torch.as_tensor(holder, device=f"cuda:{self._device}")

    def device(self, name):
        """Device view as a torch tensor (no copy)."""
        import torch
        tdt = {np.dtype(np.uint16): torch.uint16, np.dtype(np.uint32): torch.uint32, np.dtype(np.int32): torch.int32,
               np.dtype(np.float32): torch.float32}[np.dtype(VIEW_SPEC[name][0])]
        return self._device_bytes(name).view(tdt)

    def to_numpy(self, name) -> np.ndarray:
        """Copy of the device view on the host (synchronising; for tests)."""
        return self._device_bytes(name).cpu().numpy().view(VIEW_SPEC[name][0]).copy()


class EventSlot:
    """One ``pr_event``.  acquire() returns at once; poll with query()/produce() or pass ``done``."""

    def __init__(self, owner: "PixReco"):
        self.owner = owner
        p = c_void_p()
        _check(lib().pr_event_create(owner.handle, ctypes.byref(p)), "pr_event_create", owner.handle)
        self.ptr = p
        self._keep = None

    def _input(self, words, adc, want, event_id, done):
        n = int(words.shape[0])
        is_np = isinstance(words, np.ndarray)
        kind = PR_MEM_HOST_PINNED if (is_np or not words.is_cuda) else PR_MEM_DEVICE
        cb = pr_done_fn(done) if done is not None else pr_done_fn()
        return pr_input(_ptr(words) if n else None, _ptr(adc) if n else None, n, kind, want, event_id, cb, None), cb

    def acquire(self, words, adc, stream=0, want=0, event_id=0, done=None) -> int:
        """``words``/``adc``: CUDA tensors (used in place) or pinned CPU tensors / numpy views of
        pinned memory.  ``stream``: a ``torch.cuda.Stream`` or raw ``cudaStream_t`` int."""
        inp, cb = self._input(words, adc, want, event_id, done)
        self._keep = (words, adc, cb)
        s = getattr(stream, "cuda_stream", stream)
        return _check(lib().pr_acquire(self.ptr, ctypes.byref(inp), c_void_p(s)), "pr_acquire", self.owner.handle)

    def acquire_batch(self, events, stream=0, want=0, done=None) -> int:
        """``events``: list of (words, adc) pairs, all of one memory kind."""
        arr = (pr_input * len(events))()
        keep = []
        for k, (w, a) in enumerate(events):
            arr[k], cb = self._input(w, a, want, k, done if k == 0 else None)
            keep.append((w, a, cb))
        self._keep = keep
        s = getattr(stream, "cuda_stream", stream)
        return _check(lib().pr_acquire_batch(self.ptr, arr, len(events), c_void_p(s)), "pr_acquire_batch", self.owner.handle)

    def transfer(self, want, stream=0, done=None) -> int:
        """Transfer on demand: after a PR_OK produce, copy the outputs in ``want`` to pinned host memory
        with exact-size DMA copies on ``stream``; the slot is in flight again until query/produce say PR_OK."""
        cb = pr_done_fn(done) if done is not None else pr_done_fn()
        self._keep_transfer = cb
        s = getattr(stream, "cuda_stream", stream)
        return _check(lib().pr_transfer(self.ptr, want, c_void_p(s), cb, None), "pr_transfer", self.owner.handle)

    def query(self) -> int:
        return _check(lib().pr_query(self.ptr), "pr_query", self.owner.handle)

    def produce(self, raise_on_error=True):
        """Returns (code, Output|None).  code is PR_NOT_READY if called too early."""
        out = pr_output()
        code = lib().pr_produce(self.ptr, ctypes.byref(out))
        if code == PR_NOT_READY:
            return code, None
        if code < 0 and (raise_on_error or code in (PR_ERR_INVALID_ARG, PR_ERR_BAD_STATE, PR_ERR_CUDA)):
            _check(code, "pr_produce", self.owner.handle)
        return code, Output(out, self.owner.device)

    def produce_batch(self, n: int, raise_on_error=True):
        outs = (pr_output * n)()
        code = lib().pr_produce_batch(self.ptr, outs, n)
        if code == PR_NOT_READY:
            return code, None
        if code < 0 and (raise_on_error or code in (PR_ERR_INVALID_ARG, PR_ERR_BAD_STATE, PR_ERR_CUDA)):
            _check(code, "pr_produce_batch", self.owner.handle)
        return code, [Output(outs[k], self.owner.device) for k in range(n)]

    # ---- chained modules: raw -> digis | digis -> clusters + hits | digis -> occupancy
    def digis_acquire(self, words, adc, stream=0, want=0, event_id=0, done=None) -> int:
        inp, cb = self._input(words, adc, want, event_id, done)
        self._keep = (words, adc, cb)
        s = getattr(stream, "cuda_stream", stream)
        return _check(lib().pr_digis_acquire(self.ptr, ctypes.byref(inp), c_void_p(s)), "pr_digis_acquire", self.owner.handle)

    def digis_product(self) -> int:
        """The product handle (an address) of this slot's digis acquire."""
        p = c_void_p()
        _check(lib().pr_digis_product(self.ptr, ctypes.byref(p)), "pr_digis_product", self.owner.handle)
        return p.value

    def clusters_acquire(self, product, want=0, own_stream=0, done=None) -> int:
        """Returns the raw stream the work went to (the producer's for the first consumer, else ``own_stream``)."""
        cb = pr_done_fn(done) if done is not None else pr_done_fn()
        self._keep = cb
        used = c_void_p()
        s = getattr(own_stream, "cuda_stream", own_stream)
        _check(lib().pr_clusters_acquire(self.ptr, c_void_p(product), want, c_void_p(s), ctypes.byref(used), cb, None),
               "pr_clusters_acquire", self.owner.handle)
        return used.value or 0

    def occupancy_acquire(self, product, own_stream=0, done=None) -> int:
        cb = pr_done_fn(done) if done is not None else pr_done_fn()
        self._keep = cb
        used = c_void_p()
        s = getattr(own_stream, "cuda_stream", own_stream)
        _check(lib().pr_occupancy_acquire(self.ptr, c_void_p(product), c_void_p(s), ctypes.byref(used), cb, None),
               "pr_occupancy_acquire", self.owner.handle)
        return used.value or 0

    def occupancy_produce(self):
        """Returns (code, count, adc_sum): numpy views of the pinned mirrors [n_modules] (None if early)."""
        hc, ha = c_void_p(), c_void_p()
        code = lib().pr_occupancy_produce(self.ptr, None, None, ctypes.byref(hc), ctypes.byref(ha))
        if code == PR_NOT_READY:
            return code, None, None
        if code in (PR_ERR_INVALID_ARG, PR_ERR_BAD_STATE, PR_ERR_CUDA):
            _check(code, "pr_occupancy_produce", self.owner.handle)
        M = self.owner.n_modules
        mk = lambda p: np.frombuffer((ctypes.c_char * (4 * M)).from_address(p.value), dtype=np.uint32, count=M)
        return code, mk(hc), mk(ha)

    def release(self) -> int:
        code = _check(lib().pr_release(self.ptr), "pr_release", self.owner.handle)
        if code == PR_OK:
            self._keep = None
        return code

    def release_on(self, consumer_stream) -> int:
        """Release while work queued on ``consumer_stream`` may still read the device views."""
        s = getattr(consumer_stream, "cuda_stream", consumer_stream)
        code = _check(lib().pr_release_on(self.ptr, c_void_p(s)), "pr_release_on", self.owner.handle)
        if code == PR_OK:
            self._keep = None
        return code

    @property
    def cuda_event(self) -> int:
        return lib().pr_event_cuda_event(self.ptr)

    def stream_wait(self, consumer_stream) -> int:
        """make ``consumer_stream`` wait for this slot's work unless already complete."""
        s = getattr(consumer_stream, "cuda_stream", consumer_stream)
        return _check(lib().pr_stream_wait_event(self.ptr, c_void_p(s)), "pr_stream_wait_event", self.owner.handle)

    def destroy(self):
        if self.ptr:
            _check(lib().pr_event_destroy(self.ptr), "pr_event_destroy", self.owner.handle)
            self.ptr = None


class PixReco:
    """One ``pr_handle``: calibration tables + pools on one device."""

    def __init__(self, gain, pedestal, n_rows=160, n_cols=416, pixel_threshold_e=1000.0, cluster_threshold_e=4000.0,
                 device=0, max_words_hint=0, max_events_in_flight=0, max_cached_bytes_device=0, max_cached_bytes_host=0,
                 flags=0, pitch_row_um=0.0, pitch_col_um=0.0):
        gain = np.ascontiguousarray(gain, np.float32)
        pedestal = np.ascontiguousarray(pedestal, np.float32)
        if gain.shape != pedestal.shape or gain.ndim != 1:
            raise ValueError("gain/pedestal must be 1-D arrays of equal length")
        cfg = pr_config(ctypes.sizeof(pr_config), device, gain.shape[0], n_rows, n_cols, gain.ctypes.data,
                        pedestal.ctypes.data, pixel_threshold_e, cluster_threshold_e, max_words_hint,
                        max_events_in_flight, max_cached_bytes_device, max_cached_bytes_host, flags, pitch_row_um, pitch_col_um)
        h = c_void_p()
        _check(lib().pr_create(ctypes.byref(cfg), ctypes.byref(h)), "pr_create")
        self.handle, self.device, self.n_modules = h, device, int(gain.shape[0])
        self._slots = []

    def slot(self) -> EventSlot:
        s = EventSlot(self)
        self._slots.append(s)
        return s

    def host_alloc(self, nbytes: int) -> int:
        p = lib().pr_host_alloc(self.handle, nbytes)
        if not p:
            raise PixRecoError(PR_ERR_OOM, "pr_host_alloc")
        return p

    def host_array(self, count: int, dtype) -> np.ndarray:
        """A numpy array living in pinned memory from the handle's host pool."""
        dt = np.dtype(dtype)
        nbytes = max(count * dt.itemsize, 1)
        p = self.host_alloc(nbytes)
        buf = (ctypes.c_char * nbytes).from_address(p)
        arr = np.frombuffer(buf, dtype=dt, count=count)
        return arr

    def host_free(self, arr_or_ptr):
        p = arr_or_ptr.ctypes.data if isinstance(arr_or_ptr, np.ndarray) else arr_or_ptr
        _check(lib().pr_host_free(self.handle, c_void_p(p)), "pr_host_free", self.handle)

    def unpack_static(self, words, adc, out: dict, stream=0, n_words=None) -> int:
        """pr_unpack_static: raw words -> digis into the caller's CUDA tensors ``out[name]`` (names: DIGIS_OUT_FIELDS),
        no allocation anywhere; returns the C return code (PR_OK, or an error such as PR_ERR_CAPACITY) without raising."""
        n = int(words.shape[0]) if n_words is None else int(n_words)
        o = pr_digis_out(*[c_void_p(_ptr(out[k])) for k in DIGIS_OUT_FIELDS])
        return lib().pr_unpack_static(self.handle, c_void_p(_ptr(words)) if words is not None and int(words.shape[0]) else None,
                                      c_void_p(_ptr(adc)) if adc is not None and int(adc.shape[0]) else None, n, ctypes.byref(o),
                                      c_void_p(getattr(stream, "cuda_stream", stream)))

    def stats(self) -> dict:
        st = pr_stats()
        _check(lib().pr_get_stats(self.handle, ctypes.byref(st)), "pr_get_stats", self.handle)

        def conv(s):
            return {n: (conv(getattr(s, n)) if isinstance(getattr(s, n), ctypes.Structure) else
                        (float(getattr(s, n)) if t is ctypes.c_double else int(getattr(s, n))))
                    for n, t in s._fields_}
        return conv(st)

    def close(self):
        if self.handle:
            _check(lib().pr_destroy(self.handle), "pr_destroy")
            self.handle = None
            for s in self._slots:
                s.ptr = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()
