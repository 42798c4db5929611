"""Seeded synthetic inputs for the pixel local-reconstruction hot path.

This module is the single input generator shared by the CUDA path's tests/bench and by the
oracle's tests.  It contains none of the method's arithmetic (no decode, calibration, clustering
or reduction): it draws shapes and ADC values, *encodes* raw words and draws calibration tables.
It imports neither ``oracle`` nor the CUDA binding.

Workloads follow BASELINE.json ``configs[0..4]`` with the readings listed in DESIGN.md
("Input recipe").  The paper gives
no workload of its own.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 20200404
N_ROWS, N_COLS = 160, 416
PIXEL_THRESHOLD_E = 1000.0
CLUSTER_THRESHOLD_E = 4000.0
# events per workload as BASELINE.json configs[i] states them
CONFIG_EVENTS = {0: 1, 1: 1, 2: 64, 3: 256, 4: 16}
CONFIG_NAMES = {
    0: "configs[0] tiny correctness event",
    1: "configs[1] Run-3 HLT-like single event",
    2: "configs[2] concurrent-event batch (64 x configs[1] shape, 8 streams in flight)",
    3: "configs[3] high-pileup",
    4: "configs[4] clustering stress",
}

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pixgen.c")
_LIB = os.path.join(_HERE, "libpixgen.so")


class _Params(ctypes.Structure):
    _fields_ = [
        ("n_modules", ctypes.c_uint32), ("n_rows", ctypes.c_uint32), ("n_cols", ctypes.c_uint32),
        ("lambda_", ctypes.c_double), ("hot_modules", ctypes.c_uint32), ("hot_factor", ctypes.c_double),
        ("compact_mean", ctypes.c_double), ("frac_elongated", ctypes.c_double),
        ("elongated_mean", ctypes.c_double), ("frac_strip", ctypes.c_double),
        ("strip_min", ctypes.c_uint32), ("strip_max", ctypes.c_uint32), ("p_touch", ctypes.c_double),
        ("fill_pixels", ctypes.c_uint32), ("err_frac", ctypes.c_double), ("adc_law", ctypes.c_uint32),
    ]


class _Stats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_uint64) for n in
                ("n_words", "n_digis", "n_errors", "n_seeded_clusters", "max_digis_per_module")]


def build(force: bool = False) -> str:
    """Compile pixgen.c with gcc (in-tree .so).  Idempotent."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.pixgen_default_params.argtypes = [ctypes.c_uint32, ctypes.POINTER(_Params)]
        lib.pixgen_default_params.restype = ctypes.c_int
        lib.pixgen_calib.argtypes = [ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint32,
                                     ctypes.c_void_p, ctypes.c_void_p]
        lib.pixgen_calib.restype = ctypes.c_int
        lib.pixgen_event.argtypes = [ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint32,
                                     ctypes.POINTER(_Params), ctypes.POINTER(ctypes.c_void_p),
                                     ctypes.POINTER(ctypes.c_void_p), ctypes.POINTER(_Stats)]
        lib.pixgen_event.restype = ctypes.c_int
        lib.pixgen_free.argtypes = [ctypes.c_void_p]
        lib.pixgen_free.restype = None
        _lib = lib
    return _lib


@dataclass
class Calib:
    gain: np.ndarray           # f32 [M]
    pedestal: np.ndarray       # f32 [M]
    pixel_threshold_e: float = PIXEL_THRESHOLD_E
    cluster_threshold_e: float = CLUSTER_THRESHOLD_E

    @property
    def n_modules(self) -> int:
        return int(self.gain.shape[0])


@dataclass
class Event:
    words: np.ndarray          # u32 [W]
    adc: np.ndarray            # u16 [W]
    n_modules: int
    n_rows: int = N_ROWS
    n_cols: int = N_COLS
    stats: dict = field(default_factory=dict)

    @property
    def n_words(self) -> int:
        return int(self.words.shape[0])


def default_params(config: int) -> dict:
    p = _Params()
    if _load().pixgen_default_params(config, ctypes.byref(p)) != 0:
        raise ValueError(f"unknown config {config}")
    return {n: getattr(p, n) for n, _ in _Params._fields_}


def make_calib(config: int, seed: int = BASE_SEED, n_modules: int | None = None) -> Calib:
    """Per-workload calibration tables: gain ~ N(80,5) e/ADC, pedestal ~ N(0,200) e (A21)."""
    M = n_modules if n_modules is not None else default_params(config)["n_modules"]
    gain = np.empty(M, np.float32)
    ped = np.empty(M, np.float32)
    _load().pixgen_calib(seed, config, M, gain.ctypes.data, ped.ctypes.data)
    return Calib(gain, ped)


def make_event(config: int, event: int = 0, seed: int = BASE_SEED, **overrides) -> Event:
    """One seeded event of workload ``config`` (0..4); ``overrides`` replace generator knobs
    (e.g. ``n_modules=8``, ``fill_pixels=2000``, ``hot_factor=14.3``)."""
    lib = _load()
    p = _Params()
    if lib.pixgen_default_params(config, ctypes.byref(p)) != 0:
        raise ValueError(f"unknown config {config}")
    for k, v in overrides.items():
        k = "lambda_" if k == "lambda" else k
        if not hasattr(p, k):
            raise TypeError(f"unknown generator knob {k!r}")
        setattr(p, k, v)
    pw, pa, st = ctypes.c_void_p(), ctypes.c_void_p(), _Stats()
    rc = lib.pixgen_event(seed, config, event, ctypes.byref(p), ctypes.byref(pw), ctypes.byref(pa),
                          ctypes.byref(st))
    if rc != 0:
        raise ValueError("pixgen_event: bad parameters")
    W = int(st.n_words)
    try:
        words = np.ctypeslib.as_array(ctypes.cast(pw, ctypes.POINTER(ctypes.c_uint32)), (max(W, 1),))[:W].copy()
        adc = np.ctypeslib.as_array(ctypes.cast(pa, ctypes.POINTER(ctypes.c_uint16)), (max(W, 1),))[:W].copy()
    finally:
        lib.pixgen_free(pw)
        lib.pixgen_free(pa)
    stats = {n: int(getattr(st, n)) for n, _ in _Stats._fields_}
    return Event(words, adc, int(p.n_modules), int(p.n_rows), int(p.n_cols), stats)


# ---------------------------------------------------------------------------------------------
# Hand-made events for edge cases (encoding only; BASELINE.json configs[0] word format:
# bit31 = error flag, bits 30:20 module, 19:12 row, 11:3 col; bits 2:0 reserved, A1).
# ---------------------------------------------------------------------------------------------
def encode_word(module: int, row: int, col: int, low_bits: int = 0) -> int:
    return ((module & 0x7FF) << 20) | ((row & 0xFF) << 12) | ((col & 0x1FF) << 3) | (low_bits & 7)


def event_from_pixels(pixels, n_modules: int, n_rows: int = N_ROWS, n_cols: int = N_COLS) -> Event:
    """``pixels``: iterable of (module, row, col, adc) or raw ints (taken verbatim as words with
    adc 0, e.g. error words).  Order is kept as given."""
    words, adc = [], []
    for p in pixels:
        if isinstance(p, (int, np.integer)):
            words.append(int(p) & 0xFFFFFFFF)
            adc.append(0)
        else:
            m, r, c, a = p
            words.append(encode_word(m, r, c))
            adc.append(int(a))
    return Event(np.asarray(words, np.uint32).reshape(-1), np.asarray(adc, np.uint16).reshape(-1),
                 n_modules, n_rows, n_cols)


def flat_calib(n_modules: int, gain: float = 80.0, pedestal: float = 0.0,
               pixel_threshold_e: float = PIXEL_THRESHOLD_E,
               cluster_threshold_e: float = CLUSTER_THRESHOLD_E) -> Calib:
    return Calib(np.full(n_modules, gain, np.float32), np.full(n_modules, pedestal, np.float32),
                 pixel_threshold_e, cluster_threshold_e)
