"""oracle — TEST INFRASTRUCTURE, NOT PRODUCT.

ctypes front end of ``pixreco_oracle.c`` (the plain single-threaded CPU definition of the hot
path).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2004_04334_b200`` and shares no code with the CUDA path.

What the functions compute and which reading of the sources each follows is stated on the C
functions (``pixreco_oracle.c``) and in DESIGN.md.  With respect to the PAPER the path is
"parity unpinned": PAPER.md prints no value for it (L118 defers to its ref. [8]); the pins are
BASELINE.json's definitions, worked values, brute force and library routines (tests/).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

INVALID = 0xFFFFFFFF
PITCH_ROW_UM, PITCH_COL_UM = 100.0, 150.0      # A26: local x runs along the row index, local y along the col index

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pixreco_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off (nothing but the explicit fmaf may fuse).  Idempotent."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        for name in ("po_decode", "po_calibrate", "po_cluster", "po_reduce", "po_hits", "po_run", "po_check_exact_sums"):
            getattr(_lib, name).restype = ctypes.c_int
        _lib.po_decode.restype = None
        _lib.po_calibrate.restype = None
        _lib.po_occupancy.restype = None
        _lib.po_bucket.restype = None
    return _lib


def _p(a):
    return ctypes.c_void_p(a.ctypes.data)


def _u32(x):
    return ctypes.c_uint32(int(x))


@dataclass
class Result:
    """Everything the chain produces for one event (arrays trimmed to their true lengths)."""
    n_words: int
    n_digis: int
    n_errors: int
    n_kept_digis: int
    n_clusters_all: int
    n_clusters: int
    sorted_ok: bool
    module: np.ndarray      # u16 [D]
    row: np.ndarray         # u16 [D]
    col: np.ndarray         # u16 [D]
    adc: np.ndarray         # u16 [D]
    word_idx: np.ndarray    # u32 [D]
    err_word: np.ndarray    # u32 [E]
    err_idx: np.ndarray     # u32 [E]
    mod_digi_start: np.ndarray  # u32 [M+1]
    charge: np.ndarray      # f32 [D]
    kept: np.ndarray        # u8  [D]
    label: np.ndarray       # u32 [D]
    cl_label: np.ndarray    # u32 [N]
    cl_module: np.ndarray   # u16 [N]
    cl_size: np.ndarray     # u32 [N]
    cl_charge: np.ndarray   # f32 [N]
    cl_row: np.ndarray      # f32 [N]
    cl_col: np.ndarray      # f32 [N]
    clus: np.ndarray        # i32 [D]
    mod_clus_start: np.ndarray  # u32 [M+1]
    ht_x: np.ndarray        # f32 [N] local x (um), hit k belongs to cluster k
    ht_y: np.ndarray        # f32 [N]
    ht_xerr: np.ndarray     # f32 [N]
    ht_yerr: np.ndarray     # f32 [N]
    ht_rows: np.ndarray     # u32 [N] minRow | maxRow << 16
    ht_cols: np.ndarray     # u32 [N] minCol | maxCol << 16
    ht_flags: np.ndarray    # u16 [N] bit0 touches a row border, bit1 a col border


def decode(words, adc, n_modules, n_rows=160, n_cols=416):
    """O1.  Returns dict(module,row,col,adc,word_idx,err_word,err_idx,mod_digi_start,sorted_ok)."""
    words = np.ascontiguousarray(words, np.uint32)
    adc = np.ascontiguousarray(adc, np.uint16)
    W = words.shape[0]
    cap = max(W, 1)
    mod, row, col, a = (np.zeros(cap, np.uint16) for _ in range(4))
    widx, ew, ei = (np.zeros(cap, np.uint32) for _ in range(3))
    mds = np.zeros(n_modules + 1, np.uint32)
    D, E, ok = ctypes.c_uint32(), ctypes.c_uint32(), ctypes.c_uint32()
    _load().po_decode(_p(words), _p(adc), _u32(W), _u32(n_modules), _u32(n_rows), _u32(n_cols),
                      _p(mod), _p(row), _p(col), _p(a), _p(widx), _p(ew), _p(ei), _p(mds),
                      ctypes.byref(D), ctypes.byref(E), ctypes.byref(ok))
    D, E = D.value, E.value
    return dict(module=mod[:D], row=row[:D], col=col[:D], adc=a[:D], word_idx=widx[:D],
                err_word=ew[:E], err_idx=ei[:E], mod_digi_start=mds, sorted_ok=bool(ok.value))


def calibrate(adc, module, gain, pedestal, pixel_threshold_e):
    """O2.  Returns (charge f32[D], kept u8[D])."""
    adc = np.ascontiguousarray(adc, np.uint16)
    module = np.ascontiguousarray(module, np.uint16)
    gain = np.ascontiguousarray(gain, np.float32)
    pedestal = np.ascontiguousarray(pedestal, np.float32)
    D = adc.shape[0]
    charge = np.zeros(max(D, 1), np.float32)
    kept = np.zeros(max(D, 1), np.uint8)
    nk = ctypes.c_uint32()
    _load().po_calibrate(_u32(D), _p(adc), _p(module), _p(gain), _p(pedestal),
                         ctypes.c_float(pixel_threshold_e), _p(charge), _p(kept), ctypes.byref(nk))
    return charge[:D], kept[:D]


def cluster(module, row, col, kept, n_modules, n_rows=160, n_cols=416):
    """O3.  Returns label u32[D] (INVALID for not-kept digis)."""
    module = np.ascontiguousarray(module, np.uint16)
    row = np.ascontiguousarray(row, np.uint16)
    col = np.ascontiguousarray(col, np.uint16)
    kept = np.ascontiguousarray(kept, np.uint8)
    D = module.shape[0]
    label = np.zeros(max(D, 1), np.uint32)
    rc = _load().po_cluster(_u32(D), _u32(n_modules), _u32(n_rows), _u32(n_cols), _p(module), _p(row),
                            _p(col), _p(kept), _p(label))
    if rc != 0:
        raise MemoryError("po_cluster")
    return label[:D]


def reduce(label, charge, module, row, col, cluster_threshold_e, n_modules):
    """O4.  Returns dict(cl_label, cl_module, cl_size, cl_charge, cl_row, cl_col, clus,
    mod_clus_start, n_clusters_all, n_clusters)."""
    label = np.ascontiguousarray(label, np.uint32)
    charge = np.ascontiguousarray(charge, np.float32)
    module = np.ascontiguousarray(module, np.uint16)
    row = np.ascontiguousarray(row, np.uint16)
    col = np.ascontiguousarray(col, np.uint16)
    D = label.shape[0]
    cap = max(D, 1)
    cl_label, cl_size = np.zeros(cap, np.uint32), np.zeros(cap, np.uint32)
    cl_module = np.zeros(cap, np.uint16)
    cl_charge, cl_row, cl_col = (np.zeros(cap, np.float32) for _ in range(3))
    clus = np.zeros(cap, np.int32)
    mcs = np.zeros(n_modules + 1, np.uint32)
    nall, N = ctypes.c_uint32(), ctypes.c_uint32()
    rc = _load().po_reduce(_u32(D), _u32(n_modules), _p(label), _p(charge), _p(module), _p(row), _p(col),
                           ctypes.c_float(cluster_threshold_e), _p(cl_label), _p(cl_module), _p(cl_size),
                           _p(cl_charge), _p(cl_row), _p(cl_col), _p(clus), _p(mcs),
                           ctypes.byref(nall), ctypes.byref(N))
    if rc != 0:
        raise ArithmeticError("po_reduce: a kept charge is not a multiple of 2^-14 (pixel threshold < 512?)")
    N = N.value
    return dict(cl_label=cl_label[:N], cl_module=cl_module[:N], cl_size=cl_size[:N], cl_charge=cl_charge[:N],
                cl_row=cl_row[:N], cl_col=cl_col[:N], clus=clus[:D], mod_clus_start=mcs,
                n_clusters_all=nall.value, n_clusters=N)


def hits(clus, charge, row, col, n_clusters, n_rows=160, n_cols=416, pitch_row_um=PITCH_ROW_UM, pitch_col_um=PITCH_COL_UM):
    """O5.  Returns dict(ht_x, ht_y, ht_xerr, ht_yerr, ht_rows, ht_cols, ht_flags) for the kept clusters 0..N-1."""
    clus = np.ascontiguousarray(clus, np.int32)
    charge = np.ascontiguousarray(charge, np.float32)
    row = np.ascontiguousarray(row, np.uint16)
    col = np.ascontiguousarray(col, np.uint16)
    D, N = clus.shape[0], int(n_clusters)
    cap = max(N, 1)
    x, y, xe, ye = (np.zeros(cap, np.float32) for _ in range(4))
    rows, cols = np.zeros(cap, np.uint32), np.zeros(cap, np.uint32)
    flags = np.zeros(cap, np.uint16)
    rc = _load().po_hits(_u32(D), _u32(N), _u32(n_rows), _u32(n_cols), _p(clus), _p(charge), _p(row), _p(col),
                         ctypes.c_double(pitch_row_um), ctypes.c_double(pitch_col_um),
                         _p(x), _p(y), _p(xe), _p(ye), _p(rows), _p(cols), _p(flags))
    if rc != 0:
        raise MemoryError("po_hits")
    return dict(ht_x=x[:N], ht_y=y[:N], ht_xerr=xe[:N], ht_yerr=ye[:N], ht_rows=rows[:N], ht_cols=cols[:N],
                ht_flags=flags[:N])


def occupancy(module, adc, kept, n_modules):
    """Kept digis and their ADC sum per module (the second consumer of the digis, NEXT-2).  Returns (count u32[M], adc_sum u32[M])."""
    module = np.ascontiguousarray(module, np.uint16)
    adc = np.ascontiguousarray(adc, np.uint16)
    kept = np.ascontiguousarray(kept, np.uint8)
    cnt, tot = np.zeros(n_modules, np.uint32), np.zeros(n_modules, np.uint32)
    _load().po_occupancy(_u32(module.shape[0]), _u32(n_modules), _p(module), _p(adc), _p(kept), _p(cnt), _p(tot))
    return cnt, tot


class Workspace:
    """Caller-owned output arrays of capacity W for :func:`run` (so timing excludes numpy allocs)."""

    def __init__(self, capacity: int, n_modules: int):
        cap = max(int(capacity), 1)
        self.capacity, self.n_modules = cap, n_modules
        self.u16 = [np.zeros(cap, np.uint16) for _ in range(5)]   # module,row,col,adc,cl_module
        self.u32 = [np.zeros(cap, np.uint32) for _ in range(6)]   # word_idx,err_word,err_idx,label,cl_label,cl_size
        self.f32 = [np.zeros(cap, np.float32) for _ in range(4)]  # charge,cl_charge,cl_row,cl_col
        self.hit_f32 = [np.zeros(cap, np.float32) for _ in range(4)]   # ht_x,ht_y,ht_xerr,ht_yerr
        self.hit_u32 = [np.zeros(cap, np.uint32) for _ in range(2)]    # ht_rows,ht_cols
        self.hit_flags = np.zeros(cap, np.uint16)
        self.kept = np.zeros(cap, np.uint8)
        self.clus = np.zeros(cap, np.int32)
        self.mds = np.zeros(n_modules + 1, np.uint32)
        self.mcs = np.zeros(n_modules + 1, np.uint32)
        self.counters = np.zeros(8, np.uint32)


def run_raw(words, adc, n_modules, n_rows, n_cols, gain, pedestal, pix_thr, clus_thr, ws: Workspace,
            pitch_row_um=PITCH_ROW_UM, pitch_col_um=PITCH_COL_UM) -> int:
    """The whole chain O1..O5 into ``ws`` (no trimming, no copies).  Returns po_run's rc."""
    mod, row, col, a, clm = ws.u16
    widx, ew, ei, label, cll, cls = ws.u32
    q, clq, clr, clc = ws.f32
    hx, hy, hxe, hye = ws.hit_f32
    hr, hc = ws.hit_u32
    return _load().po_run(_p(words), _p(adc), _u32(words.shape[0]), _u32(n_modules), _u32(n_rows), _u32(n_cols),
                          _p(gain), _p(pedestal), ctypes.c_float(pix_thr), ctypes.c_float(clus_thr),
                          _p(mod), _p(row), _p(col), _p(a), _p(widx), _p(ew), _p(ei), _p(ws.mds),
                          _p(q), _p(ws.kept), _p(label), _p(cll), _p(clm), _p(cls), _p(clq), _p(clr), _p(clc),
                          _p(ws.clus), _p(ws.mcs), ctypes.c_double(pitch_row_um), ctypes.c_double(pitch_col_um),
                          _p(hx), _p(hy), _p(hxe), _p(hye), _p(hr), _p(hc), _p(ws.hit_flags), _p(ws.counters))


def run(words, adc, n_modules, gain, pedestal, pixel_threshold_e=1000.0, cluster_threshold_e=4000.0,
        n_rows=160, n_cols=416, pitch_row_um=PITCH_ROW_UM, pitch_col_um=PITCH_COL_UM) -> Result:
    """The whole chain O1..O5 on one event."""
    words = np.ascontiguousarray(words, np.uint32)
    adc = np.ascontiguousarray(adc, np.uint16)
    gain = np.ascontiguousarray(gain, np.float32)
    pedestal = np.ascontiguousarray(pedestal, np.float32)
    assert gain.shape[0] == n_modules and pedestal.shape[0] == n_modules and adc.shape == words.shape
    ws = Workspace(words.shape[0], n_modules)
    rc = run_raw(words, adc, n_modules, n_rows, n_cols, gain, pedestal, pixel_threshold_e,
                 cluster_threshold_e, ws, pitch_row_um, pitch_col_um)
    if rc == -2:
        raise ArithmeticError("a kept charge is not a multiple of 2^-14 (pixel threshold < 512?)")
    if rc != 0:
        raise MemoryError("po_run")
    D, E, nk, nall, N, ok = (int(x) for x in ws.counters[:6])
    mod, row, col, a, clm = ws.u16
    widx, ew, ei, label, cll, cls = ws.u32
    q, clq, clr, clc = ws.f32
    hx, hy, hxe, hye = ws.hit_f32
    hr, hc = ws.hit_u32
    return Result(words.shape[0], D, E, nk, nall, N, bool(ok), mod[:D], row[:D], col[:D], a[:D], widx[:D],
                  ew[:E], ei[:E], ws.mds, q[:D], ws.kept[:D], label[:D], cll[:N], clm[:N], cls[:N], clq[:N],
                  clr[:N], clc[:N], ws.clus[:D], ws.mcs, hx[:N], hy[:N], hxe[:N], hye[:N], hr[:N], hc[:N],
                  ws.hit_flags[:N])


def bucket(words, adc, n_modules, n_rows=160, n_cols=416):
    """O0 (A31): stable bucket sort of the words by module (error / invalid words last).  Returns (words, adc, orig)."""
    words = np.ascontiguousarray(words, np.uint32)
    adc = np.ascontiguousarray(adc, np.uint16)
    W = words.shape[0]
    ow, oa, orig = np.zeros(W, np.uint32), np.zeros(W, np.uint16), np.zeros(W, np.uint32)
    _load().po_bucket(_p(words), _p(adc), _u32(W), _u32(n_modules), _u32(n_rows), _u32(n_cols), _p(ow), _p(oa), _p(orig))
    return ow, oa, orig


def run_unordered(words, adc, n_modules, gain, pedestal, pixel_threshold_e=1000.0, cluster_threshold_e=4000.0,
                  n_rows=160, n_cols=416, pitch_row_um=PITCH_ROW_UM, pitch_col_um=PITCH_COL_UM) -> Result:
    """The chain for words in arbitrary order (A31): O0 bucket, then O1..O5 on the bucketed stream, with word_idx and
    err_idx mapped back to the positions of the words in the INPUT."""
    ow, oa, orig = bucket(words, adc, n_modules, n_rows, n_cols)
    r = run(ow, oa, n_modules, gain, pedestal, pixel_threshold_e, cluster_threshold_e, n_rows, n_cols, pitch_row_um, pitch_col_um)
    r.word_idx = orig[r.word_idx]
    r.err_idx = orig[r.err_idx]
    return r


def check_exact_sums(label, charge, col) -> int:
    """O6 (A9): 0 if the exact-sum claims hold for this event; O(D x clusters), small events only."""
    label = np.ascontiguousarray(label, np.uint32)
    charge = np.ascontiguousarray(charge, np.float32)
    col = np.ascontiguousarray(col, np.uint16)
    return _load().po_check_exact_sums(_u32(label.shape[0]), _p(label), _p(charge), _p(col))
