"""Pins of the oracle's hit step (po_hits, readings A26-A30 in DESIGN.md; the step after clustering in the paper's
Fig. 1; the paper prints no value for it, L118).  Worked values from tests/golden, closed forms,
numpy min/max for the bounding boxes and scipy.ndimage.center_of_mass for the positions."""
import numpy as np
import pytest
import scipy.ndimage as ndi

import oracle
from paper_2004_04334_b200 import workloads as wl

R, C = 160, 416


def _golden_hits(golden_dir):
    rows = []
    with open(f"{golden_dir}/worked_values.txt") as f:
        for line in f:
            t = line.split()
            if t and t[0] == "hit":
                k = t.index("->")
                px = [(int(t[i]), int(t[i + 1]), int(t[i + 2])) for i in range(1, k, 3)]
                rows.append((px, t[k + 1:]))
    return rows


def _run(px, M=2, module=1):
    ev = wl.event_from_pixels([(module, r, c, a) for r, c, a in px], M)
    cal = wl.flat_calib(M, 80.0, 0.0)
    return oracle.run(ev.words, ev.adc, M, cal.gain, cal.pedestal)


def test_worked_hits(golden_dir):
    rows = _golden_hits(golden_dir)
    assert len(rows) >= 7
    for px, want in rows:
        o = _run(px)
        assert o.n_clusters == 1, px
        x, y, xe, ye = (np.float32(float(v)) for v in want[:4])
        assert (o.ht_x[0], o.ht_y[0]) == (x, y), px
        assert (o.ht_xerr[0], o.ht_yerr[0]) == (xe, ye), px
        rmin, rmax, cmin, cmax, flags = (int(v) for v in want[4:9])
        assert int(o.ht_rows[0]) == rmin | rmax << 16 and int(o.ht_cols[0]) == cmin | cmax << 16, px
        assert int(o.ht_flags[0]) == flags, px


def test_closed_forms_strip_translation_and_permutation():
    # a strip of L equal-adc pixels along col from c0 in row r: y = (c0 + (L-1)/2 + 0.5 - 208) * 150, x = (r + 0.5 - 80) * 100
    for L, c0, r in ((2, 1, 1), (7, 100, 37), (100, 300, 80), (33, 5, 158)):
        o = _run([(r, c0 + i, 60) for i in range(L)][::-1])
        assert o.n_clusters == 1
        assert o.ht_y[0] == np.float32((c0 + (L - 1) / 2 + 0.5 - 208) * 150.0) and o.ht_x[0] == np.float32((r + 0.5 - 80) * 100.0)
        assert int(o.ht_cols[0]) == c0 | (c0 + L - 1) << 16 and int(o.ht_rows[0]) == r | r << 16 and int(o.ht_flags[0]) == 0
        assert o.ht_yerr[0] == np.float32(150.0 * 0.28867513459481287 * 0.5)
    # translation by (dr, dc): x moves by exactly 100 dr, y by 150 dc (all values exact in binary32 here); the box moves along
    base = [(10, 20, 50), (11, 21, 30), (11, 22, 100)]
    o0 = _run(base)
    o1 = _run([(r + 64, c + 128, a) for r, c, a in base])
    assert np.float64(o1.ht_x[0]) - np.float64(o0.ht_x[0]) == pytest.approx(6400.0, abs=1e-3)
    assert np.float64(o1.ht_y[0]) - np.float64(o0.ht_y[0]) == pytest.approx(19200.0, abs=4e-3)
    assert int(o1.ht_rows[0]) == int(o0.ht_rows[0]) + (64 | 64 << 16) and int(o1.ht_cols[0]) == int(o0.ht_cols[0]) + (128 | 128 << 16)
    # mirror image about the module centre: (r, c) -> (159 - r, 415 - c) flips the signs
    om = _run([(159 - r, 415 - c, a) for r, c, a in base])
    assert om.ht_x[0] == -o0.ht_x[0] and om.ht_y[0] == -o0.ht_y[0]
    # the order of the words does not matter
    op = _run(base[::-1])
    for f in ("ht_x", "ht_y", "ht_xerr", "ht_yerr", "ht_rows", "ht_cols", "ht_flags"):
        assert np.array_equal(getattr(op, f), getattr(o0, f)), f
    # other pitches scale linearly
    ev = wl.event_from_pixels([(0, r, c, a) for r, c, a in base], 1)
    cal = wl.flat_calib(1)
    o2 = oracle.run(ev.words, ev.adc, 1, cal.gain, cal.pedestal, pitch_row_um=200.0, pitch_col_um=75.0)
    assert o2.ht_x[0] == np.float32(2.0 * np.float64(o0.ht_x[0])) and o2.ht_xerr[0] == np.float32(2.0) * o0.ht_xerr[0]
    assert np.float64(o2.ht_y[0]) == pytest.approx(np.float64(o0.ht_y[0]) / 2, rel=1e-7)


def test_only_kept_clusters_get_hits_and_duplicates_count():
    # cluster below the 4000 e threshold has no hit; a sub-threshold pixel is not part of any box (A11)
    o = _run([(3, 3, 13), (3, 4, 13), (9, 9, 60), (9, 10, 12)])
    assert o.n_clusters_all == 2 and o.n_clusters == 1 and o.ht_x.shape == (1,)
    assert int(o.ht_rows[0]) == 9 | 9 << 16 and int(o.ht_cols[0]) == 9 | 9 << 16
    # two digis on one pixel (A6) both weigh in: (5,5) twice with adc 50 and one (5,6) with adc 100 -> colC 5.5
    o = _run([(5, 5, 50), (5, 6, 100), (5, 5, 50)])
    assert o.n_clusters == 1 and o.cl_size[0] == 3
    assert o.ht_y[0] == np.float32((5.5 + 0.5 - 208) * 150.0) and int(o.ht_cols[0]) == 5 | 6 << 16
    # no clusters at all
    ev = wl.event_from_pixels([], 2)
    cal = wl.flat_calib(2)
    o = oracle.run(ev.words, ev.adc, 2, cal.gain, cal.pedestal)
    assert o.n_clusters == 0 and o.ht_x.shape == (0,) and o.ht_flags.shape == (0,)


@pytest.mark.parametrize("config,event,over", [(0, 0, {}), (1, 0, {}), (3, 1, dict(n_modules=300)),
                                               (4, 0, dict(n_modules=4, fill_pixels=2500))])
def test_hits_against_numpy_and_scipy(config, event, over):
    """Bounding boxes against numpy minimum/maximum reductions over the cluster numbers, positions against
    scipy.ndimage.center_of_mass on a dense float64 charge image of each module, flags against the boxes."""
    ev = wl.make_event(config, event, **over)
    cal = wl.make_calib(config, n_modules=ev.n_modules)
    o = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
    N = o.n_clusters
    assert N > 0 and all(getattr(o, f).shape == (N,) for f in ("ht_x", "ht_y", "ht_xerr", "ht_yerr", "ht_rows", "ht_cols", "ht_flags"))
    sel = o.clus >= 0
    k = o.clus[sel]
    for arr, field in ((o.row, "ht_rows"), (o.col, "ht_cols")):
        lo = np.full(N, 1 << 20, np.int64); hi = np.full(N, -1, np.int64)
        np.minimum.at(lo, k, arr[sel].astype(np.int64)); np.maximum.at(hi, k, arr[sel].astype(np.int64))
        assert np.array_equal(getattr(o, field), (lo | hi << 16).astype(np.uint32)), field
    rmin, rmax = o.ht_rows & 0xFFFF, o.ht_rows >> 16
    cmin, cmax = o.ht_cols & 0xFFFF, o.ht_cols >> 16
    assert np.array_equal(o.ht_flags & 1, ((rmin == 0) | (rmax == R - 1)).astype(np.uint16))
    assert np.array_equal(o.ht_flags >> 1, ((cmin == 0) | (cmax == C - 1)).astype(np.uint16))
    # interior boxes with span >= 2 have half the single-pixel error, span 1 the full one, border boxes span times it
    one = np.float32(100.0 * 0.28867513459481287)
    assert set(np.unique(o.ht_xerr[(o.ht_flags & 1) == 0])) <= {one, np.float32(100.0 * 0.28867513459481287 * 0.5)}
    assert np.all(o.ht_xerr[(o.ht_flags & 1) == 0][(rmax - rmin)[(o.ht_flags & 1) == 0] == 0] == one)
    # positions: scipy centre of mass per module (float64 image; duplicate-free workloads)
    checked = 0
    for m in range(min(ev.n_modules, 40)):
        lo, hi = int(o.mod_digi_start[m]), int(o.mod_digi_start[m + 1])
        ks = np.unique(o.clus[lo:hi][o.clus[lo:hi] >= 0])
        if ks.size == 0:
            continue
        img = np.zeros((R, C)); lab = np.zeros((R, C), np.int64)
        d = np.arange(lo, hi)[o.clus[lo:hi] >= 0]
        img[o.row[d], o.col[d]] = o.charge[d].astype(np.float64)
        lab[o.row[d], o.col[d]] = o.clus[d] + 1
        com = np.array(ndi.center_of_mass(img, lab, ks + 1))
        assert np.allclose(o.ht_x[ks], (com[:, 0] + 0.5 - 80.0) * 100.0, rtol=0, atol=2e-3)
        assert np.allclose(o.ht_y[ks], (com[:, 1] + 0.5 - 208.0) * 150.0, rtol=0, atol=4e-3)
        checked += ks.size
    assert checked > 0
