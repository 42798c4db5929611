"""Pins for the oracle's decode / calibrate / reduce steps against things other than itself:
hand-worked values (tests/golden/worked_values.txt), exhaustive codec round trip, the float64
single-rounding identity, closed forms, scipy.ndimage.  CPU only."""
import os

import numpy as np
import pytest
import scipy.ndimage as ndi

import oracle
from paper_2004_04334_b200 import workloads as wl


def _golden(golden_dir):
    rows = []
    with open(os.path.join(golden_dir, "worked_values.txt")) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


def test_worked_words(golden_dir):
    for r in _golden(golden_dir):
        if r[0] == "word":
            m, row, col, w = int(r[1]), int(r[2]), int(r[3]), int(r[4], 16)
            d = oracle.decode(np.array([w], np.uint32), np.array([77], np.uint16), 2048, 256, 512)
            assert (d["module"][0], d["row"][0], d["col"][0], d["adc"][0], d["word_idx"][0]) == (m, row, col, 77, 0)
            assert len(d["err_word"]) == 0
            assert wl.encode_word(m, row, col) == w          # generator's encoder agrees with the hand value
        elif r[0] == "lowbits":
            w, m, row, col = int(r[1], 16), int(r[2]), int(r[3]), int(r[4])
            d = oracle.decode(np.array([w], np.uint32), np.array([5], np.uint16), 64)
            assert (d["module"][0], d["row"][0], d["col"][0]) == (m, row, col)
        elif r[0] == "errword":
            w = int(r[1], 16)
            d = oracle.decode(np.array([1 << 20, w, 2 << 20], np.uint32), np.array([1, 2, 3], np.uint16), 64)
            assert list(d["err_word"]) == [w] and list(d["err_idx"]) == [1]
            assert list(d["word_idx"]) == [0, 2] and list(d["adc"]) == [1, 3]


def test_out_of_range_fields_are_errors():
    # A3: unflagged word with module >= M, row >= R or col >= C goes to the error list
    M, R, C = 64, 160, 416
    ws = [wl.encode_word(64, 0, 0), wl.encode_word(0, 160, 0), wl.encode_word(0, 0, 416),
          wl.encode_word(63, 159, 415), wl.encode_word(2047, 255, 511)]
    d = oracle.decode(np.array(ws, np.uint32), np.arange(5, dtype=np.uint16), M, R, C)
    assert list(d["err_idx"]) == [0, 1, 2, 4]
    assert list(d["word_idx"]) == [3] and d["module"][0] == 63 and d["row"][0] == 159 and d["col"][0] == 415


def test_codec_exhaustive_round_trip():
    """decode(encode(m,r,c)) == (m,r,c) over ALL 2048 x 256 x 512 field values (2^28 words), and
    encode(decode(w)) == w & 0x7FFFFFF8; brute force, chunked."""
    rows = np.arange(256, dtype=np.uint32)
    cols = np.arange(512, dtype=np.uint32)
    rc = ((rows[:, None] << 12) | (cols[None, :] << 3)).reshape(-1)       # 2^17 (row,col) pairs
    step = 16                                                              # modules per chunk
    for m0 in range(0, 2048, step):
        ms = np.arange(m0, m0 + step, dtype=np.uint32)
        words = ((ms[:, None] << 20) | rc[None, :]).reshape(-1)
        low = (np.arange(words.shape[0], dtype=np.uint32) * 2654435761 >> 7) & 7   # arbitrary low bits (A1)
        adc = np.zeros(words.shape[0], np.uint16)
        d = oracle.decode(words | low, adc, 2048, 256, 512)
        assert len(d["module"]) == words.shape[0] and len(d["err_idx"]) == 0
        assert np.array_equal(d["module"], np.repeat(ms, rc.shape[0]).astype(np.uint16))
        assert np.array_equal(d["row"], np.tile(np.repeat(rows, 512), step).astype(np.uint16))
        assert np.array_equal(d["col"], np.tile(np.tile(cols, 256), step).astype(np.uint16))
        re = (d["module"].astype(np.uint32) << 20) | (d["row"].astype(np.uint32) << 12) | (d["col"].astype(np.uint32) << 3)
        assert np.array_equal(re, (words | low) & 0x7FFFFFF8)


def test_compaction_is_lossless_partition():
    ev = wl.make_event(0, 0)
    d = oracle.decode(ev.words, ev.adc, ev.n_modules)
    D, E, W = len(d["word_idx"]), len(d["err_idx"]), ev.n_words
    assert D + E == W and E > 0
    assert np.all(np.diff(d["word_idx"].astype(np.int64)) > 0) and np.all(np.diff(d["err_idx"].astype(np.int64)) > 0)
    assert np.array_equal(np.sort(np.concatenate([d["word_idx"], d["err_idx"]])), np.arange(W))
    back = np.zeros(W, np.uint32)
    back[d["word_idx"]] = (d["module"].astype(np.uint32) << 20) | (d["row"].astype(np.uint32) << 12) | (d["col"].astype(np.uint32) << 3)
    back[d["err_idx"]] = d["err_word"]
    mask = np.where(ev.words >> 31, 0xFFFFFFFF, 0x7FFFFFF8).astype(np.uint32)
    assert np.array_equal(back, ev.words & mask)
    assert np.array_equal(d["adc"], ev.adc[d["word_idx"]])
    # mod_digi_start = number of digis with module < m
    mds = np.searchsorted(d["module"], np.arange(ev.n_modules + 1), side="left")
    assert d["sorted_ok"] and np.array_equal(d["mod_digi_start"], mds)


def test_sorted_ok_and_mod_digi_start_for_unsorted_input():
    ev = wl.event_from_pixels([(2, 1, 1, 50), (0, 1, 1, 50), 0x80000000 | (5 << 20), (2, 3, 3, 50)], 4)
    d = oracle.decode(ev.words, ev.adc, 4)
    assert not d["sorted_ok"]
    assert list(d["mod_digi_start"]) == [0, 1, 1, 3, 3]          # counts of module < m, any order


def test_degenerate_events():
    # A20: W = 0 and all-error events are legal
    cal = wl.flat_calib(4)
    r = oracle.run(np.zeros(0, np.uint32), np.zeros(0, np.uint16), 4, cal.gain, cal.pedestal)
    assert (r.n_digis, r.n_errors, r.n_clusters_all, r.n_clusters) == (0, 0, 0, 0)
    assert list(r.mod_digi_start) == [0] * 5 and list(r.mod_clus_start) == [0] * 5
    w = np.array([0x80000001, 0x80100002, 0xFFFFFFFF], np.uint32)
    r = oracle.run(w, np.zeros(3, np.uint16), 4, cal.gain, cal.pedestal)
    assert (r.n_digis, r.n_errors, r.n_clusters) == (0, 3, 0) and np.array_equal(r.err_word, w)


def test_worked_calibration(golden_dir):
    for r in _golden(golden_dir):
        if r[0] != "calib":
            continue
        g, p, adc, q, kept = float(r[1]), float(r[2]), int(r[3]), float(r[4]), int(r[5])
        charge, k = oracle.calibrate(np.array([adc], np.uint16), np.zeros(1, np.uint16),
                                     np.array([g], np.float32), np.array([p], np.float32), 1000.0)
        assert charge[0] == np.float32(q) and int(k[0]) == kept, r


def test_calibration_is_single_rounding_fma():
    """float32(float64(adc)*gain + ped) is the correctly-rounded FMA (the binary64 product of a
    16-bit integer and a binary32 is exact, and the binary64 add of a binary32 stays exact for
    these magnitudes), so it pins 'one rounding' without trusting any fmaf.  Also shows the
    two-rounding variant differs somewhere, i.e. the pin has teeth."""
    rng = np.random.default_rng(7)
    n = 1 << 18
    adc = rng.integers(0, 4096, n).astype(np.uint16)
    gain = rng.normal(80, 5, 64).astype(np.float32)
    ped = rng.normal(0, 200, 64).astype(np.float32)
    mod = rng.integers(0, 64, n).astype(np.uint16)
    charge, kept = oracle.calibrate(adc, mod, gain, ped, 1000.0)
    exact = adc.astype(np.float64) * gain[mod].astype(np.float64) + ped[mod].astype(np.float64)
    assert np.array_equal(charge, exact.astype(np.float32))
    assert np.array_equal(kept.astype(bool), exact.astype(np.float32) >= np.float32(1000.0))
    two = (adc.astype(np.float32) * gain[mod]) + ped[mod]             # product rounded first
    assert np.any(two != charge)


def test_worked_reduce_and_cluster_threshold(golden_dir):
    for r in _golden(golden_dir):
        if r[0] == "reduce2":
            m = int(r[1])
            px = [(m, int(r[2]), int(r[3]), int(r[4])), (m, int(r[5]), int(r[6]), int(r[7]))]
            ev = wl.event_from_pixels(px, 8)
            cal = wl.flat_calib(8, 80.0, 0.0)
            o = oracle.run(ev.words, ev.adc, 8, cal.gain, cal.pedestal)
            assert o.n_clusters_all == 1 and o.n_clusters == 1
            assert int(o.cl_size[0]) == int(r[10]) and o.cl_charge[0] == np.float32(float(r[12]))
            assert o.cl_row[0] == np.float32(float(r[14])) and o.cl_col[0] == np.float32(float(r[16]))
            assert o.cl_module[0] == m and o.cl_label[0] == 0 and list(o.clus) == [0, 0] and list(o.label) == [0, 0]
            assert list(o.mod_clus_start) == [0] * (m + 1) + [1] * (8 - m)
        elif r[0] == "clusthr":
            g, adc, kept = float(r[1]), int(r[2]), int(r[3])
            ev = wl.event_from_pixels([(0, 5, 5, adc)], 2)
            cal = wl.flat_calib(2, g, 0.0)
            o = oracle.run(ev.words, ev.adc, 2, cal.gain, cal.pedestal)
            assert o.n_clusters_all == 1 and o.n_clusters == kept
            assert list(o.clus) == ([0] if kept else [-1]) and list(o.label) == [0]


def test_single_pixel_and_strip_closed_forms():
    cal = wl.flat_calib(4, 80.0, 0.0)
    # single pixel: centroid == (row, col) exactly, charge == q (A13)
    ev = wl.event_from_pixels([(1, 159, 415, 200)], 4)
    o = oracle.run(ev.words, ev.adc, 4, cal.gain, cal.pedestal)
    assert (o.cl_row[0], o.cl_col[0], o.cl_charge[0], o.cl_size[0]) == (159.0, 415.0, 16000.0, 1)
    # horizontal strip of L equal-adc pixels from col c0: colC = c0 + (L-1)/2, rowC = row
    for L, c0, row in ((2, 0, 0), (7, 100, 37), (100, 316, 159), (33, 5, 80)):
        px = [(2, row, c0 + i, 60) for i in range(L)]
        ev = wl.event_from_pixels(px[::-1], 4)                      # reversed order: label still index 0
        o = oracle.run(ev.words, ev.adc, 4, cal.gain, cal.pedestal)
        assert o.n_clusters == 1 and o.cl_size[0] == L and o.cl_label[0] == 0
        assert o.cl_row[0] == np.float32(row) and o.cl_col[0] == np.float32(c0 + (L - 1) / 2)
        assert o.cl_charge[0] == np.float32(4800.0 * L)
    # translation by (dr, dc) shifts the centroid by exactly that (values exact in binary32 here)
    base = [(0, 10, 20, 50), (0, 11, 21, 30), (0, 11, 22, 100)]
    o0 = oracle.run(*_ev(base), 4, cal.gain, cal.pedestal)
    o1 = oracle.run(*_ev([(m, r + 64, c + 128, a) for m, r, c, a in base]), 4, cal.gain, cal.pedestal)
    d0 = (80 * 50 * 10 + 80 * 30 * 11 + 80 * 100 * 11) / (80 * 180)
    assert o0.cl_row[0] == np.float32(d0) and o1.cl_row[0] == np.float32(d0 + 64)
    assert np.float64(o1.cl_col[0]) - np.float64(o0.cl_col[0]) == pytest.approx(128, abs=2e-5)


def _ev(px):
    ev = wl.event_from_pixels(px, 4)
    return ev.words, ev.adc


@pytest.mark.parametrize("config,event", [(0, 0), (1, 0), (1, 5)])
def test_reduce_against_scipy(config, event):
    """scipy.ndimage.sum_labels / center_of_mass in float64 on the oracle's own partition, and
    scipy.ndimage.label for the partition itself (module by module)."""
    ev = wl.make_event(config, event)
    cal = wl.make_calib(config)
    o = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
    n_all = 0
    k = 0
    for m in range(ev.n_modules):
        lo, hi = int(o.mod_digi_start[m]), int(o.mod_digi_start[m + 1])
        if lo == hi:
            continue
        sel = slice(lo, hi)
        kept = o.kept[sel].astype(bool)
        grid_q = np.zeros((ev.n_rows, ev.n_cols))
        grid_on = np.zeros((ev.n_rows, ev.n_cols), bool)
        grid_q[o.row[sel][kept], o.col[sel][kept]] = o.charge[sel][kept].astype(np.float64)
        grid_on[o.row[sel][kept], o.col[sel][kept]] = True
        lab, n = ndi.label(grid_on, structure=np.ones((3, 3)))
        n_all += n
        if n == 0:
            continue
        # same partition: scipy label -> oracle label is a bijection
        sl = lab[o.row[sel][kept], o.col[sel][kept]]
        ol = o.label[sel][kept]
        pairs = set(zip(sl.tolist(), ol.tolist()))
        assert len(pairs) == n == len(set(ol.tolist()))
        # every oracle label is the minimum digi index of its set
        for s_id, o_id in pairs:
            assert o_id == lo + np.flatnonzero(kept)[sl == s_id].min()
        idx = np.arange(1, n + 1)
        S = ndi.sum_labels(grid_q, lab, idx)
        com = np.array(ndi.center_of_mass(grid_q, lab, idx)).reshape(n, 2)
        by_label = {o_id: s_id for s_id, o_id in pairs}
        for L in sorted(by_label):
            s_id = by_label[L]
            if S[s_id - 1] >= 4000.0:
                assert o.cl_label[k] == L and o.cl_module[k] == m
                assert o.cl_charge[k] == pytest.approx(S[s_id - 1], rel=2e-7)
                assert o.cl_row[k] == pytest.approx(com[s_id - 1, 0], abs=2e-5)
                assert o.cl_col[k] == pytest.approx(com[s_id - 1, 1], abs=4e-5)
                assert o.cl_size[k] == int((sl == s_id).sum())
                k += 1
    assert n_all == o.n_clusters_all and k == o.n_clusters


def test_exact_sum_claim():
    """A9: q*2^14 integral, int64 == int128, and fp64 forward/backward sums equal S*2^-14."""
    for config in (0, 1):
        ev = wl.make_event(config, 1)
        cal = wl.make_calib(config)
        o = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
        assert oracle.check_exact_sums(o.label, o.charge, o.col) == 0
    # and the reduce refuses a pixel threshold below 512 when a kept charge is not on the 2^-14 grid
    ev = wl.event_from_pixels([(0, 1, 1, 3)], 2)
    cal = wl.Calib(np.array([33.333332, 80], np.float32), np.array([0.0001, 0], np.float32), 50.0, 60.0)
    with pytest.raises(ArithmeticError):
        oracle.run(ev.words, ev.adc, 2, cal.gain, cal.pedestal, 50.0, 60.0)


def test_occupancy_against_numpy_and_worked_values():
    """po_occupancy (second consumer of the digis): a worked example and numpy bincount on generated events."""
    ev = wl.event_from_pixels([(0, 1, 1, 60), (0, 1, 2, 12), (2, 5, 5, 200), (2, 9, 9, 13), (2, 5, 6, 255)], 4)
    cal = wl.flat_calib(4, 80.0, 0.0)
    o = oracle.run(ev.words, ev.adc, 4, cal.gain, cal.pedestal)
    cnt, tot = oracle.occupancy(o.module, o.adc, o.kept, 4)        # adc 12 -> 960 e is below the pixel threshold
    assert list(cnt) == [1, 0, 3, 0] and list(tot) == [60, 0, 200 + 13 + 255, 0]
    for config in (0, 1):
        ev = wl.make_event(config, 3)
        cal = wl.make_calib(config)
        o = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
        cnt, tot = oracle.occupancy(o.module, o.adc, o.kept, ev.n_modules)
        k = o.kept.astype(bool)
        assert np.array_equal(cnt, np.bincount(o.module[k], minlength=ev.n_modules).astype(np.uint32))
        assert np.array_equal(tot, np.bincount(o.module[k], weights=o.adc[k].astype(np.float64), minlength=ev.n_modules).astype(np.uint32))
        assert int(cnt.sum()) == o.n_kept_digis
