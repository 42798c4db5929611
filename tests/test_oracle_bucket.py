"""Pins of the oracle's bucket step O0 (reading A31: words in arbitrary order are bucketed stably by module before the
decode).  The paper gives nothing for it: the pins are a worked example, a
library routine (numpy's stable argsort) and the properties that define a stable bucket sort."""
import numpy as np

import oracle
from paper_2004_04334_b200 import workloads as wl


def enc(m, r, c, low=0):
    return np.uint32((m << 20) | (r << 12) | (c << 3) | low)


def keys_of(words, M, R=160, C=416):
    w = words.astype(np.uint64)
    mod, row, col = (w >> 20) & 0x7FF, (w >> 12) & 0xFF, (w >> 3) & 0x1FF
    bad = ((w >> 31) != 0) | (mod >= M) | (row >= R) | (col >= C)
    return np.where(bad, M, mod).astype(np.int64)


def test_worked_example():
    # six words, M = 4: modules 2, 0, (error), 2, 1, 0  ->  module 0: inputs 1 and 5; module 1: input 4; module 2: inputs 0, 3;
    # the error word (input 2) goes last.  Written out by hand.
    words = np.array([enc(2, 5, 5), enc(0, 1, 1), np.uint32(0x80000001), enc(2, 6, 6), enc(1, 9, 9), enc(0, 2, 2)], np.uint32)
    adc = np.array([10, 11, 12, 13, 14, 15], np.uint16)
    ow, oa, orig = oracle.bucket(words, adc, 4)
    assert orig.tolist() == [1, 5, 4, 0, 3, 2]
    assert oa.tolist() == [11, 15, 14, 10, 13, 12]
    assert ow.tolist() == [int(words[i]) for i in [1, 5, 4, 0, 3, 2]]
    # a word whose fields are out of range is an error word (A3) and goes to the last bucket too
    words2 = np.array([enc(3, 200, 1), enc(1, 1, 1), enc(5, 1, 1), enc(0, 1, 500)], np.uint32)     # row 200 >= 160, module 5 >= 4, col 500 >= 416
    _, _, orig2 = oracle.bucket(words2, np.zeros(4, np.uint16), 4)
    assert orig2.tolist() == [1, 0, 2, 3]


def test_equals_numpys_stable_argsort_on_shuffled_events():
    rng = np.random.default_rng(31)
    for cfg, e in ((0, 0), (1, 2), (3, 1)):
        ev = wl.make_event(cfg, e)
        perm = rng.permutation(ev.n_words)
        words, adc = ev.words[perm], ev.adc[perm]
        ow, oa, orig = oracle.bucket(words, adc, ev.n_modules)
        want = np.argsort(keys_of(words, ev.n_modules), kind="stable")
        assert np.array_equal(orig, want.astype(np.uint32))
        assert np.array_equal(ow, words[want]) and np.array_equal(oa, adc[want])
        # a permutation of the input: nothing lost, nothing twice
        assert np.array_equal(np.sort(orig), np.arange(ev.n_words, dtype=np.uint32))


def test_grouped_input_keeps_its_digi_and_error_lists():
    """An event that already obeys A5 (modules non-decreasing, error words anywhere): bucketing only moves the error words
    to the end, so the unordered chain reproduces the ordered chain output for output, indices included."""
    cal = wl.make_calib(1)
    ev = wl.make_event(1, 5)
    a = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
    b = oracle.run_unordered(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
    assert a.sorted_ok and b.sorted_ok
    for f in ("module", "row", "col", "adc", "word_idx", "err_word", "err_idx", "mod_digi_start", "label", "clus",
              "cl_label", "cl_module", "cl_size", "mod_clus_start", "ht_rows", "ht_cols", "ht_flags"):
        assert np.array_equal(getattr(a, f), getattr(b, f)), f
    assert np.array_equal(a.charge.view(np.uint32), b.charge.view(np.uint32))
    assert np.array_equal(a.cl_charge.view(np.uint32), b.cl_charge.view(np.uint32))


def test_shuffled_input_gives_the_same_clusters_as_pixel_sets():
    """Any input order: the set of pixels of every cluster, its charge and centroid do not depend on the order of the words;
    the digi list is grouped by module with the input order inside a module; word indices point into the INPUT."""
    cal = wl.make_calib(0)
    ev = wl.make_event(0, 1)
    rng = np.random.default_rng(5)
    perm = rng.permutation(ev.n_words)
    a = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
    b = oracle.run_unordered(ev.words[perm], ev.adc[perm], ev.n_modules, cal.gain, cal.pedestal)
    assert b.sorted_ok and (b.n_digis, b.n_errors, b.n_clusters_all, b.n_clusters) == (a.n_digis, a.n_errors, a.n_clusters_all, a.n_clusters)
    assert np.all(np.diff(b.module.astype(np.int64)) >= 0)
    # word_idx points into the shuffled input: the word found there is the digi's word
    w = ev.words[perm][b.word_idx]
    assert np.array_equal((w >> 20) & 0x7FF, b.module) and np.array_equal((w >> 12) & 0xFF, b.row) and np.array_equal((w >> 3) & 0x1FF, b.col)
    assert np.array_equal(ev.adc[perm][b.word_idx], b.adc)
    # inside a module the digis keep their input order
    for m in range(ev.n_modules):
        s, t = b.mod_digi_start[m], b.mod_digi_start[m + 1]
        assert np.all(np.diff(b.word_idx[s:t].astype(np.int64)) > 0)
    assert np.all(np.diff(b.err_idx.astype(np.int64)) > 0) and np.array_equal(ev.words[perm][b.err_idx], b.err_word)

    def clusters(r):
        out = {}
        for k in range(r.n_clusters):
            members = np.nonzero(r.clus == k)[0]
            key = frozenset((int(r.module[d]), int(r.row[d]), int(r.col[d])) for d in members)
            out[key] = (r.cl_size[k], r.cl_charge[k].view(np.uint32), r.cl_row[k].view(np.uint32), r.cl_col[k].view(np.uint32))
        return out
    assert clusters(a) == clusters(b)
