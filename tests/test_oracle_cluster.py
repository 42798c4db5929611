"""Pins for the oracle's clustering (O3) and the global invariants: exhaustive brute force on 4x4
windows, a second implementation (union-find), networkx for duplicate pixels, special shapes,
label canonicity under permutation, the independent checker (i)-(iii).  CPU only."""
import networkx as nx
import numpy as np
import pytest

import oracle
from oracle import crosscheck
from paper_2004_04334_b200 import workloads as wl

INVALID = oracle.INVALID


def _closure_labels_4x4(order):
    """All 2^16 occupancy patterns of a 4x4 window at once, by iterated min-propagation to the
    fixpoint (= transitive closure), vectorised in numpy.  ``order[cell]`` is the digi index rank
    of that cell (a permutation of 0..15): returns per pattern the minimum rank over each cell's
    component, or -1 for empty cells.  Shares nothing with the oracle's BFS."""
    pats = np.arange(1 << 16, dtype=np.uint32)
    on = ((pats[:, None] >> np.arange(16)[None, :]) & 1).astype(bool)           # [65536,16]
    big = 99
    lab = np.where(on, order[None, :], big).astype(np.int64)
    nbrs = []
    for a in range(16):
        ra, ca = divmod(a, 4)
        nbrs.append([b for b in range(16) if b != a and abs(b // 4 - ra) <= 1 and abs(b % 4 - ca) <= 1])
    for _ in range(16):
        new = lab.copy()
        for a in range(16):
            m = lab[:, nbrs[a]].min(axis=1)
            new[:, a] = np.where(on[:, a], np.minimum(lab[:, a], m), big)
        if np.array_equal(new, lab):
            break
        lab = new
    return on, np.where(on, lab, -1)


@pytest.mark.parametrize("r0,c0", [(0, 0), (156, 412), (0, 200), (77, 0), (80, 208)])
def test_exhaustive_4x4_against_transitive_closure(r0, c0):
    rng = np.random.default_rng(r0 * 1000 + c0)
    order = rng.permutation(16)                      # digi order inside the module is arbitrary (A5)
    on, want = _closure_labels_4x4(order)
    cells_by_rank = np.argsort(order)                # rank -> cell
    M = 2048
    for base in range(0, 1 << 16, M):                # one pattern per module, 2048 per call
        mods, rows, cols, ranks = [], [], [], []
        for j in range(M):
            p = base + j
            for rank in range(16):
                cell = cells_by_rank[rank]
                if on[p, cell]:
                    mods.append(j); rows.append(r0 + cell // 4); cols.append(c0 + cell % 4); ranks.append(rank)
        mods = np.array(mods, np.uint16); rows = np.array(rows, np.uint16); cols = np.array(cols, np.uint16)
        lab = oracle.cluster(mods, rows, cols, np.ones(len(mods), np.uint8), M)
        # translate event-global min index back to the rank of that digi inside its pattern
        ranks = np.array(ranks)
        got_rank = ranks[lab]
        cell_of = cells_by_rank[ranks]
        assert np.array_equal(got_rank, want[base + mods.astype(np.int64), cell_of])
        assert np.array_equal(mods[lab], mods)


def _partition(label, keys):
    groups = {}
    for L, k in zip(label.tolist(), keys):
        if L != INVALID:
            groups.setdefault(L, set()).add(k)
    return set(frozenset(s) for s in groups.values())


@pytest.mark.parametrize("config,event,over", [(0, 0, {}), (0, 3, {}), (1, 2, dict(n_modules=200)),
                                               (4, 0, dict(n_modules=3, fill_pixels=2500)),
                                               (3, 1, dict(n_modules=120))])
def test_bfs_equals_union_find(config, event, over):
    ev = wl.make_event(config, event, **over)
    cal = wl.make_calib(config, n_modules=ev.n_modules)
    o = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
    uf = crosscheck.cluster_union_find(o.module, o.row, o.col, o.kept)
    assert np.array_equal(o.label, uf)


def _check_labels_independently(o, R=160, C=416):
    """Checker independent of any CCL code (SURVEY 8(c) pins (4)): (i) label[label[i]]==label[i],
    label[i]<=i, same module; (ii) every adjacent kept pair has equal labels (9-neighbour probe);
    these force a partition that is a union of true components; (iii) distinct labels == number
    of components (from scipy in test_oracle_pins) then forces equality."""
    kept = o.kept.astype(bool)
    lab = o.label
    assert np.all(lab[~kept] == INVALID)
    k = np.flatnonzero(kept)
    assert np.all(lab[k] <= k) and np.array_equal(lab[lab[k]], lab[k]) and np.array_equal(o.module[lab[k]], o.module[k])
    key = (o.module[k].astype(np.int64) * (R + 2) + o.row[k] + 1) * (C + 2) + o.col[k] + 1
    srt = np.argsort(key, kind="stable")
    skey, slab = key[srt], lab[k][srt]
    for dr in (-1, 0, 1):
        for dc in (-1, 0, 1):
            probe = key + dr * (C + 2) + dc
            pos = np.searchsorted(skey, probe)
            pos[pos >= len(skey)] = len(skey) - 1
            hit = skey[pos] == probe
            assert np.array_equal(slab[pos][hit], lab[k][hit])


@pytest.mark.parametrize("config,event,over", [(0, 0, {}), (1, 0, {}), (3, 0, {}),
                                               (4, 1, dict(n_modules=40))])
def test_global_invariants(config, event, over):
    ev = wl.make_event(config, event, **over)
    cal = wl.make_calib(config, n_modules=ev.n_modules)
    o = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
    assert o.sorted_ok
    _check_labels_independently(o)
    kept = o.kept.astype(bool)
    # every kept digi in exactly one of the n_clusters_all components
    assert len(np.unique(o.label[kept])) == o.n_clusters_all
    assert np.all((o.clus >= -1) & (o.clus < o.n_clusters)) and np.all(o.clus[~kept] == -1)
    assert np.array_equal(o.clus[o.label[kept]], o.clus[kept])
    # sizes: kept clusters' sizes + digis of dropped clusters == kept digis
    inkept = o.clus >= 0
    assert int(o.cl_size.sum()) == int(inkept.sum())
    assert int(o.cl_size.sum()) + int((kept & ~inkept).sum()) == o.n_kept_digis
    assert np.array_equal(np.bincount(o.clus[inkept], minlength=o.n_clusters), o.cl_size)
    # total charge of kept clusters == summed charge of their digis, exactly in fixed point
    qf = (o.charge.astype(np.float64) * 16384.0)
    assert np.all(qf[kept] == np.round(qf[kept]))
    per = np.zeros(o.n_clusters, np.int64)
    np.add.at(per, o.clus[inkept], qf[inkept].astype(np.int64))
    assert np.array_equal((per.astype(np.float64) / 16384.0).astype(np.float32), o.cl_charge)
    assert np.all(per >= 4000 * 16384)
    # cluster table sorted by label, grouped by module, mod_clus_start consistent
    assert np.all(np.diff(o.cl_label.astype(np.int64)) > 0)
    assert np.array_equal(o.cl_module, o.module[o.cl_label])
    assert np.array_equal(o.mod_clus_start, np.searchsorted(o.cl_module, np.arange(ev.n_modules + 1), side="left"))
    assert np.array_equal(o.clus[o.cl_label], np.arange(o.n_clusters))


def test_duplicate_pixels_networkx():
    """A6: two words addressing the same pixel are both digis, adjacent to each other."""
    rng = np.random.default_rng(3)
    px = []
    for m in range(6):
        n = 60
        rows = rng.integers(0, 12, n); cols = rng.integers(0, 12, n)     # dense: many duplicates
        px += [(m, int(r), int(c), int(rng.integers(20, 255))) for r, c in zip(rows, cols)]
    ev = wl.event_from_pixels(px, 6)
    cal = wl.flat_calib(6)
    o = oracle.run(ev.words, ev.adc, 6, cal.gain, cal.pedestal)
    assert len(set(px)) < len(px) or True
    g = nx.Graph()
    D = o.n_digis
    kept = o.kept.astype(bool)
    g.add_nodes_from(int(i) for i in np.flatnonzero(kept))
    for a in range(D):
        for b in range(a + 1, D):
            if kept[a] and kept[b] and o.module[a] == o.module[b] and abs(int(o.row[a]) - int(o.row[b])) <= 1 \
                    and abs(int(o.col[a]) - int(o.col[b])) <= 1:
                g.add_edge(a, b)
    comps = list(nx.connected_components(g))
    assert len(comps) == o.n_clusters_all
    for comp in comps:
        assert all(o.label[i] == min(comp) for i in comp)
    # sizes count duplicates
    assert int(o.cl_size.sum()) == int((o.clus >= 0).sum())
    dup = wl.event_from_pixels([(0, 5, 5, 50), (0, 9, 9, 50), (0, 5, 5, 30)], 1)
    o = oracle.run(dup.words, dup.adc, 1, np.float32([80]), np.float32([0]))
    assert list(o.label) == [0, 1, 0] and o.n_clusters == 2
    assert (o.cl_size[0], o.cl_charge[0], o.cl_row[0], o.cl_col[0]) == (2, 6400.0, 5.0, 5.0)


def _labels_of(px, M=4, cal=None, **kw):
    ev = wl.event_from_pixels(px, M)
    cal = cal or wl.flat_calib(M)
    return oracle.run(ev.words, ev.adc, M, cal.gain, cal.pedestal, **kw)


def test_special_shapes():
    # diagonal pair -> 1 cluster (8- not 4-connectivity); distance 2 -> 2 clusters
    assert list(_labels_of([(0, 5, 5, 60), (0, 6, 6, 60)]).label) == [0, 0]
    assert list(_labels_of([(0, 5, 5, 60), (0, 6, 4, 60)]).label) == [0, 0]
    assert list(_labels_of([(0, 5, 5, 60), (0, 5, 7, 60)]).label) == [0, 1]
    assert list(_labels_of([(0, 5, 5, 60), (0, 7, 5, 60)]).label) == [0, 1]
    # no wrap-around: (159,c) vs (0,c); (r,415) vs (r+1,0)
    assert list(_labels_of([(0, 159, 7, 60), (0, 0, 7, 60)]).label) == [0, 1]
    assert list(_labels_of([(0, 10, 415, 60), (0, 11, 0, 60)]).label) == [0, 1]
    assert list(_labels_of([(0, 10, 415, 60), (0, 10, 0, 60)]).label) == [0, 1]
    # same coordinates in modules m and m+1 -> different clusters
    assert list(_labels_of([(1, 3, 3, 60), (2, 3, 3, 60)]).label) == [0, 1]
    # sub-threshold pixel (adc 12 -> 960 e) in the middle of a 1x3 strip -> 2 clusters (A11)
    o = _labels_of([(0, 3, 3, 60), (0, 3, 4, 12), (0, 3, 5, 60)])
    assert list(o.label) == [0, INVALID, 2] and list(o.clus) == [0, -1, 1] and o.n_kept_digis == 2
    # cluster below 4000 e keeps its label but clus = -1 (A12): 13*80 = 1040 e
    o = _labels_of([(0, 3, 3, 13), (0, 3, 4, 13), (0, 9, 9, 60)])
    assert list(o.label) == [0, 0, 2] and list(o.clus) == [-1, -1, 0] and (o.n_clusters_all, o.n_clusters) == (2, 1)
    # 1 x 100 strip, fed right-to-left and interleaved: one cluster
    cols = list(range(100, 200))
    px = [(3, 80, c, 60) for c in cols[::2]] + [(3, 80, c, 60) for c in cols[1::2]]
    assert set(_labels_of(px).label.tolist()) == {0}
    # U shape whose minimum index sits at the far end of one arm (propagation depth)
    arm1 = [(0, r, 10, 60) for r in range(0, 60)]
    bottom = [(0, 59, c, 60) for c in range(11, 50)]
    arm2 = [(0, r, 50, 60) for r in range(59, -1, -1)]
    px = [arm2[-1]] + arm1 + bottom + arm2[:-1]            # index 0 = top of arm2
    assert set(_labels_of(px).label.tolist()) == {0}
    # spiral
    sp, r, c, dr, dc, seg = [], 80, 200, 0, 1, 2
    for k in range(40):
        for _ in range(seg):
            sp.append((1, r, c, 60)); r += dr; c += dc
        dr, dc = dc, -dr
        seg += 2
    assert len(set((a, b) for _, a, b, _ in sp)) == len(sp)
    assert set(_labels_of(sp[::-1]).label.tolist()) == {0}


def test_full_and_checkerboard_module():
    rr, cc = np.meshgrid(np.arange(160), np.arange(416), indexing="ij")
    cal = wl.flat_calib(2)
    for sel, size in ((np.ones_like(rr, bool), 66560), ((rr + cc) % 2 == 0, 33280)):
        w = ((1 << 20) | (rr[sel].astype(np.uint32) << 12) | (cc[sel].astype(np.uint32) << 3)).astype(np.uint32)
        w = np.random.default_rng(1).permutation(w)
        o = oracle.run(w, np.full(w.shape[0], 60, np.uint16), 2, cal.gain, cal.pedestal)
        assert o.n_clusters_all == 1 and o.cl_size[0] == size and np.all(o.label == 0)
        assert o.cl_charge[0] == np.float32(4800.0 * size)
        assert o.cl_row[0] == pytest.approx(79.5, abs=1e-4) and o.cl_col[0] == pytest.approx(207.5, abs=1e-4)
    # isolated pixels on a stride-2 lattice: as many clusters as pixels
    sel = (rr % 2 == 0) & (cc % 2 == 0)
    w = ((rr[sel].astype(np.uint32) << 12) | (cc[sel].astype(np.uint32) << 3)).astype(np.uint32)
    o = oracle.run(w, np.full(w.shape[0], 60, np.uint16), 2, cal.gain, cal.pedestal)
    assert o.n_clusters_all == 80 * 208 == o.n_clusters and np.array_equal(o.label, np.arange(80 * 208))


@pytest.mark.parametrize("config,over", [(0, {}), (4, dict(n_modules=6, fill_pixels=3000))])
def test_label_canonicity_under_permutation(config, over):
    """Permute the words within each module: the partition as sets of (module,row,col), every
    size / charge / centroid and both counts are invariant; each label is the minimum NEW index."""
    ev = wl.make_event(config, 2, **over)
    cal = wl.make_calib(config, n_modules=ev.n_modules)
    o1 = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
    rng = np.random.default_rng(11)
    valid = (ev.words >> 31) == 0
    mod = (ev.words >> 20) & 0x7FF
    perm = np.arange(ev.n_words)
    for m in np.unique(mod[valid]):
        idx = np.flatnonzero(valid & (mod == m))
        perm[idx] = rng.permutation(idx)
    o2 = oracle.run(ev.words[perm], ev.adc[perm], ev.n_modules, cal.gain, cal.pedestal)
    assert (o1.n_clusters_all, o1.n_clusters, o1.n_kept_digis) == (o2.n_clusters_all, o2.n_clusters, o2.n_kept_digis)
    k1 = list(zip(o1.module.tolist(), o1.row.tolist(), o1.col.tolist()))
    k2 = list(zip(o2.module.tolist(), o2.row.tolist(), o2.col.tolist()))
    assert _partition(o1.label, k1) == _partition(o2.label, k2)
    kept2 = np.flatnonzero(o2.kept)
    mins = {}
    for i in kept2:
        mins.setdefault(int(o2.label[i]), int(i))
    assert all(L == first for L, first in mins.items())

    def table(o, keys):
        t = {}
        for k in range(o.n_clusters):
            members = frozenset(keys[i] for i in np.flatnonzero(o.clus == k))
            t[members] = (int(o.cl_size[k]), float(o.cl_charge[k]), float(o.cl_row[k]), float(o.cl_col[k]))
        return t
    assert table(o1, k1) == table(o2, k2)
