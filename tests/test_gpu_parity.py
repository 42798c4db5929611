"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on the
same seeded inputs.  Bit-exact for every integer/index output; cluster charge within 1e-5
relative and centroids within 1e-4 pixel (BASELINE.json north_star; A14) — and in fact the exact
fixed-point reduce makes those bit-exact too, which is asserted as well."""
import time

import numpy as np
import pytest

import oracle
from paper_2004_04334_b200 import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def pr():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the product path has no CPU fallback")
    from paper_2004_04334_b200 import pixreco
    pixreco.lib()
    return pixreco


def to_dev(a):
    """numpy u32/u16 -> CUDA tensor with the same bytes (16-byte aligned by the torch allocator)."""
    if a.shape[0] == 0:
        return torch.empty(0, dtype=torch.int32 if a.dtype == np.uint32 else torch.int16, device="cuda")
    v = a.view(np.int32) if a.dtype == np.uint32 else a.view(np.int16)
    return torch.from_numpy(v.copy()).cuda()


def wait(slot, timeout=60.0):
    t0 = time.time()
    while slot.query() == 1:
        if time.time() - t0 > timeout:
            raise TimeoutError("event did not complete")
        time.sleep(0.0002)


INT_FIELDS = ["module", "row", "col", "adc", "word_idx", "err_word", "err_idx", "mod_digi_start", "label", "clus",
              "cl_label", "cl_module", "cl_size", "mod_clus_start", "ht_rows", "ht_cols", "ht_flags"]
HIT_FLOATS = ["ht_x", "ht_y", "ht_xerr", "ht_yerr"]


def compare(out, ref, getter, strict_float=True):
    assert (out.n_words, out.n_digis, out.n_errors, out.n_kept_digis, out.n_clusters_all, out.n_clusters) == \
        (ref.n_words, ref.n_digis, ref.n_errors, ref.n_kept_digis, ref.n_clusters_all, ref.n_clusters)
    assert out.status_bits == 0
    for f in INT_FIELDS:
        got = getter(f)
        if got is None:
            continue
        assert np.array_equal(got, getattr(ref, f)), f
    q = getter("charge")
    if q is not None:
        assert np.array_equal(q.view(np.uint32), ref.charge.view(np.uint32)), "charge bits (A7: single fmaf)"
    c = getter("cl_charge")
    if c is not None:
        assert np.all(np.abs(c - ref.cl_charge) <= 1e-5 * np.abs(ref.cl_charge))
        assert np.all(np.abs(getter("cl_row") - ref.cl_row) <= 1e-4) and np.all(np.abs(getter("cl_col") - ref.cl_col) <= 1e-4)
        if strict_float:
            for f in ("cl_charge", "cl_row", "cl_col"):
                assert np.array_equal(getter(f).view(np.uint32), getattr(ref, f).view(np.uint32)), f
    if getter("ht_x") is not None:
        # hits (A26-A30): positions within 1e-4 pixel = 0.01 / 0.015 um (BASELINE.json's centroid tolerance times the
        # pitch), errors within 1e-5 relative — and bit-equal, because both sides do the same binary64 operations
        assert np.all(np.abs(getter("ht_x") - ref.ht_x) <= 1e-2) and np.all(np.abs(getter("ht_y") - ref.ht_y) <= 1.5e-2)
        for f in ("ht_xerr", "ht_yerr"):
            assert np.all(np.abs(getter(f) - getattr(ref, f)) <= 1e-5 * getattr(ref, f)), f
        if strict_float:
            for f in HIT_FLOATS:
                assert np.array_equal(getter(f).view(np.uint32), getattr(ref, f).view(np.uint32)), f


def run_device(pr, ev, cal, **kw):
    """Device-resident input, device views copied back by the test."""
    with pr.PixReco(cal.gain, cal.pedestal, ev.n_rows, ev.n_cols, cal.pixel_threshold_e, cal.cluster_threshold_e, **kw) as p:
        slot = p.slot()
        w, a = to_dev(ev.words), to_dev(ev.adc)
        s = torch.cuda.Stream()
        slot.acquire(w, a, stream=s)
        wait(slot)
        code, out = slot.produce()
        assert code == 0
        got = {f: out.to_numpy(f) for f in pr.VIEW_SPEC}
        slot.release()
        return out, got


def oracle_of(ev, cal):
    return oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal, cal.pixel_threshold_e,
                      cal.cluster_threshold_e, ev.n_rows, ev.n_cols)


@pytest.mark.parametrize("config,event,over", [
    (0, 0, {}), (0, 1, {}), (1, 0, {}), (1, 7, {}), (3, 0, {}), (3, 5, {}),
    (4, 0, dict(n_modules=24)),                      # ~6.7k digis per module: workspace tier
    (4, 1, dict(n_modules=6, fill_pixels=1900)),     # shared-memory tier with long strips and merges
])
def test_chain_parity_on_workloads(pr, config, event, over):
    ev = wl.make_event(config, event, **over)
    cal = wl.make_calib(config, n_modules=ev.n_modules)
    out, got = run_device(pr, ev, cal)
    compare(out, oracle_of(ev, cal), lambda f: got[f])


def test_host_input_with_all_mirrors_and_callback(pr):
    ev = wl.make_event(1, 3)
    cal = wl.make_calib(1)
    ref = oracle_of(ev, cal)
    fired = []
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        hw = p.host_array(ev.n_words, np.uint32)
        ha = p.host_array(ev.n_words, np.uint16)
        hw[:] = ev.words
        ha[:] = ev.adc
        slot = p.slot()
        s = torch.cuda.Stream()
        slot.acquire(hw, ha, stream=s, want=pr.PR_WANT_ALL, event_id=42, done=lambda user, status: fired.append(status))
        wait(slot)
        t0 = time.time()
        while not fired and time.time() - t0 < 10:
            time.sleep(0.001)
        assert fired == [0]
        code, out = slot.produce()
        assert code == 0 and out.event_id == 42
        compare(out, ref, lambda f: out.host(f))              # exact-size pinned mirrors
        compare(out, ref, lambda f: out.to_numpy(f))          # and the device views
        slot.release()
        st = p.stats()
        assert st["callbacks_fired"] == 1 and st["events_produced"] == 1 and st["digis"] == ref.n_digis
        p.host_free(hw)
        p.host_free(ha)


def test_want_subset_gives_only_those_mirrors(pr):
    ev = wl.make_event(0, 2)
    cal = wl.make_calib(0)
    ref = oracle_of(ev, cal)
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        slot.acquire(to_dev(ev.words), to_dev(ev.adc), want=pr.PR_WANT_CLUSTERS)
        wait(slot)
        _, out = slot.produce()
        assert out.host("module") is None and out.host("label") is None and out.host("err_word") is None
        for f in ("cl_label", "cl_size", "cl_module", "mod_clus_start"):
            assert np.array_equal(out.host(f), getattr(ref, f))
        assert np.array_equal(out.host("cl_charge").view(np.uint32), ref.cl_charge.view(np.uint32))
        slot.release()


def hand(pixels, M):
    return wl.event_from_pixels(pixels, M)


def test_edge_cases(pr):
    cal = wl.flat_calib(4)
    cases = {
        "empty": hand([], 4),
        "all_errors": hand([0x80000001, 0x80100002, 0xFFFFFFFF], 4),
        "one": hand([(3, 159, 415, 255)], 4),
        "low_bits_and_out_of_range": wl.Event(np.array([wl.encode_word(1, 2, 3, 7), wl.encode_word(4, 0, 0), wl.encode_word(1, 160, 0),
                                                        wl.encode_word(1, 0, 416), wl.encode_word(1, 2, 4, 5)], np.uint32),
                                              np.array([60, 60, 60, 60, 60], np.uint16), 4),
        "duplicates": hand([(0, 5, 5, 50), (0, 9, 9, 50), (0, 5, 5, 30), (0, 5, 6, 20), (0, 5, 5, 99)], 4),
        "subthreshold_bridge": hand([(0, 3, 3, 60), (0, 3, 4, 12), (0, 3, 5, 60)], 4),
        "dropped_cluster": hand([(0, 3, 3, 13), (0, 3, 4, 13), (0, 9, 9, 60)], 4),
        "no_wrap": hand([(0, 159, 7, 60), (0, 0, 7, 60), (1, 10, 415, 60), (1, 11, 0, 60), (1, 10, 0, 60)], 4),
        "module_boundary": hand([(1, 3, 3, 60), (2, 3, 3, 60), (2, 4, 4, 60)], 4),
        "ragged_9_words": hand([(0, 1, c, 60) for c in range(9)], 4),
        # several small modules clustered in one register pass: same pixels in neighbouring modules stay apart,
        # an empty module in between, duplicates, a module boundary right next to a sub-threshold digi
        "pack_same_pixels": hand([(0, 10, 10, 60), (0, 10, 11, 60), (1, 10, 10, 60), (1, 10, 11, 60), (1, 11, 12, 60),
                                  (3, 10, 10, 60), (3, 9, 9, 12), (3, 10, 10, 70), (3, 11, 11, 20)], 4),
        "pack_exactly_32": hand([(0, 5, c, 60) for c in range(16)] + [(1, 5, c, 60) for c in range(0, 32, 2)], 4),
        "pack_33": hand([(0, 5, c, 60) for c in range(16)] + [(1, 5, c, 60) for c in range(17)], 4),
    }
    # U shape / spiral with the minimum index at the far end; strip interleaved
    arm1 = [(0, r, 10, 60) for r in range(60)]
    bottom = [(0, 59, c, 60) for c in range(11, 50)]
    arm2 = [(0, r, 50, 60) for r in range(59, -1, -1)]
    cases["u_shape"] = hand([arm2[-1]] + arm1 + bottom + arm2[:-1], 4)
    sp, r, c, dr, dc, seg = [], 80, 200, 0, 1, 2
    for _ in range(40):
        for _ in range(seg):
            sp.append((1, r, c, 60)); r += dr; c += dc
        dr, dc = dc, -dr
        seg += 2
    cases["spiral_reversed"] = hand(sp[::-1], 4)
    cols = list(range(100, 200))
    cases["strip"] = hand([(3, 80, c, 60) for c in cols[::2]] + [(3, 80, c, 60) for c in cols[1::2]], 4)
    for name, ev in cases.items():
        out, got = run_device(pr, ev, cal)
        compare(out, oracle_of(ev, cal), lambda f: got[f])


def test_full_and_checkerboard_and_lattice_module(pr):
    """Maximum sizes: 66 560 digis in one module (one cluster), 33 280 (checkerboard, one cluster),
    16 640 isolated pixels (as many clusters as digis: per-cluster workspace tier)."""
    rr, cc = np.meshgrid(np.arange(160), np.arange(416), indexing="ij")
    cal = wl.flat_calib(2)
    for sel in (np.ones_like(rr, bool), (rr + cc) % 2 == 0, (rr % 2 == 0) & (cc % 2 == 0)):
        w = ((1 << 20) | (rr[sel].astype(np.uint32) << 12) | (cc[sel].astype(np.uint32) << 3)).astype(np.uint32)
        w = np.random.default_rng(1).permutation(w)
        ev = wl.Event(w, np.full(w.shape[0], 60, np.uint16), 2)
        out, got = run_device(pr, ev, cal)
        compare(out, oracle_of(ev, cal), lambda f: got[f])


def test_general_geometry_and_thresholds(pr):
    """Largest field values (2048 modules of 256 x 512) and non-default thresholds."""
    rng = np.random.default_rng(5)
    n = 40000
    mods = np.sort(rng.integers(0, 2048, n)).astype(np.uint32)
    rows = rng.integers(0, 256, n).astype(np.uint32)
    cols = rng.integers(200, 512, n).astype(np.uint32)
    cols[: n // 2] = rng.integers(480, 512, n // 2)          # dense near the last column
    rows[: n // 2] = rng.integers(250, 256, n // 2)
    w = ((mods << 20) | (rows << 12) | (cols << 3)).astype(np.uint32)
    ev = wl.Event(w, rng.integers(0, 4096, n).astype(np.uint16), 2048, 256, 512)
    cal = wl.Calib(rng.uniform(1, 127, 2048).astype(np.float32), rng.normal(0, 3000, 2048).astype(np.float32), 600.0, 25000.0)
    out, got = run_device(pr, ev, cal)
    compare(out, oracle_of(ev, cal), lambda f: got[f])


def test_input_order_violation_is_reported_not_silent(pr):
    cal = wl.flat_calib(4)
    ev = hand([(2, 1, 1, 60), (0, 1, 1, 60), 0x80000000 | (5 << 20), (2, 3, 3, 60)], 4)
    fired = []
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        slot.acquire(to_dev(ev.words), to_dev(ev.adc), done=lambda u, s: fired.append(s))
        wait(slot)
        code, out = slot.produce(raise_on_error=False)
        assert code == pr.PR_ERR_INPUT_ORDER and out.status_bits & 1
        assert (out.n_digis, out.n_errors) == (3, 1)
        t0 = time.time()
        while not fired and time.time() - t0 < 10:
            time.sleep(0.001)
        assert fired == [pr.PR_ERR_INPUT_ORDER]
        slot.release()
        # the slot stays usable
        good = wl.make_event(0, 0, n_modules=4)
        slot.acquire(to_dev(good.words), to_dev(good.adc))
        wait(slot)
        code, out = slot.produce()
        assert code == 0
        ref = oracle.run(good.words, good.adc, 4, cal.gain, cal.pedestal)
        assert out.n_clusters == ref.n_clusters and np.array_equal(out.to_numpy("label"), ref.label)
        slot.release()
    # violation across a tile boundary (words 2047 | 2048) in a large event
    big = wl.make_event(1, 0)
    w = big.words.copy()
    valid = np.flatnonzero((w >> 31) == 0)
    i, j = valid[valid < 2048][-1], valid[valid >= 2048][0]
    w[i], w[j] = (w[i] & 0x800FFFFF) | (900 << 20), (w[j] & 0x800FFFFF) | (3 << 20)
    bad = wl.Event(w, big.adc, big.n_modules)
    calb = wl.make_calib(1)
    with pr.PixReco(calb.gain, calb.pedestal) as p:
        slot = p.slot()
        slot.acquire(to_dev(bad.words), to_dev(bad.adc))
        wait(slot)
        code, out = slot.produce(raise_on_error=False)
        assert code == pr.PR_ERR_INPUT_ORDER
        assert not oracle.decode(bad.words, bad.adc, bad.n_modules)["sorted_ok"]
        slot.release()


def test_batch_matches_single_events(pr):
    """pr_acquire_batch: 12 events of mixed sizes (incl. an empty one) in one chain of launches."""
    cal = wl.make_calib(1)
    evs = [wl.make_event(1, e) for e in range(5)] + [wl.make_event(3, e) for e in range(3)]
    evs += [wl.Event(np.zeros(0, np.uint32), np.zeros(0, np.uint16), 1856)]
    evs += [wl.make_event(1, 9), wl.make_event(3, 9),
            wl.event_from_pixels([(1855, 159, 415, 200)], 1856)]
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        dev = [(to_dev(e.words), to_dev(e.adc)) for e in evs]
        s = torch.cuda.Stream()
        slot.acquire_batch(dev, stream=s, want=pr.PR_WANT_CLUSTERS)
        wait(slot)
        code, outs = slot.produce_batch(len(evs))
        assert code == 0 and len(outs) == len(evs)
        for k, (e, out) in enumerate(zip(evs, outs)):
            assert out.event_id == k
            ref = oracle_of(e, cal)
            got = {f: out.to_numpy(f) for f in pr.VIEW_SPEC}
            compare(out, ref, lambda f: got[f])
            assert np.array_equal(out.host("cl_label"), ref.cl_label)
        slot.release()


@pytest.mark.parametrize("config,n_events", [(1, 64), (3, 256), (4, 1)])
def test_full_size_launches_as_bench_times_them(pr, config, n_events):
    """The launch configurations bench.py times, at BASELINE.json's full sizes: the 64-event configs[1] batch, a
    the 256-event configs[3] batch, one whole configs[4] event
    (12.4 M digis, dense path with the global workspace tier).  Every output array against the oracle."""
    cal = wl.make_calib(config)
    evs = [wl.make_event(config, 100 + e) for e in range(n_events)]
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        dev = [(to_dev(e.words), to_dev(e.adc)) for e in evs]
        if n_events > 1:
            slot.acquire_batch(dev, stream=torch.cuda.Stream())
        else:
            slot.acquire(*dev[0], stream=torch.cuda.Stream())
        wait(slot, timeout=300.0)
        code, outs = slot.produce_batch(n_events)
        assert code == 0
        for e, out in zip(evs, outs):
            ref = oracle_of(e, cal)
            got = {f: out.to_numpy(f) for f in pr.VIEW_SPEC}
            compare(out, ref, lambda f: got[f])
        slot.release()


@pytest.mark.parametrize("layout", ["one_span", "separate", "misaligned_span"])
def test_host_input_batch_staging_paths(pr, layout):
    """Pinned host inputs of a batch: one dense span (staged by one copy per array), separately allocated
    buffers and a span whose events are not 16-byte aligned relative to each other (one copy per event)."""
    cal = wl.make_calib(1)
    evs = [wl.make_event(1, 20 + e) for e in range(4)] + [wl.Event(np.zeros(0, np.uint32), np.zeros(0, np.uint16), 1856)]
    evs += [wl.make_event(3, 21), wl.event_from_pixels([(7, 3, 5, 90), (7, 3, 6, 120)], 1856)]
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        if layout == "separate":
            bufs = []
            for e in evs:
                hw, ha = p.host_array(max(e.n_words, 1), np.uint32), p.host_array(max(e.n_words, 1), np.uint16)
                hw[:e.n_words], ha[:e.n_words] = e.words, e.adc
                bufs.append((hw[:e.n_words], ha[:e.n_words]))
        else:
            step = 8 if layout == "one_span" else 3               # element alignment of each event inside the pool
            offs, tot = [], 0
            for e in evs:
                offs.append(tot)
                tot += (e.n_words + step - 1) // step * step + (0 if layout == "one_span" else 1)
            W, A = p.host_array(tot + 8, np.uint32), p.host_array(tot + 8, np.uint16)
            bufs = []
            for e, o in zip(evs, offs):
                W[o:o + e.n_words], A[o:o + e.n_words] = e.words, e.adc
                bufs.append((W[o:o + e.n_words], A[o:o + e.n_words]))
        slot = p.slot()
        st0 = p.stats()
        slot.acquire_batch(bufs, stream=torch.cuda.Stream(), want=pr.PR_WANT_ALL)
        wait(slot)
        code, outs = slot.produce_batch(len(evs))
        assert code == 0
        copies = p.stats()["memcpy_calls"] - st0["memcpy_calls"]
        n_nonempty = sum(1 for e in evs if e.n_words)
        if layout == "separate":                                   # pool blocks may or may not happen to be adjacent
            assert copies in (3, 2 * n_nonempty + 1)
        else:
            assert copies == (3 if layout == "one_span" else 2 * n_nonempty + 1)     # + the descriptor/export-table block
        for e, out in zip(evs, outs):
            ref = oracle_of(e, cal)
            compare(out, ref, lambda f: out.host(f))
        slot.release()


def _blob_module(rng, m, n, dup_frac=0.0, box=40):
    """n digis of module m packed into a small box (many merges, long chains), random order,
    ADC spanning both thresholds; optionally some duplicate pixels (A6)."""
    r0, c0 = int(rng.integers(0, 160 - box)), int(rng.integers(0, 416 - box))
    cells = rng.permutation(box * box)[: max(n - int(n * dup_frac), 1)]
    pix = [(m, r0 + int(x) // box, c0 + int(x) % box) for x in cells]
    while len(pix) < n:
        pix.append(pix[int(rng.integers(0, len(pix)))])
    order = rng.permutation(len(pix))
    return [(*pix[k], int(rng.integers(5, 256))) for k in order]


@pytest.mark.parametrize("sizes,dup", [
    ([1, 2, 31, 32, 33, 63, 64, 65, 127, 128, 129, 255, 256, 257, 0, 0, 300, 300, 511, 512, 513, 5, 1024, 3], 0.0),
    ([256] * 9 + [257] * 3 + [40] * 30, 0.0),
    ([17, 100, 256, 250, 257, 600, 20, 20], 0.15),
    ([3] * 700, 0.0),                                    # hundreds of modules per 512-digi window
    ([3000, 5, 40, 300, 9000, 0, 700, 33, 8192, 8193], 0.1),   # large on average: the large ones go to k_dense (both of its tiers)
    # both sides of the single-warp path's upper end (1024 digis) and of the dense path's shared-memory tier (2048), next to
    # runs of small modules that share a unit (at most four) and a ticket
    ([1023, 1024, 1025, 1500, 2048, 2049, 200, 100, 100, 100, 100] + [30] * 9 + [1, 0, 255, 2, 60, 60, 60, 60, 60, 7], 0.05),
])
def test_module_size_boundaries(pr, sizes, dup):
    """Modules on both sides of every path boundary of k_cluster (register packs up to 32 digis, units of up to four
    modules and 256 digis, one warp with global arrays up to 1024, the CTA-wide dense path beyond and its tiers)."""
    rng = np.random.default_rng(len(sizes) * 1000 + int(dup * 100))
    M = len(sizes) + 3
    pix = []
    for m, n in enumerate(sizes):
        if n:
            pix += _blob_module(rng, m + 1, n, dup, box=12 if n <= 64 else 40 if n <= 1500 else 64)
    ev = hand(pix, M)
    cal = wl.Calib(rng.uniform(60, 100, M).astype(np.float32), rng.normal(0, 200, M).astype(np.float32), 1000.0, 4000.0)
    out, got = run_device(pr, ev, cal)
    compare(out, oracle_of(ev, cal), lambda f: got[f])


@pytest.mark.parametrize("config,event,batch", [(0, 0, 1), (1, 3, 1), (3, 2, 1), (1, 20, 5)])
def test_words_in_arbitrary_order_are_bucketed_by_module_on_the_device(pr, config, event, batch):
    """A31 (PR_FLAG_UNORDERED_INPUT; the step before the decode in the paper's Fig. 1): every word of the event at a
    random place.  The device buckets the words stably by module, then runs the chain; every output equals the oracle's
    bucket step followed by its unchanged chain, word and error indices pointing into the shuffled INPUT.  Without the
    flag the same input ends with PR_ERR_INPUT_ORDER."""
    cal = wl.make_calib(config)
    rng = np.random.default_rng(100 + config)
    evs = []
    for k in range(batch):
        ev = wl.make_event(config, event + k)
        perm = rng.permutation(ev.n_words)
        evs.append(wl.Event(ev.words[perm].copy(), ev.adc[perm].copy(), ev.n_modules))
    if batch > 1:
        evs[2] = wl.Event(np.zeros(0, np.uint32), np.zeros(0, np.uint16), evs[0].n_modules)        # an empty event inside the batch
    refs = [oracle.run_unordered(e.words, e.adc, e.n_modules, cal.gain, cal.pedestal) for e in evs]
    with pr.PixReco(cal.gain, cal.pedestal, flags=pr.PR_FLAG_UNORDERED_INPUT) as p:
        slot = p.slot()
        for kind in ("device", "host"):
            if kind == "device":
                ins = [(to_dev(e.words), to_dev(e.adc)) for e in evs]
            else:
                ins = []
                for e in evs:
                    hw, ha = p.host_array(max(e.n_words, 1), np.uint32)[:e.n_words], p.host_array(max(e.n_words, 1), np.uint16)[:e.n_words]
                    hw[:], ha[:] = e.words, e.adc
                    ins.append((hw, ha))
            slot.acquire_batch(ins, stream=torch.cuda.Stream(), want=pr.PR_WANT_ALL if kind == "host" else 0)
            wait(slot)
            code, outs = slot.produce_batch(len(evs))
            assert code == 0
            for out, ref in zip(outs, refs):
                getter = (lambda f, o=out: o.host(f)) if kind == "host" else (lambda f, o=out: o.to_numpy(f))
                compare(out, ref, getter)
            slot.release()
        assert lib_code_of(pr, lambda: slot.digis_acquire(to_dev(evs[0].words), to_dev(evs[0].adc))) == pr.PR_ERR_INVALID_ARG
    if config == 1 and batch == 1:
        with pr.PixReco(cal.gain, cal.pedestal) as p:                       # the ordered contract (A5) still holds without the flag
            slot = p.slot()
            slot.acquire(to_dev(evs[0].words), to_dev(evs[0].adc), stream=torch.cuda.Stream())
            wait(slot)
            code, _ = slot.produce(raise_on_error=False)
            assert code == pr.PR_ERR_INPUT_ORDER
            slot.release()


def lib_code_of(pr, fn):
    try:
        return fn()
    except pr.PixRecoError as e:
        return e.code


def test_a_module_beyond_the_exact_sum_limit_is_reported_not_truncated(pr):
    """A9: the exact int64 sums are overflow-free up to 2^17 - 1 digis per module.  A module with 2^17 digis (every pixel
    of the module twice, minus a few) must end with PR_ERR_CAPACITY / PR_STATUS_CAPACITY — never a silently wrong answer
    (SURVEY 8(b) "Capacity") — the other modules of the event are clustered as usual, and the slot stays usable."""
    M, R, C = 4, 160, 416
    n_big = 1 << 17
    rng = np.random.default_rng(17)
    cells = np.concatenate([np.arange(R * C), rng.permutation(R * C)[: n_big - R * C]]).astype(np.uint32)
    rng.shuffle(cells)
    big = (np.uint32(2) << 20) | ((cells // C) << 12) | ((cells % C) << 3)
    small_pix = [(1, 10, 10, 200), (1, 10, 11, 200), (1, 50, 50, 200), (3, 7, 7, 200)]
    small = wl.event_from_pixels(small_pix, M)
    m1 = small.words[(small.words >> 20) == 1]; m3 = small.words[(small.words >> 20) == 3]
    words = np.concatenate([m1, big.astype(np.uint32), m3]).astype(np.uint32)
    adc = np.full(words.shape[0], 200, np.uint16)
    cal = wl.flat_calib(M)
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        slot.acquire(to_dev(words), to_dev(adc), stream=torch.cuda.Stream())
        wait(slot)
        code, out = slot.produce(raise_on_error=False)
        assert code == pr.PR_ERR_CAPACITY
        slot.release()
        # the same slot, an ordinary event: the status does not stick
        slot.acquire(to_dev(small.words), to_dev(small.adc), stream=torch.cuda.Stream())
        wait(slot)
        code, out = slot.produce()
        assert code == 0
        compare(out, oracle_of(small, cal), lambda f: out.to_numpy(f))
        slot.release()
