"""GPU: the chained modules (section 4.2): raw -> digis | digis -> clusters +
hits | digis -> occupancy as separate acquire/produce modules that pass a product {device, stream, event, views} and
never wait on the host in between.  Every output is compared with the oracle; the ScopedContext rule (first consumer
reuses the producer's stream, the others bring their own and wait on the event) is checked on the streams used."""
import ctypes
import time

import numpy as np
import pytest

import oracle
from paper_2004_04334_b200 import workloads as wl
from test_gpu_parity import compare, oracle_of, to_dev, wait

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def pr():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the product path has no CPU fallback")
    from paper_2004_04334_b200 import pixreco
    pixreco.lib()
    return pixreco


def make(pr, ev, cal, **kw):
    return pr.PixReco(cal.gain, cal.pedestal, ev.n_rows, ev.n_cols, cal.pixel_threshold_e, cal.cluster_threshold_e, **kw)


DIGI_FIELDS = ["module", "row", "col", "adc", "word_idx", "mod_digi_start", "err_word", "err_idx"]


def check_digis(out, ref, getter):
    assert (out.n_words, out.n_digis, out.n_errors) == (ref.n_words, ref.n_digis, ref.n_errors)
    for f in DIGI_FIELDS:
        assert np.array_equal(getter(f), getattr(ref, f)), f
    assert np.array_equal(getter("charge").view(np.uint32), ref.charge.view(np.uint32))


@pytest.mark.parametrize("config,event,over", [
    (0, 0, {}), (1, 3, {}), (3, 2, {}),
    (4, 0, dict(n_modules=24)),            # large modules: the consumer takes the k_dense route
])
def test_two_branch_dag_without_a_host_wait(pr, config, event, over):
    """digis on stream s0 behind a delay; clusters (first consumer) and occupancy (second consumer) are enqueued while
    the producer has not even started: nothing waits on the host between the modules."""
    ev = wl.make_event(config, event, **over)
    cal = wl.make_calib(config, n_modules=ev.n_modules)
    ref = oracle_of(ev, cal)
    with make(pr, ev, cal) as p:
        prod, clus, occ = p.slot(), p.slot(), p.slot()
        w, a = to_dev(ev.words), to_dev(ev.adc)
        s0, s1, s2 = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
        # Two passes: the first one fills the handle's pools (a fresh handle's first pinned and device allocations can
        # take longer than any delay one would want to queue: on a cold box they used to outlast the 0.2 s below once in
        # a while), the second one is the one that proves the point — it allocates nothing, so the host gets through
        # its three acquires long before the delay ahead of the producer is over.
        for delayed in (False, True):
            torch.cuda.synchronize()
            if delayed:
                with torch.cuda.stream(s0):
                    torch.cuda._sleep(1_000_000_000)                           # ~0.5 s of queue ahead of the producer
            prod.digis_acquire(w, a, stream=s0, event_id=77)
            product = prod.digis_product()
            used1 = clus.clusters_acquire(product, want=pr.PR_WANT_ALL, own_stream=s1)
            used2 = occ.occupancy_acquire(product, own_stream=s2)
            if delayed:
                assert prod.query() == pr.PR_NOT_READY, "the producer was complete before its consumers were enqueued: test proves nothing"
            # ScopedContext rule: first consumer on the producer's stream, second on its own
            assert used1 == s0.cuda_stream and used2 == s2.cuda_stream
            dev, st, evt = ctypes.c_int32(), ctypes.c_void_p(), ctypes.c_void_p()
            assert pr.lib().pr_product_info(ctypes.c_void_p(product), ctypes.byref(dev), ctypes.byref(st), ctypes.byref(evt)) == 0
            assert dev.value == 0 and (st.value or 0) == s0.cuda_stream and evt.value == prod.cuda_event
            # produce of a consumer is PR_NOT_READY while early, and the producer cannot be released under its consumers
            if delayed:
                assert clus.produce()[0] == pr.PR_NOT_READY and occ.occupancy_produce()[0] == pr.PR_NOT_READY
            wait(prod); wait(clus); wait(occ)
            assert prod.release() == pr.PR_NOT_READY

            code, dout = prod.produce()
            assert code == 0 and dout.event_id == 77 and dout.n_clusters == 0 and not dout.raw.d_cl_label
            check_digis(dout, ref, dout.to_numpy)
            code, cout = clus.produce()
            assert code == 0 and cout.event_id == 77
            compare(cout, ref, cout.host)                                      # pinned mirrors of every array
            compare(cout, ref, cout.to_numpy)                                  # device views
            code, cnt, tot = occ.occupancy_produce()
            assert code == 0
            ocnt, otot = oracle.occupancy(ref.module, ref.adc, ref.kept, ev.n_modules)
            assert np.array_equal(cnt, ocnt) and np.array_equal(tot, otot)
            assert int(cnt.sum()) == ref.n_kept_digis

            assert clus.release() == 0
            assert prod.release() == pr.PR_NOT_READY                           # the occupancy consumer still holds it
            assert occ.release() == 0
            assert prod.release() == 0
        st = p.stats()
        assert st["events_acquired"] == 2 and st["events_produced"] == 2 and st["digis"] == 2 * ref.n_digis and st["clusters"] == 2 * ref.n_clusters


def test_first_come_takes_the_stream_whatever_the_module(pr):
    """The order of the consumers' acquire calls decides who reuses the producer's stream, and a consumer of a
    product that is already complete does not wait at all."""
    ev = wl.make_event(1, 5)
    cal = wl.make_calib(1)
    ref = oracle_of(ev, cal)
    with make(pr, ev, cal) as p:
        prod, clus, occ, late = p.slot(), p.slot(), p.slot(), p.slot()
        w, a = to_dev(ev.words), to_dev(ev.adc)
        s0, s1, s2, s3 = (torch.cuda.Stream() for _ in range(4))
        prod.digis_acquire(w, a, stream=s0)
        product = prod.digis_product()
        assert occ.occupancy_acquire(product, own_stream=s2) == s0.cuda_stream
        assert clus.clusters_acquire(product, own_stream=s1) == s1.cuda_stream
        wait(prod); wait(clus); wait(occ)
        assert late.clusters_acquire(product, want=pr.PR_WANT_CLUSTERS | pr.PR_WANT_HITS, own_stream=s3) == s3.cuda_stream
        wait(late)
        for slot in (clus, late):
            code, out = slot.produce()
            assert code == 0
            compare(out, ref, out.to_numpy)
        compare(late.produce()[1], ref, late.produce()[1].host)
        code, cnt, tot = occ.occupancy_produce()
        ocnt, otot = oracle.occupancy(ref.module, ref.adc, ref.kept, ev.n_modules)
        assert code == 0 and np.array_equal(cnt, ocnt) and np.array_equal(tot, otot)
        for slot in (clus, occ, late, prod):
            assert slot.release() == 0


def test_chain_from_pinned_host_input_with_digi_mirrors_and_callbacks(pr):
    ev = wl.make_event(1, 9)
    cal = wl.make_calib(1)
    ref = oracle_of(ev, cal)
    fired = []
    with make(pr, ev, cal) as p:
        hw, ha = p.host_array(ev.n_words, np.uint32), p.host_array(ev.n_words, np.uint16)
        hw[:], ha[:] = ev.words, ev.adc
        prod, clus = p.slot(), p.slot()
        s0 = torch.cuda.Stream()
        prod.digis_acquire(hw, ha, stream=s0, want=pr.PR_WANT_DIGIS | pr.PR_WANT_CHARGE | pr.PR_WANT_ERRORS,
                           done=lambda user, status: fired.append(("digis", status)))
        clus.clusters_acquire(prod.digis_product(), want=pr.PR_WANT_CLUSTERS, own_stream=0,
                              done=lambda user, status: fired.append(("clusters", status)))
        wait(prod); wait(clus)
        t0 = time.time()
        while len(fired) < 2 and time.time() - t0 < 10:
            time.sleep(0.001)
        assert fired == [("digis", 0), ("clusters", 0)]                    # same stream: in order
        code, dout = prod.produce()
        assert code == 0
        check_digis(dout, ref, dout.host)
        code, cout = clus.produce()
        assert code == 0
        compare(cout, ref, cout.host)
        while clus.release() == pr.PR_NOT_READY or prod.release() == pr.PR_NOT_READY:
            time.sleep(0.001)
        p.host_free(hw); p.host_free(ha)


def test_input_order_violation_travels_with_the_product(pr):
    ev = wl.make_event(0, 2)
    cal = wl.make_calib(0)
    words = ev.words.copy()
    mods = (words >> 20) & 0xFFF
    i = int(np.nonzero(mods[1:] != mods[:-1])[0][0])
    words[[i, i + 1]] = words[[i + 1, i]]                                  # a module change out of order
    with make(pr, ev, cal) as p:
        prod, clus, occ = p.slot(), p.slot(), p.slot()
        w, a = to_dev(words), to_dev(ev.adc)
        s0, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        prod.digis_acquire(w, a, stream=s0)
        product = prod.digis_product()
        clus.clusters_acquire(product, own_stream=0)
        occ.occupancy_acquire(product, own_stream=s2)
        wait(prod); wait(clus); wait(occ)
        assert prod.produce(raise_on_error=False)[0] == pr.PR_ERR_INPUT_ORDER
        code, out = clus.produce(raise_on_error=False)
        assert code == pr.PR_ERR_INPUT_ORDER and out.n_clusters == 0 and out.status_bits & pr.PR_STATUS_INPUT_ORDER
        code, cnt, tot = occ.occupancy_produce()
        assert code == pr.PR_ERR_INPUT_ORDER and not cnt.any() and not tot.any()
        for slot in (clus, occ, prod):
            assert slot.release() == 0


def test_chain_argument_and_state_errors(pr):
    ev = wl.make_event(0, 0)
    cal = wl.make_calib(0)
    L = None
    with make(pr, ev, cal) as p:
        L = pr.lib()
        prod, clus = p.slot(), p.slot()
        out = ctypes.c_void_p()
        assert L.pr_digis_product(prod.ptr, ctypes.byref(out)) == pr.PR_ERR_BAD_STATE          # nothing acquired
        assert L.pr_digis_product(None, ctypes.byref(out)) == pr.PR_ERR_INVALID_ARG
        assert L.pr_clusters_acquire(clus.ptr, None, 0, None, None, pr.pr_done_fn(), None) == pr.PR_ERR_INVALID_ARG
        assert L.pr_occupancy_acquire(clus.ptr, None, None, None, pr.pr_done_fn(), None) == pr.PR_ERR_INVALID_ARG
        assert L.pr_occupancy_produce(clus.ptr, None, None, None, None) == pr.PR_ERR_BAD_STATE
        w, a = to_dev(ev.words), to_dev(ev.adc)
        inp, cb = prod._input(w, a, pr.PR_WANT_CLUSTERS, 0, None)
        assert L.pr_digis_acquire(prod.ptr, ctypes.byref(inp), None) == pr.PR_ERR_INVALID_ARG  # this module makes no clusters
        prod.digis_acquire(w, a, stream=0)
        product = prod.digis_product()
        assert L.pr_clusters_acquire(prod.ptr, ctypes.c_void_p(product), 0, None, None, pr.pr_done_fn(), None) == pr.PR_ERR_INVALID_ARG   # its own product
        assert L.pr_clusters_acquire(clus.ptr, ctypes.c_void_p(product), 1 << 9, None, None, pr.pr_done_fn(), None) == pr.PR_ERR_INVALID_ARG
        clus.clusters_acquire(product)
        assert L.pr_clusters_acquire(clus.ptr, ctypes.c_void_p(product), 0, None, None, pr.pr_done_fn(), None) == pr.PR_ERR_BAD_STATE     # busy slot
        wait(prod); wait(clus)
        assert L.pr_occupancy_produce(clus.ptr, None, None, None, None) == pr.PR_ERR_BAD_STATE # not an occupancy slot
        assert L.pr_event_destroy(prod.ptr) == pr.PR_ERR_BAD_STATE                             # a consumer holds its product
        assert clus.release() == 0 and prod.release() == 0
        assert L.pr_clusters_acquire(clus.ptr, ctypes.c_void_p(product), 0, None, None, pr.pr_done_fn(), None) == pr.PR_ERR_INVALID_ARG   # product gone with its slot's release
        # the slots go on to serve the fused path
        clus.acquire(w, a, stream=0)
        wait(clus)
        code, o = clus.produce()
        assert code == 0
        compare(o, oracle_of(ev, cal), o.to_numpy)
        clus.release()


def test_chain_in_steady_state_allocates_nothing_and_matches_the_fused_path(pr):
    """16 events through the three-module DAG on rotating slots: same tables as the fused pr_acquire, pool misses stop."""
    cal = wl.make_calib(1)
    evs = [wl.make_event(1, k) for k in range(16)]
    with make(pr, evs[0], cal) as p:
        trip = [(p.slot(), p.slot(), p.slot(), torch.cuda.Stream(), torch.cuda.Stream()) for _ in range(4)]
        dev = [(to_dev(e.words), to_dev(e.adc)) for e in evs]
        misses = None
        for rnd in range(3):
            for k, e in enumerate(evs):
                prod, clus, occ, s0, s1 = trip[k % 4]
                prod.digis_acquire(*dev[k], stream=s0)
                product = prod.digis_product()
                clus.clusters_acquire(product, own_stream=s1)
                occ.occupancy_acquire(product, own_stream=s1)
                if k % 4 == 3:
                    for j in range(k - 3, k + 1):
                        pj, cj, oj, _, _ = trip[j % 4]
                        wait(pj); wait(cj); wait(oj)
                        if rnd == 2:
                            ref = oracle_of(evs[j], cal)
                            out = cj.produce()[1]
                            compare(out, ref, out.to_numpy)
                            _, cnt, tot = oj.occupancy_produce()
                            ocnt, otot = oracle.occupancy(ref.module, ref.adc, ref.kept, evs[j].n_modules)
                            assert np.array_equal(cnt, ocnt) and np.array_equal(tot, otot)
                        assert cj.release() == 0 and oj.release() == 0 and pj.release() == 0
            st = p.stats()
            m = st["device_pool"]["misses"] + st["host_pool"]["misses"]
            if rnd == 2:
                assert m == misses, "pool misses in steady state"
            misses = m
