"""GPU boundary behaviour: the acquire/produce contract of the paper, tested on the C ABI.

  * acquire launches work and returns; the thread is free
  * completion via callback on a non-framework thread, exactly once, carrying status (L35, L94)
  * work in one stream is serial, different streams concurrent (L82, L86); results identical
  * pool amortises runtime allocations: zero new cudaMalloc in steady state (L88-90)
  * a consumer on another stream waits on the product's event (L108)
  * transfers only when asked (L112)
"""
import ctypes
import threading
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
    v = a.view(np.int32) if a.dtype == np.uint32 else a.view(np.int16)
    return torch.from_numpy(v.copy()).cuda()


def wait(slot, timeout=60.0):
    t0 = time.time()
    while slot.query() == 1:
        assert time.time() - t0 < timeout
        time.sleep(0.0002)


def lib_code(fn):
    """The pr_* code of a binding call that raises PixRecoError."""
    from paper_2004_04334_b200 import pixreco
    try:
        return fn()
    except pixreco.PixRecoError as e:
        return e.code


def test_acquire_returns_at_once_behind_a_long_queue(pr):
    """A ~300 ms spin kernel sits in front on the same stream: pr_acquire must still return in
    well under that, pr_query/pr_produce must say NOT_READY without waiting."""
    ev, cal = wl.make_event(1, 0), wl.make_calib(1)
    with pr.PixReco(cal.gain, cal.pedestal, max_words_hint=60000, max_events_in_flight=8) as p:
        w, a = to_dev(ev.words), to_dev(ev.adc)
        slots = [p.slot() for _ in range(8)]
        streams = [torch.cuda.Stream() for _ in range(8)]
        for sl, s in zip(slots, streams):          # warm every slot (ctl buffers, pool bins)
            sl.acquire(w, a, stream=s); wait(sl); sl.produce(); sl.release()
        torch.cuda.synchronize()
        # warm the process for CONCURRENT streams too: the first launches behind busy streams make the driver set up its
        # per-stream work queues (2-30 ms per call, once per process, whatever is launched) — not part of an acquire
        for s in streams:
            with torch.cuda.stream(s):
                torch.cuda._sleep(int(0.02 * 2.0e9))
        for sl, s in zip(slots, streams):
            sl.acquire(w, a, stream=s)
        for sl in slots:
            wait(sl); sl.produce(); sl.release()
        torch.cuda.synchronize()
        spin_cycles = int(0.3 * 2.0e9)                # ~300 ms at the B200's 1.97 GHz
        for s in streams:
            with torch.cuda.stream(s):
                torch.cuda._sleep(spin_cycles)
        t_each = []
        for sl, s in zip(slots, streams):
            t0 = time.perf_counter()
            sl.acquire(w, a, stream=s)
            t_each.append(time.perf_counter() - t0)
        t_acq = sum(t_each)
        t0 = time.perf_counter()
        states = [sl.query() for sl in slots]
        codes = [sl.produce()[0] for sl in slots]
        t_poll = time.perf_counter() - t0
        assert states == [pr.PR_NOT_READY] * 8 and codes == [pr.PR_NOT_READY] * 8
        # typically 10-40 us per acquire through ctypes ("<< 1 ms"), against a 300 ms queue in front
        assert float(np.median(t_each)) < 1e-3, f"median acquire {np.median(t_each) * 1e6:.0f} us: {t_each}"
        assert t_acq < 0.02, f"8 acquires took {t_acq * 1e3:.2f} ms behind a 300 ms queue: {t_each}"
        assert t_poll < 0.02
        assert slots[0].release() == pr.PR_NOT_READY            # nothing is released while in flight
        with pytest.raises(pr.PixRecoError):                    # acquire on a busy slot
            slots[0].acquire(w, a, stream=streams[0])
        for sl in slots:
            wait(sl)
            assert sl.produce()[0] == 0
            sl.release()


def test_callback_fires_once_on_another_thread_with_outputs_visible(pr):
    ev, cal = wl.make_event(0, 0), wl.make_calib(0)
    ref = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
    seen = []
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        holder = {}

        def done(user, status):
            # runs on a CUDA-internal thread: only record; outputs must already be visible
            raw = pr.pr_output()
            seen.append((threading.get_ident(), status))

        for rep in range(5):
            slot.acquire(to_dev(ev.words), to_dev(ev.adc), stream=torch.cuda.Stream(), want=pr.PR_WANT_CLUSTERS, done=done)
            t0 = time.time()
            while len(seen) <= rep:
                assert time.time() - t0 < 20
                time.sleep(0.0005)
            code, out = slot.produce()             # after the callback: must be ready at once
            assert code == 0 and out.n_clusters == ref.n_clusters
            assert np.array_equal(out.host("cl_label"), ref.cl_label)
            slot.release()
        time.sleep(0.05)
        assert len(seen) == 5 and all(s == 0 for _, s in seen)
        assert all(t != threading.get_ident() for t, _ in seen)
        assert p.stats()["callbacks_fired"] == 5
        del holder


def test_concurrent_streams_same_results_and_zero_steady_state_malloc(pr):
    """configs[2] in small: 64 events, 8 in flight, slot = stream = e mod 8 (A25); every event's
    counters and cluster labels equal the oracle's; no cudaMalloc/cudaHostAlloc after warm-up."""
    cal = wl.make_calib(1)
    evs = [wl.make_event(1, e) for e in range(64)]
    refs = [oracle.run(e.words, e.adc, e.n_modules, cal.gain, cal.pedestal) for e in evs]
    dev = [(to_dev(e.words), to_dev(e.adc)) for e in evs]
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slots = [p.slot() for _ in range(8)]
        streams = [torch.cuda.Stream() for _ in range(8)]

        def one_pass(check):
            pending = {}
            for e in range(64):
                i = e % 8
                if i in pending:
                    wait(slots[i])
                    code, out = slots[i].produce()
                    check(pending.pop(i), code, out)
                    slots[i].release()
                slots[i].acquire(*dev[e], stream=streams[i], event_id=e)
                pending[i] = e
            for i, e in pending.items():
                wait(slots[i])
                code, out = slots[i].produce()
                check(e, code, out)
                slots[i].release()

        def check(e, code, out):
            r = refs[e]
            assert code == 0 and out.event_id == e
            assert (out.n_digis, out.n_errors, out.n_kept_digis, out.n_clusters_all, out.n_clusters) == \
                (r.n_digis, r.n_errors, r.n_kept_digis, r.n_clusters_all, r.n_clusters)
            assert np.array_equal(out.to_numpy("cl_label"), r.cl_label)
            assert np.array_equal(out.to_numpy("label"), r.label)

        one_pass(check)                             # warm-up fills the pools
        s0 = p.stats()
        spans = []                                  # (event, device ns when its first kernel started / its counters were out)

        def light(e, code, out):
            if not (code == 0 and out.n_clusters == refs[e].n_clusters):
                pytest.fail("mismatch")
            assert out.t_end_ns > out.t_start_ns > 0
            spans.append((e, out.t_start_ns, out.t_end_ns))
        for _ in range(3):
            one_pass(light)
        s1 = p.stats()
        # P:L86 "work in different streams may run concurrently": the device intervals of events on different
        # streams overlap (each event alone is far too small to fill the GPU)
        spans.sort(key=lambda x: x[1])
        overlapping = sum(1 for a, b in zip(spans, spans[1:]) if b[1] < a[2])
        assert overlapping >= len(spans) // 4, f"only {overlapping} of {len(spans)} consecutive events overlapped on the device"

        assert s1["device_pool"]["backend_allocs"] == s0["device_pool"]["backend_allocs"]
        assert s1["host_pool"]["backend_allocs"] == s0["host_pool"]["backend_allocs"]
        assert s1["device_pool"]["backend_frees"] == 0
        assert s1["max_events_in_flight"] == 8
        assert s1["events_produced"] == 4 * 64


def test_consumer_on_another_stream_waits_on_the_product_event(pr):
    """cudaStreamWaitEvent(consumerStream, productEvent) instead of a host wait."""
    ev, cal = wl.make_event(1, 1), wl.make_calib(1)
    ref = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        prod, cons = torch.cuda.Stream(), torch.cuda.Stream()
        w, a = to_dev(ev.words), to_dev(ev.adc)
        # learn the (stable) output addresses from a first run on this slot
        slot.acquire(w, a, stream=prod); wait(slot)
        _, out0 = slot.produce()
        charge_ptr, n = out0.raw.d_charge, out0.n_digis
        slot.release()
        with torch.cuda.stream(prod):
            torch.cuda._sleep(int(0.1 * 2.0e9))                   # ~0.1 s of queue ahead of the producer
        slot.acquire(w, a, stream=prod)
        assert slot.query() == pr.PR_NOT_READY
        assert slot.stream_wait(cons) == 0                      # cudaStreamWaitEvent, no host wait
        with torch.cuda.stream(cons):                           # consumer work queued BEFORE completion
            class _Cai:
                __cuda_array_interface__ = {"shape": (n,), "typestr": "<f4", "data": (charge_ptr, False), "version": 2, "strides": None}
            early_total = torch.as_tensor(_Cai(), device="cuda").double().sum()
        wait(slot)
        _, out = slot.produce()
        assert out.raw.d_charge == charge_ptr and out.n_digis == n      # same block reused (pool)
        with torch.cuda.stream(cons):
            total = out.device("charge").double().sum()
        assert float(total.item()) == pytest.approx(float(ref.charge.astype(np.float64).sum()), rel=1e-12)
        assert float(early_total.item()) == float(total.item())
        assert slot.stream_wait(cons) == 0                      # complete: returns at once
        slot.release()


def test_transfers_only_when_asked(pr):
    ev, cal = wl.make_event(0, 0), wl.make_calib(0)
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        slot.acquire(to_dev(ev.words), to_dev(ev.adc), want=0); wait(slot)
        _, out = slot.produce()
        assert all(out.host(f) is None for f in pr.VIEW_SPEC)
        slot.release()
        st = p.stats()
        # device input, no mirrors: 3 kernels and no copy at all (the slot's CUDA graph holds three kernel nodes whose
        # parameters carry the event's descriptor)
        assert st["memcpy_calls"] == 0 and st["kernel_launches"] == 3
        slot.acquire(to_dev(ev.words), to_dev(ev.adc), want=pr.PR_WANT_ERRORS); wait(slot)
        _, out = slot.produce()
        assert out.host("err_idx") is not None and out.host("cl_label") is None
        slot.release()
        assert p.stats()["kernel_launches"] == 7                            # + export kernel


def test_transfer_on_demand_is_a_stage_of_its_own(pr):
    """the copy to the host runs only when a consumer turns up, as an External-Worker stage of
    its own: pr_transfer after pr_produce, exact-size DMA copies, completion by query or callback."""
    cal = wl.make_calib(1)
    evs = [wl.make_event(1, 40), wl.make_event(1, 41), wl.Event(np.zeros(0, np.uint32), np.zeros(0, np.uint16), 1856)]
    refs = [oracle.run(e.words, e.adc, e.n_modules, cal.gain, cal.pedestal) for e in evs]
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        assert lib_code(lambda: slot.transfer(pr.PR_WANT_CLUSTERS)) == pr.PR_ERR_BAD_STATE          # nothing acquired
        slot.acquire_batch([(to_dev(e.words), to_dev(e.adc)) for e in evs], stream=torch.cuda.Stream(), want=pr.PR_WANT_ERRORS)
        wait(slot)
        code, outs = slot.produce_batch(len(evs))
        assert code == 0 and all(o.host("cl_label") is None and o.host("err_idx") is not None for o in outs)
        m0 = p.stats()["memcpy_calls"]
        fired = []
        consumer = torch.cuda.Stream()                                    # a consumer's stream, not the producer's
        slot.transfer(pr.PR_WANT_CLUSTERS | pr.PR_WANT_LABELS | pr.PR_WANT_ERRORS, stream=consumer, done=lambda u, st: fired.append(st))
        wait(slot)
        code, outs = slot.produce_batch(len(evs))
        assert code == 0
        # 19 arrays (clusters: 6 + mod_clus_start, labels: 2, per non-empty event; errors were mirrored already): more
        # than four, so they are gathered on the device and leave with ONE copy (+ one for the gather table)
        assert p.stats()["memcpy_calls"] - m0 == 2
        for o, r in zip(outs, refs):
            assert np.array_equal(o.host("cl_label"), r.cl_label) and np.array_equal(o.host("cl_size"), r.cl_size)
            assert np.array_equal(o.host("cl_module"), r.cl_module) and np.array_equal(o.host("mod_clus_start"), r.mod_clus_start)
            assert np.array_equal(o.host("cl_charge").view(np.uint32), r.cl_charge.view(np.uint32))
            assert np.array_equal(o.host("cl_row").view(np.uint32), r.cl_row.view(np.uint32))
            assert np.array_equal(o.host("cl_col").view(np.uint32), r.cl_col.view(np.uint32))
            assert np.array_equal(o.host("label"), r.label) and np.array_equal(o.host("clus"), r.clus)
            assert np.array_equal(o.host("err_idx"), r.err_idx) and o.host("charge") is None
        t0 = time.time()
        while not fired and time.time() - t0 < 10:
            time.sleep(0.001)
        assert fired == [0]
        st = p.stats()
        assert st["events_produced"] == len(evs) and st["events_in_flight"] == 0     # the stage does not count the events again
        slot.release()
        assert lib_code(lambda: slot.transfer(pr.PR_WANT_DIGIS)) == pr.PR_ERR_BAD_STATE             # released
        # a single event and few arrays: plain exact-size copies, no kernel
        slot.acquire(to_dev(evs[0].words), to_dev(evs[0].adc), want=0); wait(slot)
        assert slot.produce()[0] == 0
        s0 = p.stats()
        slot.transfer(pr.PR_WANT_CHARGE | pr.PR_WANT_ERRORS); wait(slot)
        code, out = slot.produce()
        s1 = p.stats()
        assert code == 0 and s1["memcpy_calls"] - s0["memcpy_calls"] == 3 and s1["kernel_launches"] == s0["kernel_launches"]
        assert np.array_equal(out.host("charge").view(np.uint32), refs[0].charge.view(np.uint32))
        assert np.array_equal(out.host("err_word"), refs[0].err_word) and np.array_equal(out.host("err_idx"), refs[0].err_idx)
        slot.release()


def test_argument_and_state_errors(pr):
    ev, cal = wl.make_event(0, 0), wl.make_calib(0)
    lib = pr.lib()
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        out = pr.pr_output()
        assert lib.pr_produce(slot.ptr, ctypes.byref(out)) == pr.PR_ERR_BAD_STATE      # produce before acquire
        assert lib.pr_query(slot.ptr) == pr.PR_ERR_BAD_STATE
        assert lib.pr_release(slot.ptr) == pr.PR_ERR_BAD_STATE
        pageable_w, pageable_a = ev.words.copy(), ev.adc.copy()
        inp = pr.pr_input(pageable_w.ctypes.data, pageable_a.ctypes.data, ev.n_words, pr.PR_MEM_HOST_PINNED, 0, 0, pr.pr_done_fn(), None)
        assert lib.pr_acquire(slot.ptr, ctypes.byref(inp), None) == pr.PR_ERR_INVALID_ARG   # pageable host memory
        w, a = to_dev(ev.words), to_dev(ev.adc)
        inp = pr.pr_input(w.data_ptr() + 4, a.data_ptr(), ev.n_words - 1, pr.PR_MEM_DEVICE, 0, 0, pr.pr_done_fn(), None)
        assert lib.pr_acquire(slot.ptr, ctypes.byref(inp), None) == pr.PR_ERR_INVALID_ARG   # misaligned device input
        inp = pr.pr_input(w.data_ptr(), a.data_ptr(), ev.n_words, 7, 0, 0, pr.pr_done_fn(), None)
        assert lib.pr_acquire(slot.ptr, ctypes.byref(inp), None) == pr.PR_ERR_INVALID_ARG
        inp = pr.pr_input(w.data_ptr(), a.data_ptr(), ev.n_words, pr.PR_MEM_DEVICE, 0x100, 0, pr.pr_done_fn(), None)
        assert lib.pr_acquire(slot.ptr, ctypes.byref(inp), None) == pr.PR_ERR_INVALID_ARG
        # still usable, on the legacy default stream (NULL)
        slot.acquire(w, a); wait(slot)
        assert slot.produce()[0] == 0
        slot.release()
        slot.destroy()


def test_legacy_aos_consumer_of_the_transfer_stage(pr):
    """P:L112-114 / SURVEY 8(f) NEXT-1, the consumer half: a CPU module that wants one record per cluster turns up after
    the event was produced without mirrors; pr_transfer fetches the cluster and hit tables (a stage of its own), and
    prd_clusters_to_aos turns the structure of arrays into an array of structures on the host — compared with the oracle."""
    cal = wl.make_calib(1)
    ev = wl.make_event(1, 11)
    r = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal)
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        slot.acquire(to_dev(ev.words), to_dev(ev.adc), stream=torch.cuda.Stream(), want=0)
        wait(slot)
        code, out = slot.produce()
        assert code == 0 and out.host("cl_label") is None
        assert lib_code(lambda: pr.clusters_to_aos(out)) == pr.PR_ERR_BAD_STATE      # no mirrors yet: nothing to convert
        slot.transfer(pr.PR_WANT_CLUSTERS | pr.PR_WANT_HITS, stream=torch.cuda.Stream())
        wait(slot)
        code, out = slot.produce()
        assert code == 0
        aos = pr.clusters_to_aos(out)
        assert len(aos) == r.n_clusters > 1000
        assert np.array_equal(aos["label"], r.cl_label) and np.array_equal(aos["size"], r.cl_size)
        assert np.array_equal(aos["module"], r.cl_module) and np.array_equal(aos["flags"], r.ht_flags)
        for f, ref in (("charge", r.cl_charge), ("row", r.cl_row), ("col", r.cl_col), ("x_um", r.ht_x), ("y_um", r.ht_y),
                       ("xerr_um", r.ht_xerr), ("yerr_um", r.ht_yerr)):
            assert np.array_equal(aos[f].view(np.uint32), ref.view(np.uint32)), f
        assert np.array_equal(aos["row_min"], r.ht_rows & 0xFFFF) and np.array_equal(aos["row_max"], r.ht_rows >> 16)
        assert np.array_equal(aos["col_min"], r.ht_cols & 0xFFFF) and np.array_equal(aos["col_max"], r.ht_cols >> 16)
        slot.release()


def test_a_slot_may_alternate_between_its_graph_and_plain_launches(pr):
    """The slot's CUDA graph (device input, no mirrors) has no memset node: its kernels leave the control words zeroed
    behind them.  An acquire outside the graph (mirrors wanted, a batch, a chained module) leaves its counters in the
    control block; the next graph launch must not see them.  Every step is compared with the oracle."""
    cal = wl.make_calib(1)
    evs = [wl.make_event(1, 30 + k) for k in range(4)]
    refs = [oracle.run(e.words, e.adc, e.n_modules, cal.gain, cal.pedestal) for e in evs]
    dev = [(to_dev(e.words), to_dev(e.adc)) for e in evs]
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slot = p.slot()
        stream = torch.cuda.Stream()

        def check(out, r):
            assert (out.n_digis, out.n_errors, out.n_kept_digis, out.n_clusters_all, out.n_clusters, out.status_bits) == \
                (r.n_digis, r.n_errors, r.n_kept_digis, r.n_clusters_all, r.n_clusters, 0)
            assert np.array_equal(out.to_numpy("clus"), r.clus) and np.array_equal(out.to_numpy("cl_label"), r.cl_label)
        plan = ["graph", "graph", "mirrors", "graph", "batch", "graph", "chain", "graph", "graph"]
        for step, kind in enumerate(plan):
            k = step % 4
            if kind == "batch":
                slot.acquire_batch([dev[k], dev[(k + 1) % 4]], stream=stream)
                wait(slot)
                code, outs = slot.produce_batch(2)
                assert code == 0
                check(outs[0], refs[k]); check(outs[1], refs[(k + 1) % 4])
            elif kind == "chain":
                slot.digis_acquire(*dev[k], stream=stream)
                wait(slot)
                code, out = slot.produce()
                assert code == 0 and out.n_digis == refs[k].n_digis
            else:
                slot.acquire(*dev[k], stream=stream, want=pr.PR_WANT_LABELS if kind == "mirrors" else 0)
                wait(slot)
                code, out = slot.produce()
                assert code == 0
                check(out, refs[k])
            slot.release()


def test_graph_acquire_is_complete_when_its_flag_is_up(pr):
    """A one-event acquire replayed from the slot's graph completes on a word in mapped pinned memory that the last CTA
    of k_finalize raises after a system-scope fence (no cudaEventQuery).  When pr_produce says PR_OK every output of
    the acquire must be visible to ANY stream: 300 events back to back, each read at once on a side stream that is not
    ordered with the slot's stream, and compared with the oracle (the next event is already queued behind it on the
    slot's stream: the slot's buffers come back from the pool, so a stale or partial table would show)."""
    cal = wl.make_calib(1)
    evs = [wl.make_event(1, 60 + k) for k in range(6)]
    refs = [oracle.run(e.words, e.adc, e.n_modules, cal.gain, cal.pedestal) for e in evs]
    dev = [(to_dev(e.words), to_dev(e.adc)) for e in evs]
    side = torch.cuda.Stream()
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slots = [p.slot(), p.slot()]
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        st0 = p.stats()
        slots[0].acquire(*dev[0], stream=streams[0])
        for it in range(300):
            cur, nxt = slots[it & 1], slots[(it + 1) & 1]
            nxt.acquire(*dev[(it + 1) % 6], stream=streams[(it + 1) & 1])     # keeps the device busy beside the read-back
            wait(cur)
            code, out = cur.produce()
            assert code == 0
            r = refs[it % 6]
            assert (out.n_digis, out.n_kept_digis, out.n_clusters_all, out.n_clusters) == \
                (r.n_digis, r.n_kept_digis, r.n_clusters_all, r.n_clusters), it
            with torch.cuda.stream(side):
                clus = out._device_bytes("clus").clone()
                lab = out._device_bytes("cl_label").clone()
                x = out._device_bytes("ht_x").clone()
            side.synchronize()
            assert np.array_equal(clus.cpu().numpy().view(np.int32), r.clus), it
            assert np.array_equal(lab.cpu().numpy().view(np.uint32), r.cl_label), it
            assert np.array_equal(x.cpu().numpy().view(np.float32), r.ht_x), it
            cur.release()
        wait(slots[0]); slots[0].produce(); slots[0].release()
        st = p.stats()
        assert st["memcpy_calls"] == st0["memcpy_calls"]             # all 301 went through the graph (no copies, no mirrors)
