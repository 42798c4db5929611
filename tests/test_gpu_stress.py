"""GPU stress of the boundary (section 8(b) "Threading"):
several issuing host threads with every event checked against the oracle, the device pool under eight streams with
blocks that carry their owner's mark, and k_unpack launched with more CTAs than fit the device."""
import ctypes

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
    pixreco.driver()
    return pixreco


def to_dev(a):
    v = a.view(np.int32) if a.dtype == np.uint32 else a.view(np.int16)
    return torch.from_numpy(v.copy()).cuda()


def fnv1a32_np(a):
    """FNV-1a (64 bit) over 32-bit words, the fingerprint of prd_event_record, evaluated with Python integers on the
    oracle's array (the C++ driver evaluates the same recurrence on the pinned mirror)."""
    h = 1469598103934665603
    for v in np.asarray(a, np.uint32).tolist():
        h = ((h ^ v) * 1099511628211) & 0xFFFFFFFFFFFFFFFF
    return h


@pytest.mark.timeout(600)
def test_four_host_threads_drive_eight_slots_and_every_event_matches_the_oracle(pr):
    """framework tasks call acquire() from many threads.  Four C++ host threads issue pr_acquire /
    pr_produce / pr_release on eight slots (slot = stream = e mod 8, A25; thread t owns the slots s with s mod 4 == t),
    one event per acquire, 4 x 48 events; every event's counters, its label[] and its cluster labels are compared
    with the oracle through the pinned mirrors the issuing thread saw (fingerprints taken inside the thread)."""
    n_ev, passes = 48, 4
    cal = wl.make_calib(1)
    evs = [wl.make_event(1, e) for e in range(n_ev)]
    refs = [oracle.run(e.words, e.adc, e.n_modules, cal.gain, cal.pedestal) for e in evs]
    want_hash = [(fnv1a32_np(r.label), fnv1a32_np(r.cl_label)) for r in refs]
    dev = [(to_dev(e.words), to_dev(e.adc)) for e in evs]
    inp = (pr.pr_input * n_ev)()
    for k, (w, a) in enumerate(dev):
        inp[k] = pr.pr_input(w.data_ptr(), a.data_ptr(), evs[k].n_words, pr.PR_MEM_DEVICE,
                             pr.PR_WANT_LABELS | pr.PR_WANT_CLUSTERS, k, pr.pr_done_fn(), None)
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        slots = [p.slot() for _ in range(8)]
        streams = [torch.cuda.Stream() for _ in range(8)]
        torch.cuda.synchronize()
        for n_threads in (4, 2):
            d = pr.run_streams(slots, streams, inp, n_ev * passes, n_threads=n_threads, records=True)
            assert d["status"] == 0 and d["events"] == n_ev * passes
            threads_seen = set()
            for e in range(n_ev * passes):
                q, r = d["records"][e], refs[e % n_ev]
                assert q.event_id == e % n_ev and q.status_bits == 0
                assert (q.n_digis, q.n_errors, q.n_kept_digis, q.n_clusters_all, q.n_clusters) == \
                    (r.n_digis, r.n_errors, r.n_kept_digis, r.n_clusters_all, r.n_clusters), e
                assert (q.hash_label, q.hash_cl_label) == want_hash[e % n_ev], e
                assert q.thread == (e % 8) % n_threads
                threads_seen.add(q.thread)
            assert threads_seen == set(range(n_threads))
        s = p.stats()
        assert s["max_events_in_flight"] >= 4                  # several events were in flight at once (8 slots, 4 threads)


def _cudart():
    for name in ("libcudart.so.12", "libcudart.so"):
        try:
            return ctypes.CDLL(name)
        except OSError:
            continue
    pytest.fail("libcudart not loadable")


@pytest.mark.timeout(600)
def test_device_pool_under_eight_streams_never_hands_out_a_block_that_is_still_written(pr):
    """P:L88-90 / A23 on the real backend: a block freed on stream A with its work still queued must not reach
    another stream before that work is over.  Eight streams, random sizes out of a few bins (so that blocks do move
    between streams); every block is filled with its owner's mark by a long fill queued on the owner's stream, read
    back on the same stream and freed at once (not complete).  If the pool ever handed a block to a second owner
    while the first owner's fill was still queued, the late fill would overwrite the second owner's mark."""
    rt = _cudart()
    rt.cudaMemsetAsync.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t, ctypes.c_void_p]
    rt.cudaMemcpyAsync.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int, ctypes.c_void_p]
    pool = ctypes.c_void_p()
    assert pr.pr_pool_create(pr.PR_POOL_DEVICE, 0, 0, ctypes.byref(pool)) == 0
    streams = [torch.cuda.Stream() for _ in range(8)]
    rng = np.random.default_rng(7)
    sizes = [24 << 20, 30 << 20, 48 << 20, 6 << 20]          # three bins: 24 and 30 MiB round to the same one
    probe = 4096
    n_iter = 160
    host = torch.empty((n_iter, 2, probe), dtype=torch.uint8).pin_memory()
    marks = []
    try:
        for it in range(n_iter):
            s = streams[int(rng.integers(8))]
            size = sizes[int(rng.integers(len(sizes)))]
            ptr = pr.pr_pool_alloc(pool, size, ctypes.c_void_p(s.cuda_stream))
            assert ptr
            mark = 1 + it % 250
            marks.append(mark)
            # two long fills (a lower and an upper half) keep the block busy well after the host has moved on
            assert rt.cudaMemsetAsync(ptr, mark, size, ctypes.c_void_p(s.cuda_stream)) == 0
            assert rt.cudaMemsetAsync(ptr, mark, size, ctypes.c_void_p(s.cuda_stream)) == 0
            for k, off in enumerate((0, size - probe)):
                assert rt.cudaMemcpyAsync(host[it, k].data_ptr(), ptr + off, probe, 2, ctypes.c_void_p(s.cuda_stream)) == 0
            assert pr.pr_pool_free(pool, ctypes.c_void_p(ptr), ctypes.c_void_p(s.cuda_stream), 0) == 0
        torch.cuda.synchronize()
        got = host.numpy()
        for it, mark in enumerate(marks):
            assert (got[it] == mark).all(), f"block of iteration {it} was written by another owner"
        st = pr.pr_pool_stats()
        assert pr.pr_pool_get_stats(pool, ctypes.byref(st)) == 0
        assert st.hits > 0 and st.backend_allocs < n_iter, "the cache was used"
        assert st.cross_stream_reuses > 0, "blocks did move between streams (after their event)"
    finally:
        torch.cuda.synchronize()
        assert pr.pr_pool_destroy(pool) == 0


@pytest.mark.timeout(600)
def test_unpack_ends_with_more_ctas_than_fit_the_device_beside_other_streams(pr):
    """k_unpack hands out its tiles by ticket: a tile only waits for tiles of CTAs that are already running, whatever
    the order in which the hardware starts CTAs.  PR_FLAG_UNPACK_OVERSUBSCRIBE launches eight times as many CTAs as can
    be resident; eight streams run batches at once (their k_cluster / k_unpack CTAs share the SMs); every batch must
    end, and with the oracle's results."""
    n_ev = 24
    cal = wl.make_calib(3)
    evs = [wl.make_event(3, e) for e in range(n_ev)]
    refs = [oracle.run(e.words, e.adc, e.n_modules, cal.gain, cal.pedestal) for e in evs]
    dev = [(to_dev(e.words), to_dev(e.adc)) for e in evs]
    with pr.PixReco(cal.gain, cal.pedestal, flags=pr.PR_FLAG_UNPACK_OVERSUBSCRIBE) as p:
        slots = [p.slot() for _ in range(8)]
        streams = [torch.cuda.Stream() for _ in range(8)]
        for rep in range(3):
            for i, sl in enumerate(slots):
                sl.acquire_batch([dev[(3 * i + k + rep) % n_ev] for k in range(12)], stream=streams[i])
            for i, sl in enumerate(slots):
                import time
                t0 = time.time()
                while sl.query() == 1:
                    assert time.time() - t0 < 120, "a batch did not end"
                    time.sleep(0.0005)
                code, outs = sl.produce_batch(12)
                assert code == 0
                for k, out in enumerate(outs):
                    r = refs[(3 * i + k + rep) % n_ev]
                    assert (out.n_digis, out.n_errors, out.n_kept_digis, out.n_clusters_all, out.n_clusters) == \
                        (r.n_digis, r.n_errors, r.n_kept_digis, r.n_clusters_all, r.n_clusters)
                    if rep == 2 and k % 4 == 0:
                        assert np.array_equal(out.to_numpy("label"), r.label)
                        assert np.array_equal(out.to_numpy("cl_label"), r.cl_label)
                sl.release()
