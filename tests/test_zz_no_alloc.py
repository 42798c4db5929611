"""pr_unpack_static: raw words -> digis with the caller's buffers and a file-scope __device__ scratch array, no
allocation anywhere (include/pixreco.h).  Its output against the existing path's (pr_acquire: same kernel, pool-backed
buffers) and against the oracle, bit for bit as the digi lists are everywhere else in tests/, on calls in a row that
share the scratch.  Collected last on purpose (the name): a failure here hides no other test under ``pytest -x``."""
import numpy as np
import pytest

import oracle
from paper_2004_04334_b200 import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

GUARD = 64            # elements of guard behind every output buffer: the call may not write beyond cap / M + 1
FILL = 0x5A


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


def wait(slot):
    import time
    t0 = time.time()
    while slot.query() == 1:
        assert time.time() - t0 < 60, "event did not complete"
        time.sleep(0.0002)


SIZES = {"d_module": 2, "d_row": 2, "d_col": 2, "d_adc": 2, "d_word_idx": 4, "d_charge": 4, "d_err_word": 4, "d_err_idx": 4,
         "d_mod_digi_start": 4, "d_counters": 4}
NP_TYPES = {"d_module": np.uint16, "d_row": np.uint16, "d_col": np.uint16, "d_adc": np.uint16, "d_word_idx": np.uint32,
            "d_charge": np.float32, "d_err_word": np.uint32, "d_err_idx": np.uint32, "d_mod_digi_start": np.uint32,
            "d_counters": np.uint32}
VIEW_OF = {"d_module": "module", "d_row": "row", "d_col": "col", "d_adc": "adc", "d_word_idx": "word_idx", "d_charge": "charge",
           "d_err_word": "err_word", "d_err_idx": "err_idx", "d_mod_digi_start": "mod_digi_start"}


def make_buffers(pr, cap, M):
    """The caller's output buffers (bytes, filled with a pattern), each with a guard behind it."""
    counts = {k: cap for k in pr.DIGIS_OUT_FIELDS}
    counts["d_mod_digi_start"], counts["d_counters"] = M + 1, 8
    bufs = {k: torch.full(((counts[k] + GUARD) * SIZES[k],), FILL, dtype=torch.uint8, device="cuda") for k in pr.DIGIS_OUT_FIELDS}
    return bufs, counts


def existing_path(pr, p, ev):
    """The digi part of pr_acquire (pool-backed buffers), copied to the host."""
    slot = p.slot()
    w, a = to_dev(ev.words), to_dev(ev.adc)
    slot.acquire(w, a, stream=torch.cuda.Stream())
    wait(slot)
    code, out = slot.produce()
    assert code == 0
    got = {k: out.to_numpy(v) for k, v in VIEW_OF.items()}
    counters = (out.n_words, out.n_digis, out.n_errors, out.status_bits)
    slot.release()
    return got, counters


def check_call(pr, p, ev, dev, cal, bufs, counts, stream, want, want_counters):
    w, a = dev
    for b in bufs.values():
        b.fill_(FILL)
    torch.cuda.synchronize()
    assert p.unpack_static(w, a, bufs, stream=stream) == 0
    stream.synchronize()
    host = {k: bufs[k].cpu().numpy() for k in bufs}
    c = host["d_counters"].view(np.uint32)
    n_words, n_digis, n_errors, status = int(c[0]), int(c[1]), int(c[2]), int(c[6])
    assert (n_words, n_digis, n_errors, status) == want_counters
    assert tuple(int(x) for x in c[3:6]) == (0, 0, 0) and int(c[7]) == 0
    ref = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal, cal.pixel_threshold_e, cal.cluster_threshold_e,
                     ev.n_rows, ev.n_cols)
    assert (n_words, n_digis, n_errors) == (ref.n_words, ref.n_digis, ref.n_errors)
    used = {k: n_digis for k in bufs}
    used["d_err_word"] = used["d_err_idx"] = n_errors
    used["d_mod_digi_start"], used["d_counters"] = ev.n_modules + 1, 8
    for k in pr.DIGIS_OUT_FIELDS:
        raw, n, sz = host[k], used[k], SIZES[k]
        got = raw[: n * sz].view(np.uint32 if k == "d_charge" else NP_TYPES[k])
        if k != "d_counters":
            exp = want[k][:n]
            assert np.array_equal(got, exp.view(np.uint32) if k == "d_charge" else exp), (k, "existing path")
            o = getattr(ref, VIEW_OF[k])[:n]
            assert np.array_equal(got, o.view(np.uint32) if k == "d_charge" else o), (k, "oracle")
        # nothing beyond the elements the call owns: the rest of the buffer and its guard keep the caller's pattern
        assert (raw[n * sz:] == FILL).all(), (k, "written beyond its size")


def test_static_unpack_matches_the_existing_path_on_calls_in_a_row(pr):
    cal = wl.make_calib(1)
    # a large event first, then smaller ones, then the large one again: the second call runs on the scratch the first one
    # left behind (more tiles than it needs itself), the last one on what a short event left
    evs = [wl.make_event(3, 1), wl.make_event(1, 4), wl.make_event(1, 5), wl.make_event(3, 1)]
    M = evs[0].n_modules
    cap = max((e.n_words + 7) // 8 * 8 for e in evs)
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        assert pr.pr_static_scratch_bytes() == 256 + 8 * (pr.PR_STATIC_MAX_WORDS // 2048) == 65792
        assert pr.pr_static_setup(p.handle) == 0
        want = [existing_path(pr, p, e) for e in evs]
        bufs, counts = make_buffers(pr, cap, M)
        outs2, _ = make_buffers(pr, cap, M)
        dev = [(to_dev(e.words), to_dev(e.adc)) for e in evs]   # (every device buffer of the test exists before the calls)
        stream = torch.cuda.Stream()
        st0 = p.stats()
        free0 = None
        for k, e in enumerate(evs):
            if k == 1:
                torch.cuda.synchronize()
                free0 = torch.cuda.mem_get_info()[0]          # (the first call may still load its kernels' code)
            check_call(pr, p, e, dev[k], cal, bufs, counts, stream, want[k][0], want[k][1])
        torch.cuda.synchronize()
        st = p.stats()
        for pool in ("device_pool", "host_pool"):              # the pools were not touched: no hit, no miss, no backend call
            assert st[pool] == st0[pool], pool
        assert st["memcpy_calls"] == st0["memcpy_calls"]
        assert torch.cuda.mem_get_info()[0] >= free0           # and the device has as much free memory as before
        # two calls back to back on one stream with no host wait in between: the second one's results are the last word
        assert p.unpack_static(*dev[0], bufs, stream=stream) == 0
        assert p.unpack_static(*dev[1], outs2, stream=stream) == 0
        stream.synchronize()
        for b, (got, cnt) in ((bufs, want[0]), (outs2, want[1])):
            c = b["d_counters"].cpu().numpy().view(np.uint32)
            assert (int(c[0]), int(c[1]), int(c[2]), int(c[6])) == cnt
            for k in ("d_module", "d_word_idx", "d_charge", "d_mod_digi_start"):
                n = M + 1 if k == "d_mod_digi_start" else cnt[1]
                g = b[k].cpu().numpy()[: n * SIZES[k]].view(np.uint32 if k == "d_charge" else NP_TYPES[k])
                e = got[k][:n]
                assert np.array_equal(g, e.view(np.uint32) if k == "d_charge" else e), k


def test_static_unpack_edge_cases_and_limits(pr):
    cal = wl.flat_calib(4)
    M = 4
    with pr.PixReco(cal.gain, cal.pedestal) as p:
        stream = torch.cuda.Stream()
        # beyond the maximum: a clear error, nothing enqueued, the buffers untouched
        bufs, counts = make_buffers(pr, 8, M)
        w = torch.zeros(8, dtype=torch.int32, device="cuda")
        a = torch.zeros(8, dtype=torch.int16, device="cuda")
        st0 = p.stats()
        rc = p.unpack_static(w, a, bufs, stream=stream, n_words=pr.PR_STATIC_MAX_WORDS + 1)
        assert rc == pr.PR_ERR_CAPACITY and pr.pr_strerror(rc) == b"internal capacity exceeded"
        assert p.stats()["kernel_launches"] == st0["kernel_launches"]
        stream.synchronize()
        assert all(bool((b == FILL).all()) for b in bufs.values())
        # a misaligned or missing buffer
        bad = dict(bufs); bad["d_charge"] = bufs["d_charge"][4:]
        assert p.unpack_static(w, a, bad, stream=stream) == pr.PR_ERR_INVALID_ARG
        # an empty event, an all-error event, one digi, a ragged tail of 9 words (after a larger call)
        rows = [[], None, [(3, 159, 415, 255)], [(0, 1, c, 60) for c in range(9)]]
        for spec in rows:
            if spec is None:
                ev = wl.Event(np.array([0x80000001, 0x80100002, 0xFFFFFFFF], np.uint32), np.array([1, 2, 3], np.uint16), M)
            else:
                ev = wl.Event(np.array([wl.encode_word(*x[:3]) for x in spec], np.uint32), np.array([x[3] for x in spec], np.uint16), M)
            ref = oracle.run(ev.words, ev.adc, M, cal.gain, cal.pedestal, cal.pixel_threshold_e, cal.cluster_threshold_e, ev.n_rows, ev.n_cols)
            bufs, counts = make_buffers(pr, 16, M)
            if ev.n_words:
                rc = p.unpack_static(to_dev(ev.words), to_dev(ev.adc), bufs, stream=stream)
            else:
                rc = p.unpack_static(None, None, bufs, stream=stream, n_words=0)
            assert rc == 0
            stream.synchronize()
            c = bufs["d_counters"].cpu().numpy().view(np.uint32)[:8]
            assert (int(c[0]), int(c[1]), int(c[2]), int(c[6])) == (ref.n_words, ref.n_digis, ref.n_errors, 0)
            for k, v in VIEW_OF.items():
                n = M + 1 if k == "d_mod_digi_start" else ref.n_errors if k.startswith("d_err") else ref.n_digis
                raw = bufs[k].cpu().numpy()
                got = raw[: n * SIZES[k]].view(np.uint32 if k == "d_charge" else NP_TYPES[k])
                exp = getattr(ref, v)[:n]
                assert np.array_equal(got, exp.view(np.uint32) if k == "d_charge" else exp), k
                assert (raw[n * SIZES[k]:] == FILL).all(), k
