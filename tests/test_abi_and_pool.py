"""CPU-only: the C-ABI library loads and exports every symbol include/pixreco.h declares, argument
validation that needs no device, and the caching allocator's host logic on the fake backend
(A23)."""
import ctypes
import os
import re

import pytest

from paper_2004_04334_b200 import pixreco as pr

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_every_declared_symbol_is_exported_and_bound():
    hdr = open(os.path.join(ROOT, "include", "pixreco.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pr_[a-z_]+)\s*\(", hdr)) - {"pr_done_fn"}
    assert declared == set(pr.SIGNATURES), declared ^ set(pr.SIGNATURES)
    lib = pr.lib()
    for name in declared:
        assert getattr(lib, name) is not None
    assert lib.pr_abi_version() == 4
    assert lib.pr_strerror(pr.PR_ERR_INPUT_ORDER).decode().startswith("input words")


def test_struct_layouts_match_the_header():
    # sizes the C side checks (struct_size) or relies on
    assert ctypes.sizeof(pr.pr_config) == 80
    assert ctypes.sizeof(pr.pr_input) == 56
    assert ctypes.sizeof(pr.pr_output) == 8 + 8 * 4 + 2 * 8 + 50 * 8       # event_id, counters, two device time stamps, 2 x 25 views
    assert ctypes.sizeof(pr.pr_pool_stats) == 64


def test_create_rejects_bad_arguments_without_a_device():
    import numpy as np
    lib = pr.lib()
    g, p = np.full(4, 80, np.float32), np.zeros(4, np.float32)

    def cfg(**kw):
        c = pr.pr_config(ctypes.sizeof(pr.pr_config), 0, 4, 160, 416, g.ctypes.data, p.ctypes.data, 1000.0, 4000.0, 0, 0, 0, 0, 0)
        for k, v in kw.items():
            setattr(c, k, v)
        return c
    h = ctypes.c_void_p()
    assert lib.pr_create(None, ctypes.byref(h)) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_create(ctypes.byref(cfg(struct_size=10)), ctypes.byref(h)) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_create(ctypes.byref(cfg(n_modules=0)), ctypes.byref(h)) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_create(ctypes.byref(cfg(n_modules=2049)), ctypes.byref(h)) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_create(ctypes.byref(cfg(n_rows=257)), ctypes.byref(h)) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_create(ctypes.byref(cfg(n_cols=513)), ctypes.byref(h)) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_create(ctypes.byref(cfg(pixel_threshold_e=100.0)), ctypes.byref(h)) == pr.PR_ERR_BAD_CALIB   # A9: >= 512
    assert lib.pr_create(ctypes.byref(cfg(pitch_row_um=-1.0)), ctypes.byref(h)) == pr.PR_ERR_INVALID_ARG      # A26
    g[2] = 0.0
    assert lib.pr_create(ctypes.byref(cfg()), ctypes.byref(h)) == pr.PR_ERR_BAD_CALIB
    g[2] = float("nan")
    assert lib.pr_create(ctypes.byref(cfg()), ctypes.byref(h)) == pr.PR_ERR_BAD_CALIB
    g[2] = 128.0
    assert lib.pr_create(ctypes.byref(cfg()), ctypes.byref(h)) == pr.PR_ERR_BAD_CALIB
    g[2] = 80.0
    p[1] = 70000.0
    assert lib.pr_create(ctypes.byref(cfg()), ctypes.byref(h)) == pr.PR_ERR_BAD_CALIB
    assert not h.value


def test_sources_keep_the_papers_rules():
    """PAPER.md L31 fn. 1 and L82-88 as static checks on the sources: the blocking CUDA calls appear only in
    pr_create / pr_destroy (job start / job end), and device code neither asserts, traps nor prints."""
    csrc = os.path.join(ROOT, "paper_2004_04334_b200", "csrc")
    api = open(os.path.join(csrc, "pixreco_api.cu")).read()
    blocking = re.compile(r"\bcuda(DeviceSynchronize|StreamSynchronize|EventSynchronize|Memcpy|Memset|Malloc|Free|HostAlloc|FreeHost)\s*\(")
    # split the file into top-level functions by their opening line
    funcs = re.split(r"\n(?=(?:int|void\*?|const char\*|uint64_t)\s+pr_[a-z_]+\s*\()", api)
    for f in funcs:
        m = re.match(r"(?:int|void\*?|const char\*|uint64_t)\s+(pr_[a-z_]+)", f)
        name = m.group(1) if m else "<helpers>"
        hits = set(x.group(0).rstrip("( ") for x in blocking.finditer(f))
        if name in ("pr_create", "pr_destroy"):
            continue
        assert not hits, (name, hits)
    # the pool: blocking or allocating CUDA calls only inside the backends' mem_alloc / mem_free (reached from a miss,
    # from trim and from destroy); a wait on an event or a stream nowhere at all
    pool = re.sub(r"//.*", "", open(os.path.join(csrc, "pool.cpp")).read())
    assert not re.search(r"\bcuda(DeviceSynchronize|StreamSynchronize|EventSynchronize|StreamWaitEvent|Memcpy|Memset)\w*\s*\(", pool)
    for m in re.finditer(r"\bcuda(Malloc|Free|HostAlloc|FreeHost)\w*\s*\(", pool):
        line_start = pool.rfind("\n", 0, m.start()) + 1
        head = pool[pool.rfind("\n", 0, pool.rfind("override", 0, m.end()) if "override" in pool[line_start:m.start()] else line_start):m.start()]
        fn_decl = max(pool.rfind("mem_alloc(", 0, m.start()), pool.rfind("mem_free(", 0, m.start()))
        other = max(pool.rfind(name, 0, m.start()) for name in ("event_create(", "event_destroy(", "event_record(", "event_done(", "::alloc(", "::free(", "::trim"))
        assert fn_decl > other, ("pool.cpp", m.group(0), pool[line_start:pool.find("\n", m.end())])
    for fn in os.listdir(csrc):
        if fn.endswith(".cuh"):
            code = re.sub(r"//.*", "", open(os.path.join(csrc, fn)).read())
            assert not re.search(r"(?<![_a-z])assert\s*\(|__trap\s*\(|\bprintf\s*\(", code), fn


def test_null_slots_are_rejected_without_a_device():
    """Every slot-level entry point checks its handle before touching CUDA."""
    lib = pr.lib()
    out = pr.pr_output()
    inp = pr.pr_input(None, None, 0, pr.PR_MEM_DEVICE, 0, 0, pr.pr_done_fn(), None)
    assert lib.pr_acquire(None, ctypes.byref(inp), None) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_acquire_batch(None, ctypes.byref(inp), 1, None) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_query(None) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_produce(None, ctypes.byref(out)) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_release(None) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_release_on(None, None) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_transfer(None, pr.PR_WANT_CLUSTERS, None, pr.pr_done_fn(), None) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_stream_wait_event(None, None) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_event_destroy(None) == pr.PR_ERR_INVALID_ARG
    assert lib.pr_destroy(None) == pr.PR_ERR_INVALID_ARG
    assert not lib.pr_event_cuda_event(None)


# ------------------------------------------------------------------ allocator on the fake backend
class Pool:
    def __init__(self, max_cached=0):
        self.lib = pr.lib()
        p = ctypes.c_void_p()
        assert self.lib.pr_pool_create(pr.PR_POOL_FAKE, 0, max_cached, ctypes.byref(p)) == 0
        self.p = p

    def alloc(self, n, stream):
        return self.lib.pr_pool_alloc(self.p, n, ctypes.c_void_p(stream))

    def free(self, ptr, stream, completed=0):
        return self.lib.pr_pool_free(self.p, ctypes.c_void_p(ptr), ctypes.c_void_p(stream), completed)

    def complete(self, stream):
        self.lib.pr_pool_fake_complete(self.p, ctypes.c_void_p(stream))

    def stats(self):
        st = pr.pr_pool_stats()
        self.lib.pr_pool_get_stats(self.p, ctypes.byref(st))
        return {n: int(getattr(st, n)) for n, _ in st._fields_}

    def close(self):
        self.lib.pr_pool_destroy(self.p)


def test_bin_sizes():
    lib = pr.lib()
    assert lib.pr_pool_bin_bytes(1) == 256 and lib.pr_pool_bin_bytes(256) == 256
    assert lib.pr_pool_bin_bytes(257) == 320 and lib.pr_pool_bin_bytes(512) == 512 and lib.pr_pool_bin_bytes(513) == 640
    assert lib.pr_pool_bin_bytes((1 << 36) + 1) == 0
    prev = 0
    for n in [1, 300, 1000, 5000, 123456, 10 ** 7, 10 ** 9, 3 * 10 ** 10]:
        b = lib.pr_pool_bin_bytes(n)
        assert b >= n and b <= max(256, int(n * 1.25) + 1) and b >= prev and b % 64 == 0
        prev = b


def test_same_stream_reuse_is_immediate_and_cross_stream_waits_for_the_event():
    pool = Pool()
    S1, S2 = 0x1000, 0x2000
    a = pool.alloc(1000, S1)
    assert a and pool.stats()["misses"] == 1
    assert pool.free(a, S1) == 0                    # not known complete: an event is recorded on S1
    # same stream: stream order makes reuse safe at once
    b = pool.alloc(900, S1)
    assert b == a and pool.stats()["hits"] == 1
    pool.free(b, S1)
    # other stream: must NOT get the block while S1's work is pending
    c = pool.alloc(1000, S2)
    assert c != a and pool.stats()["misses"] == 2 and pool.stats()["cross_stream_reuses"] == 0
    pool.free(c, S2)
    # once S1's event completes, the block may move to S2
    pool.complete(S1)
    d = pool.alloc(1000, 0x3000)
    assert d == a and pool.stats()["cross_stream_reuses"] == 1
    # `completed` frees are reusable anywhere at once
    pool.free(d, 0x3000, completed=1)
    e = pool.alloc(1024, 0x4000)
    assert e == a
    pool.free(e, 0x4000, 1)
    assert pool.free(0xDEAD0000, S1) == pr.PR_ERR_INVALID_ARG      # unknown pointer
    pool.close()


def test_steady_state_has_no_backend_calls_and_trim_returns_memory():
    pool = Pool()
    streams = [0x100 * (i + 1) for i in range(8)]
    sizes = [300_000, 1_200_000, 50_000, 7_000_000]
    import random
    rnd = random.Random(1)
    live = {}
    for it in range(2000):
        s = rnd.choice(streams)
        if s in live and rnd.random() < 0.7:
            for ptr in live.pop(s):
                pool.free(ptr, s)
            pool.complete(s)
        else:
            live.setdefault(s, []).append(pool.alloc(rnd.choice(sizes), s))
        if it == 1000:
            warm = pool.stats()["backend_allocs"]
    st = pool.stats()
    assert st["backend_allocs"] - warm <= 2, "cache must absorb the steady state"     # P:L90 amortisation
    assert st["backend_frees"] == 0
    assert len({p for v in live.values() for p in v}) == sum(len(v) for v in live.values())   # no double hand-out
    for s, v in live.items():
        for ptr in v:
            pool.free(ptr, s, 1)
    st = pool.stats()
    assert st["bytes_live"] == 0 and st["bytes_cached"] > 0
    pool.lib.pr_pool_trim(pool.p, 0)
    st = pool.stats()
    assert st["bytes_cached"] == 0 and st["backend_frees"] == st["backend_allocs"]
    pool.close()


def test_cache_cap_trims_oldest_first_and_never_a_pending_block():
    pool = Pool(max_cached=3000)
    S = 0x10
    ptrs = [pool.alloc(1024, S) for _ in range(4)]
    for ptr in ptrs[:3]:
        pool.free(ptr, S, 1)
    assert pool.stats()["bytes_cached"] == 2048 and pool.stats()["backend_frees"] == 1      # cap enforced, oldest went
    pool.free(ptrs[3], S, 0)                        # pending (event not complete): cannot be given back
    st = pool.stats()
    assert st["bytes_cached"] <= 3072 and st["backend_frees"] >= 1
    got = {pool.alloc(1024, 0x20) for _ in range(2)}
    assert ptrs[3] not in got                       # pending on S, other stream must not receive it
    pool.close()
