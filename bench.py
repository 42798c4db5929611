#!/usr/bin/env python
"""bench.py — pixel local reconstruction throughput on B200 (BASELINE.json `metric`: events/s & Mdigis/s; achieved
HBM GB/s vs ~8 TB/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--slots S] [--no-extra]

Headline workload (`config.workload`): BASELINE.json configs[3], the largest batch workload that fits one GPU —
256-event high-pile-up batches (1856 modules, ~200k digis and ~30k clusters per event), each batch ONE
pr_acquire_batch / pr_produce_batch through the C ABI, `--slots` batches in flight on their own streams, timed
wall-clock on the device (CUDA events around a gate/join of all streams) from the first acquire to the last produce.
One *step* = `batches_per_step` such batches back to back (chosen from the warm-up so that K steps last >= 0.6 s
even at K = 20); every step is one pass of the whole hot path (unpack + calibrate + compact, cluster + reduce +
numbering + hits, counters to the host) over its events.

  value     device-resident inputs (R1).
  e2e       the same API with pinned HOST inputs and the cluster + hit tables copied back (R2): H2D and D2H inside the
            timed region.
  roofline  dominant kernel of the step from a PR_FLAG_KERNEL_TIMING pass (CUDA events on the launching stream, one
            batch in flight), every kernel with its own bound; chain fractions of the bytes-moved roofline; and
            `by_config`: all five BASELINE.json configs wall-clock through pr_acquire*/pr_produce* (configs[2] as worded:
            one pr_acquire per event on its own stream, 8 in flight, issued by 1, 2 and 4 C++ host threads).
  cpu_baseline  the oracle (oracle/, as it stands) on one host core AND on all host cores (one process per core), on a
            bounded sample of every config.

After every timed loop the last step's outputs are compared with the oracle (untimed).  Inputs are larger than the
126 MB L2 (a 256-event batch is 309 MB of input and ~10 GB of slab).  N>1 (torchrun): every rank runs the same
per-GPU workload on its own device (events are independent: no collective on the data path), time = max over ranks,
value = all ranks' events / that time ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import ctypes
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

HEAD_CONFIG = 3
HEAD_BATCH = 256             # events per pr_acquire_batch (BASELINE.json configs[3]: 256 events)
HEAD_POOL_BATCHES = 2        # distinct batches the steps rotate through (2 x 309 MB of input)
CFG1_BATCH = 64
STREAMS_IN_FLIGHT = 8        # configs[2]
NOMINAL_GBS = 8000.0         # BASELINE.json: "~8 TB/s"
# Thread-level operations the method needs per digi for a3 + a4 + hits (DESIGN.md section 6 derives it): the
# numerator of the ALU roofline of k_cluster; the denominator is 148 SMs x 128 lane-operations per cycle x the clock.
CLUSTER_OPS_PER_DIGI = 96.0
UNPACK_OPS_PER_WORD = 40.0


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--slots", type=int, default=2, help="batches in flight, device-resident (two keep the GPU busy back to back; with three the "
                                                         "third buys nothing: 1 %% slower)")
    ap.add_argument("--e2e-slots", type=int, default=3, help="batches in flight, end to end (the PCIe copies of one batch overlap the kernels of others)")
    ap.add_argument("--no-extra", action="store_true", help="skip roofline.by_config and the all-config CPU baseline")
    ap.add_argument("--only", default=None, choices=["configs1", "configs3", "configs4"],
                    help="run a few lone launches of this config's shape and exit (for ncu captures)")
    ap.add_argument("--reps", type=int, default=3, help="launches with --only")
    ap.add_argument("--min-seconds", type=float, default=0.6, help="length of the timed region the step size is chosen for")
    return ap.parse_args()


def load_profile(kernel):
    """Per-launch DRAM bytes / warp instructions of `kernel` on the headline launch, from profiles/traffic.json
    (written by `python -m paper_2004_04334_b200.ncu_summary` from an ncu --set full capture), or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            return json.load(f)["kernels"][kernel]
    except Exception:
        return None


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------ clocks
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index=0):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "50"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for n, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


# ------------------------------------------------------------------ workload
def make_pool(wl, config, n_events, first_event=0):
    return [wl.make_event(config, first_event + e) for e in range(n_events)]


def algorithmic_bytes(W, D, E, N, M):
    """DESIGN.md 'algorithmic bytes per unit', per event: k_unpack, k_cluster, chain minimum."""
    unpack = 6 * W + 16 * D + 8 * E + 4 * (M + 1)            # a1+a2 fused: read words+adc, write digi SoA+charge+errors
    cluster = 16 * D + 24 * N + 8 * (M + 1)                  # a3+a4 fused: read row,col,charge; write label,clus; cluster SoA
    chain = 6 * W + 24 * D + 24 * N + 8 * E + 8 * (M + 1) + 32
    return unpack, cluster, chain


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


# ------------------------------------------------------------------ the oracle, timed (reference arm and cpu_baseline)
def _oracle_worker(args):
    """One process = one oracle instance over its own events for about `budget` seconds.  Returns (events, digis, seconds)."""
    import oracle
    events, cal, budget, min_events = args
    ws = oracle.Workspace(max(e.n_words for e in events), cal.n_modules)
    n = d = 0
    t0 = time.perf_counter()
    while True:
        e = events[n % len(events)]
        oracle.run_raw(e.words, e.adc, e.n_modules, e.n_rows, e.n_cols, cal.gain, cal.pedestal,
                       cal.pixel_threshold_e, cal.cluster_threshold_e, ws)
        n += 1
        d += int(ws.counters[0])
        dt = time.perf_counter() - t0
        if (dt >= budget and n >= min_events) or n >= 1 << 20:
            return n, d, dt


_REF = {}     # the reference arm's events and calibration: set before the fork, inherited by the worker processes


def _ref_worker(args):
    """One step's share of one process of the reference arm: its own `per_proc` events (inherited through the fork, no
    copy per step), the oracle's workspace kept across steps.  Returns (events, digis)."""
    import oracle
    i, per_proc = args
    events, cal = _REF["pool"][i * per_proc:(i + 1) * per_proc], _REF["cal"]
    ws = _REF.get("ws")
    if ws is None:
        ws = _REF["ws"] = oracle.Workspace(max(e.n_words for e in _REF["pool"]), cal.n_modules)
    d = 0
    for e in events:
        oracle.run_raw(e.words, e.adc, e.n_modules, e.n_rows, e.n_cols, cal.gain, cal.pedestal,
                       cal.pixel_threshold_e, cal.cluster_threshold_e, ws)
        d += int(ws.counters[0])
    return len(events), d


def oracle_rates(pool, cal, budget_s, cores):
    """The oracle as it stands on 1 core and on `cores` cores (one independent process per core, each over its own
    slice of `pool`; if the pool has fewer events than cores the slices repeat, said in `sample`)."""
    import multiprocessing as mp
    n1, d1, t1 = _oracle_worker((pool, cal, budget_s, 1))
    res = {"cores_1": {"events_per_s": n1 / t1, "mdigis_per_s": d1 / t1 / 1e6, "sample": f"{n1} events in {t1:.2f} s"}}
    if cores > 1:
        slices = [pool[i::cores] if len(pool) >= cores else [pool[i % len(pool)]] for i in range(cores)]
        ctx = mp.get_context("fork")
        t0 = time.perf_counter()
        with ctx.Pool(cores) as p:
            out = p.map(_oracle_worker, [(s, cal, budget_s, 1) for s in slices])
        wall = time.perf_counter() - t0
        ev, dg, tmax = sum(o[0] for o in out), sum(o[1] for o in out), max(o[2] for o in out)
        res[f"cores_{cores}"] = {"events_per_s": ev / tmax, "mdigis_per_s": dg / tmax / 1e6,
                                 "sample": f"{ev} events, slowest process {tmax:.2f} s (wall incl. fork {wall:.2f} s)"
                                           + ("" if len(pool) >= cores else f"; {len(pool)} distinct events shared by the processes")}
    return res


def run_reference(args, rank):
    """The reference arm of the contract for this tier: the oracle on the box's host cores, same metric and workload."""
    if rank != 0:
        return
    from paper_2004_04334_b200 import workloads as wl
    import multiprocessing as mp
    cores = os.cpu_count() or 1
    cal = wl.make_calib(HEAD_CONFIG)
    per_proc = 8
    pool = make_pool(wl, HEAD_CONFIG, cores * per_proc)
    _REF["pool"], _REF["cal"] = pool, cal
    sample = len(pool)                                      # events per step: every process does `per_proc` events
    steps, warm = min(args.steps, 40), min(max(args.warmup, 1), 3)
    ctx = mp.get_context("fork")
    with ctx.Pool(cores) as p:
        jobs = [(i, per_proc) for i in range(cores)]
        for _ in range(warm):
            p.map(_ref_worker, jobs, chunksize=1)
        t0 = time.perf_counter()
        digis = 0
        for _ in range(steps):
            digis += sum(o[1] for o in p.map(_ref_worker, jobs, chunksize=1))
        dt = time.perf_counter() - t0
    v = sample * steps / dt
    line = {"impl": "reference", "metric": "pixel-reco events/s", "value": v, "unit": "events/s", "n_gpus": args.gpus,
            "steps": steps, "warmup": warm, "ms_per_step": dt / steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u32+f32 (exact int64 sums)", "data": "synthetic", "mdigis_per_s": digis / dt / 1e6,
            "config": {"workload": "configs[3] high-pile-up events (1856 modules, ~200k digis, ~30k clusters per event); the oracle on the host cores",
                       "sample": f"a step = {sample} events = {per_proc} per process on {cores} processes (a bounded sample of our arm's step)",
                       "cpu_model": cpu_model()},
            "cpu_baseline": {"value": v, "unit": "events/s", "cores": cores, "kind": "oracle",
                             "sample": f"{sample * steps} events of the configs[3] shape, one process per core"},
            "e2e": {"value": v, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------ our arm
class Bench:
    def __init__(self, torch, pr, device, cal, flags=0):
        self.torch, self.pr, self.device, self.cal = torch, pr, device, cal
        self.p = pr.PixReco(cal.gain, cal.pedestal, device=device, flags=flags)
        self.lib = pr.lib()
        self._keep = []

    def close(self):
        self.p.close()
        self._keep = []

    # -- inputs
    def upload(self, pool):
        """Device-resident copies (one big buffer each, 256-byte aligned slices)."""
        torch = self.torch
        offs, tot = [], 0
        for e in pool:
            offs.append(tot)
            tot += (e.n_words + 63) // 64 * 64
        W = np.zeros(max(tot, 64), np.uint32); A = np.zeros(max(tot, 64), np.uint16)
        for e, o in zip(pool, offs):
            W[o:o + e.n_words] = e.words; A[o:o + e.n_words] = e.adc
        dW = torch.from_numpy(W.view(np.int32)).to(f"cuda:{self.device}")
        dA = torch.from_numpy(A.view(np.int16)).to(f"cuda:{self.device}")
        self._keep.append((dW, dA))
        return [(dW.data_ptr() + 4 * o, dA.data_ptr() + 2 * o, e.n_words) for e, o in zip(pool, offs)]

    def pin(self, pool, per_batch=None):
        """Pinned host copies from the library's host pool; one block per `per_batch` events (a DAQ buffer)."""
        per_batch = per_batch or len(pool)
        ptrs = []
        for b0 in range(0, len(pool), per_batch):
            chunk = pool[b0:b0 + per_batch]
            offs, tot = [], 0
            for e in chunk:
                offs.append(tot)
                tot += (e.n_words + 63) // 64 * 64
            W = self.p.host_array(max(tot, 64), np.uint32); A = self.p.host_array(max(tot, 64), np.uint16)
            for e, o in zip(chunk, offs):
                W[o:o + e.n_words] = e.words; A[o:o + e.n_words] = e.adc
            self._keep.append((W, A))
            ptrs += [(W.ctypes.data + 4 * o, A.ctypes.data + 2 * o, e.n_words) for e, o in zip(chunk, offs)]
        return ptrs

    def inputs(self, ptrs, kind, want):
        pr = self.pr
        arr = (pr.pr_input * len(ptrs))()
        for k, (w, a, n) in enumerate(ptrs):
            arr[k] = pr.pr_input(w, a, n, kind, want, k, pr.pr_done_fn(), None)
        return arr

    @staticmethod
    def at(pr, arr, k):
        """POINTER(pr_input) to element k of a pr_input array."""
        return ctypes.cast(ctypes.addressof(arr) + k * ctypes.sizeof(pr.pr_input), ctypes.POINTER(pr.pr_input))

    # -- timed region helper: device time between a gate event and the join of all streams
    def timed(self, streams, fn):
        torch = self.torch
        gate = torch.cuda.Stream(device=self.device)
        start, end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(self.device)
        t0 = time.perf_counter()
        start.record(gate)
        for s in streams:
            s.wait_event(start)
        fn()
        for s in streams:
            gate.wait_stream(s)
        end.record(gate)
        torch.cuda.synchronize(self.device)
        wall = time.perf_counter() - t0
        return start.elapsed_time(end) * 1e-3, wall

    # -- batches of `nb` events, len(slots) batches in flight; returns (digis, clusters, outputs of the last batch, its index)
    def run_batches(self, inp, n_pool, nb, n_batches, slots, streams, first=0):
        lib, pr = self.lib, self.pr
        outs = [(pr.pr_output * nb)() for _ in slots]
        pool_batches = n_pool // nb
        busy = [None] * len(slots)
        tot = [0, 0]
        last = [None, None]

        def finish(i):
            while True:
                r = lib.pr_produce_batch(slots[i].ptr, outs[i], nb)
                if r != pr.PR_NOT_READY:
                    break
            if r != 0:
                raise RuntimeError(f"pr_produce_batch -> {r}")
            for k in range(nb):
                tot[0] += outs[i][k].n_digis; tot[1] += outs[i][k].n_clusters
            last[0], last[1] = i, busy[i]
        for s in range(n_batches):
            i = s % len(slots)
            if busy[i] is not None:
                finish(i)
                lib.pr_release(slots[i].ptr)
            b = (first + s) % pool_batches
            r = lib.pr_acquire_batch(slots[i].ptr, self.at(pr, inp, b * nb), nb, ctypes.c_void_p(streams[i].cuda_stream))
            if r != 0:
                raise RuntimeError(f"pr_acquire_batch -> {r}: {lib.pr_last_cuda_error(self.p.handle).decode()}")
            busy[i] = b
        order = sorted((i for i in range(len(slots)) if busy[i] is not None), key=lambda i: (i - (n_batches % len(slots))) % len(slots))
        for i in order:
            finish(i)
        self.last = (outs[last[0]], last[1] * nb, slots[last[0]]) if last[0] is not None else None
        return tot[0], tot[1]

    def release_all(self, slots):
        for s in slots:
            self.lib.pr_release(s.ptr)

    # -- one pr_acquire per event, Python loop (latency probes and the Python-driven configs[2])
    def run_single(self, inp, n_pool, n_events, slots, streams, first=0):
        lib, pr = self.lib, self.pr
        out = pr.pr_output()
        busy = [False] * len(slots)
        digis = clusters = 0
        ptrs = [self.at(pr, inp, k) for k in range(n_pool)]

        def finish(i):
            nonlocal digis, clusters
            while True:
                r = lib.pr_produce(slots[i].ptr, ctypes.byref(out))
                if r != pr.PR_NOT_READY:
                    break
            if r != 0:
                raise RuntimeError(f"pr_produce -> {r}")
            digis += out.n_digis; clusters += out.n_clusters
            lib.pr_release(slots[i].ptr)
            busy[i] = False
        for e in range(n_events):
            i = e % len(slots)
            if busy[i]:
                finish(i)
            r = lib.pr_acquire(slots[i].ptr, ptrs[(first + e) % n_pool], ctypes.c_void_p(streams[i].cuda_stream))
            if r != 0:
                raise RuntimeError(f"pr_acquire -> {r}: {lib.pr_last_cuda_error(self.p.handle).decode()}")
            busy[i] = True
        for i in range(len(slots)):
            if busy[i]:
                finish(i)
        return digis, clusters


def verify_against_oracle(pr, device, outs, events, cal, sample):
    """Untimed: events `sample` (indices into outs/events) of a finished step against the oracle — every counter, the
    cluster table and the hit table (device views copied back).  Raises on any difference."""
    import oracle
    for k in sample:
        ev = events[k]
        ref = oracle.run(ev.words, ev.adc, ev.n_modules, cal.gain, cal.pedestal, cal.pixel_threshold_e, cal.cluster_threshold_e,
                         ev.n_rows, ev.n_cols)
        o = pr.Output(outs[k], device)
        got = (o.n_words, o.n_digis, o.n_errors, o.n_kept_digis, o.n_clusters_all, o.n_clusters, o.status_bits)
        want = (ref.n_words, ref.n_digis, ref.n_errors, ref.n_kept_digis, ref.n_clusters_all, ref.n_clusters, 0)
        if got != want:
            raise RuntimeError(f"bench verification: counters {got} != oracle {want} (event {k})")
        for f in ("label", "clus", "cl_label", "cl_size", "cl_module", "mod_clus_start", "ht_rows", "ht_cols", "ht_flags"):
            if not np.array_equal(o.to_numpy(f), getattr(ref, f)):
                raise RuntimeError(f"bench verification: {f} differs from the oracle (event {k})")
        for f in ("charge", "cl_charge", "cl_row", "cl_col", "ht_x", "ht_y", "ht_xerr", "ht_yerr"):
            if not np.array_equal(o.to_numpy(f).view(np.uint32), getattr(ref, f).view(np.uint32)):
                raise RuntimeError(f"bench verification: {f} differs from the oracle (event {k})")
    return len(sample)


def chain_entry(events, digis, seconds, W, D, N, M, peak, E=None):
    E = W - D if E is None else E
    _, _, bchain = algorithmic_bytes(W, D, E, N, M)
    eps = events / seconds
    return {"events_per_s": eps, "mdigis_per_s": digis / seconds / 1e6, "chain_bytes_per_event": bchain,
            "chain_gbs": bchain * eps / 1e9, "chain_frac_of_measured_peak": bchain * eps / 1e9 / peak,
            "chain_frac_of_8TBs": bchain * eps / 1e9 / NOMINAL_GBS}


def run_ours(args, rank, world):
    from paper_2004_04334_b200 import workloads as wl
    peak, peak_src = load_peaks()
    K, Wm = args.steps, max(args.warmup, 3)
    cores = os.cpu_count() or 1
    extra = not args.no_extra

    # ---------------- inputs (seeded, synthetic; every rank its own events: weak scaling)
    cal3 = wl.make_calib(HEAD_CONFIG)
    M = cal3.n_modules
    n_pool = HEAD_BATCH * HEAD_POOL_BATCHES
    pool3 = make_pool(wl, HEAD_CONFIG, n_pool, first_event=rank * n_pool)
    meanW = float(np.mean([e.n_words for e in pool3]))

    # ---------------- the oracle on the host cores, before this process touches CUDA (fork-safe); rank 0 at N = 1 only
    cpu = None
    if rank == 0 and world == 1:
        budget = 1.5
        by = {"configs[3]": oracle_rates(pool3[:max(cores, 8)], cal3, budget, cores)}
        if extra:
            for cfg, n_ev in ((0, max(cores, 8)), (1, max(cores, 8)), (4, 2)):
                by[f"configs[{cfg}]"] = oracle_rates(make_pool(wl, cfg, n_ev), wl.make_calib(cfg), budget if cfg != 4 else 0.5, cores)
            by["configs[2]"] = {"note": "the events of configs[2] are 64 events of the configs[1] shape: same per-event oracle rate as configs[1]",
                                **by["configs[1]"]}
        head = by["configs[3]"]
        best = head.get(f"cores_{cores}", head["cores_1"])
        cpu = {"value": best["events_per_s"], "unit": "events/s", "cores": cores if f"cores_{cores}" in head else 1, "kind": "oracle",
               "sample": "configs[3] events: " + best["sample"] + "; one process per core over disjoint events",
               "value_1_core": head["cores_1"]["events_per_s"], "cpu_model": cpu_model(), "host_cores": cores, "by_config": by}

    import torch
    from paper_2004_04334_b200 import pixreco as pr
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    local = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(local)

    def max_over_ranks(x):
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=f"cuda:{local}")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    b = Bench(torch, pr, local, cal3)
    inp_dev = b.inputs(b.upload(pool3), pr.PR_MEM_DEVICE, 0)
    nslots = max(1, args.slots)
    slots = [b.p.slot() for _ in range(nslots)]
    streams = [torch.cuda.Stream(device=local) for _ in range(nslots)]

    # ---------------- R1: device-resident (the headline `value`)
    b.run_batches(inp_dev, n_pool, HEAD_BATCH, Wm * 2, slots, streams); b.release_all(slots)      # warm-up (fills the pools)
    t_probe, _ = b.timed(streams, lambda: b.run_batches(inp_dev, n_pool, HEAD_BATCH, 2 * nslots, slots, streams)); b.release_all(slots)
    t_batch = max_over_ranks(t_probe) / (2 * nslots)
    bps = int(min(64, max(1, np.ceil(args.min_seconds / (K * t_batch)))))              # batches per step
    st0 = b.p.stats()
    barrier()
    clk = ClockSampler(local)
    res = {}
    t_dev, t_wall = b.timed(streams, lambda: res.update(dc=b.run_batches(inp_dev, n_pool, HEAD_BATCH, K * bps, slots, streams, first=1)))
    barrier()
    clocks = clk.stop()
    st1 = b.p.stats()
    t_dev = max_over_ranks(t_dev)
    digis, clusters = res["dc"]
    n_events = K * bps * HEAD_BATCH
    value = world * n_events / t_dev
    launches = st1["kernel_launches"] - st0["kernel_launches"]
    new_mallocs = st1["device_pool"]["backend_allocs"] - st0["device_pool"]["backend_allocs"]
    outs_last, first_ev, _ = b.last
    verified = verify_against_oracle(pr, local, outs_last, pool3[first_ev:first_ev + HEAD_BATCH], cal3, (0, 97, HEAD_BATCH - 1))
    b.release_all(slots)
    Dm, Nm = digis / n_events, clusters / n_events
    head_chain = chain_entry(world * n_events, world * digis, t_dev, meanW, Dm, Nm, M, peak)

    # ---------------- R2: end to end — pinned host inputs, cluster + hit tables back, same API
    want_e2e = pr.PR_WANT_CLUSTERS | pr.PR_WANT_HITS
    inp_host = b.inputs(b.pin(pool3, per_batch=HEAD_BATCH), pr.PR_MEM_HOST_PINNED, want_e2e)
    n2 = max(1, args.e2e_slots)
    while len(slots) < n2:
        slots.append(b.p.slot()); streams.append(torch.cuda.Stream(device=local))
    slots2, streams2 = slots[:n2], streams[:n2]
    b.run_batches(inp_host, n_pool, HEAD_BATCH, 2 * n2, slots2, streams2); b.release_all(slots2)
    n_e2e = max(2 * n2, min(K * bps, 24))
    barrier()
    t_e2e, _ = b.timed(streams2, lambda: b.run_batches(inp_host, n_pool, HEAD_BATCH, n_e2e, slots2, streams2, first=1))
    barrier()
    t_e2e = max_over_ranks(t_e2e)
    outs_last, first_ev, _ = b.last
    o = pr.Output(outs_last[5], local)
    import oracle
    ev5 = pool3[first_ev + 5]
    ref5 = oracle.run(ev5.words, ev5.adc, ev5.n_modules, cal3.gain, cal3.pedestal)
    if not (np.array_equal(o.host("cl_label"), ref5.cl_label) and np.array_equal(o.host("ht_x").view(np.uint32), ref5.ht_x.view(np.uint32))):
        raise RuntimeError("bench verification: end-to-end host mirrors differ from the oracle")
    b.release_all(slots2)
    e2e_value = world * n_e2e * HEAD_BATCH / t_e2e
    h2d = int(6 * meanW * HEAD_BATCH * bps)
    d2h = int((48 * Nm + 4 * (M + 1) + 40) * HEAD_BATCH * bps)
    b.close()

    line = {"metric": "pixel-reco events/s", "value": value, "unit": "events/s", "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": t_dev / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u32+f32 (exact int64 sums)", "data": "synthetic",
            "mdigis_per_s": world * digis / t_dev / 1e6,
            "config": {"workload": "configs[3] high-pile-up: batches of 256 events (1856 modules, ~200k digis, ~30k clusters per event), "
                                   "one pr_acquire_batch/pr_produce_batch per batch",
                       "events_per_batch": HEAD_BATCH, "batches_per_step": bps, "events_per_step": HEAD_BATCH * bps,
                       "batches_in_flight": nslots, "mean_words_per_event": meanW, "mean_digis_per_event": Dm, "mean_clusters_per_event": Nm,
                       "timed_region_s": t_dev,
                       "l2_policy": f"inputs larger than L2: a batch reads {meanW * 6 * HEAD_BATCH / 1e6:.0f} MB and writes ~{(24 * Dm + 48 * Nm) * HEAD_BATCH / 1e6:.0f} MB; "
                                    f"steps rotate through {HEAD_POOL_BATCHES} distinct batches",
                       "residency": "R1 device-resident inputs, counters to mapped pinned host",
                       "verified_vs_oracle": f"{verified} events of the last timed batch: counters, labels, cluster and hit tables bit-equal (untimed)"},
            "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": e2e_value, "unit": "events/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": t_e2e / n_e2e * bps * 1e3, "batches_timed": n_e2e, "batches_in_flight": n2,
                    "what": "pinned host inputs (one block per batch from pr_host_alloc), want = CLUSTERS | HITS, same batch API; PCIe-bound in both directions at once (0.31 GB in and 0.31 GB out per 256-event batch; a DMA copy in and kernel stores out measured 45 GB/s each way together on this box, 55 / 53 GB/s alone): the mirrors leave through k_export's stores to mapped pinned memory, 32 CTAs streaming item after item; fetching them by a pr_transfer stage (gather + one DMA copy) instead measured 22k events/s"},
            "steady_state_cudaMalloc": int(new_mallocs), "wall_s": t_wall}

    if rank == 0:
        # ---------------- kernel timing pass for the roofline (same batches, PR_FLAG_KERNEL_TIMING, ONE batch in flight)
        bt = Bench(torch, pr, local, cal3, flags=pr.PR_FLAG_KERNEL_TIMING)
        it = bt.inputs(bt.upload(pool3), pr.PR_MEM_DEVICE, 0)
        sl = [bt.p.slot()]
        bt.run_batches(it, n_pool, HEAD_BATCH, 3, sl, streams[:1]); bt.release_all(sl)
        s0 = bt.p.stats()
        nrep = max(6, min(K * bps, 20))
        dg, cl = bt.run_batches(it, n_pool, HEAD_BATCH, nrep, sl, streams[:1], first=1); bt.release_all(sl)
        torch.cuda.synchronize(local)
        s1 = bt.p.stats()
        nt = s1["timed_acquires"] - s0["timed_acquires"]
        t_un = (s1["unpack_ms"] - s0["unpack_ms"]) / nt * 1e-3
        t_cl = (s1["cluster_ms"] - s0["cluster_ms"]) / nt * 1e-3
        t_fi = (s1["finalize_ms"] - s0["finalize_ms"]) / nt * 1e-3
        bt.close()
        Dk, Nk = dg / (nrep * HEAD_BATCH), cl / (nrep * HEAD_BATCH)
        bu, bc, bchain = algorithmic_bytes(meanW, Dk, meanW - Dk, Nk, M)
        sm_mhz = clocks.get("sm_mhz") or 1965.0
        alu_peak = 148 * 128 * sm_mhz * 1e6 / 1e9                                    # G thread-operations per second
        kern = {
            "k_unpack": {"bound": "hbm", "ms": t_un * 1e3, "algorithmic_bytes": bu * HEAD_BATCH, "gbs": bu * HEAD_BATCH / t_un / 1e9,
                         "frac_of_measured_peak": bu * HEAD_BATCH / t_un / 1e9 / peak, "frac_of_8TBs": bu * HEAD_BATCH / t_un / 1e9 / NOMINAL_GBS,
                         "profile": load_profile("k_unpack")},
            "k_cluster": {"bound": "alu", "ms": t_cl * 1e3, "algorithmic_bytes": bc * HEAD_BATCH, "gbs": bc * HEAD_BATCH / t_cl / 1e9,
                          "frac_of_measured_peak": bc * HEAD_BATCH / t_cl / 1e9 / peak, "frac_of_8TBs": bc * HEAD_BATCH / t_cl / 1e9 / NOMINAL_GBS,
                          "algorithmic_gops": CLUSTER_OPS_PER_DIGI * Dk * HEAD_BATCH / t_cl / 1e9, "alu_peak_gops": alu_peak,
                          "alu_frac": CLUSTER_OPS_PER_DIGI * Dk * HEAD_BATCH / t_cl / 1e9 / alu_peak, "profile": load_profile("k_cluster"),
                          "note": "a3 + a4 = k_cluster + k_finalize: the algorithmic bytes of the fused step are charged to k_cluster"},
            "k_finalize": {"bound": "hbm", "ms": t_fi * 1e3, "algorithmic_bytes": (8 * Dk + 92 * Nk + 4 * (M + 1)) * HEAD_BATCH,
                           "gbs": (8 * Dk + 92 * Nk + 4 * (M + 1)) * HEAD_BATCH / t_fi / 1e9,
                           "frac_of_measured_peak": (8 * Dk + 92 * Nk + 4 * (M + 1)) * HEAD_BATCH / t_fi / 1e9 / peak,
                           "profile": load_profile("k_finalize"),
                           "note": "what this kernel itself moves: clus read + written, the staged record of every kept cluster read (40 B of its 48), cluster and hit records written (52 B)"}}
        dom = max(kern, key=lambda k: kern[k]["ms"])
        prof = kern[dom]["profile"] or {}
        if dom == "k_cluster":
            roof = {"bound": "alu", "kernel": dom, "achieved": kern[dom]["algorithmic_gops"], "peak": alu_peak, "unit": "Gop/s",
                    "frac": kern[dom]["alu_frac"],
                    "peak_source": f"148 SMs x 128 lane-operations per cycle x {sm_mhz:.0f} MHz (sampled clock); {CLUSTER_OPS_PER_DIGI:.0f} thread-operations per digi (DESIGN.md 6)",
                    "hbm": {"achieved": kern[dom]["gbs"], "peak": peak, "unit": "GB/s", "frac": kern[dom]["frac_of_measured_peak"],
                            "frac_of_8TBs_nominal": kern[dom]["frac_of_8TBs"], "peak_source": peak_src}}
        else:
            roof = {"bound": "hbm", "kernel": dom, "achieved": kern[dom]["gbs"], "peak": peak, "unit": "GB/s",
                    "frac": kern[dom]["frac_of_measured_peak"], "frac_of_8TBs_nominal": kern[dom]["frac_of_8TBs"], "peak_source": peak_src}
        roof.update({"traffic": prof.get("dram_bytes_per_launch"), "algorithmic_bytes_per_launch": kern[dom]["algorithmic_bytes"],
                     "ms_per_launch": kern[dom]["ms"], "units_per_launch": f"{HEAD_BATCH} events", "kernels": kern,
                     "chain": {"bytes_per_event": bchain, "gbs": head_chain["chain_gbs"], "frac": head_chain["chain_frac_of_measured_peak"],
                               "frac_of_8TBs_nominal": head_chain["chain_frac_of_8TBs"],
                               "lone_launch_ms": (t_un + t_cl + t_fi) * 1e3, "lone_launch_frac": bchain * HEAD_BATCH / (t_un + t_cl + t_fi) / 1e9 / peak}})
        if extra:
            roof["by_config"] = run_by_config(torch, pr, wl, local, peak, head_chain)
        line["roofline"] = roof
        if cpu is not None:
            line["cpu_baseline"] = cpu
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


# ------------------------------------------------------------------ all five configs, wall-clock through the C ABI
def run_by_config(torch, pr, wl, local, peak, head_chain):
    out = {"configs[3]": {"what": "the headline: 256-event batches, device-resident", **head_chain}}
    # ---- configs[1]: 64-event batches of Run-3-like events, 2 batches in flight (measured: 1: 239k, 2: 325k, 3: 317k, 4: 311k, 6: 298k events/s)
    cal = wl.make_calib(1)
    pool = make_pool(wl, 1, 512)
    meanW = float(np.mean([e.n_words for e in pool]))
    b = Bench(torch, pr, local, cal)
    inp = b.inputs(b.upload(pool), pr.PR_MEM_DEVICE, 0)
    slots = [b.p.slot() for _ in range(STREAMS_IN_FLIGHT)]
    streams = [torch.cuda.Stream(device=local) for _ in range(STREAMS_IN_FLIGHT)]
    b.run_batches(inp, 512, CFG1_BATCH, 16, slots[:2], streams[:2]); b.release_all(slots[:2])
    nb = 1500
    r = {}
    t, _ = b.timed(streams[:2], lambda: r.update(dc=b.run_batches(inp, 512, CFG1_BATCH, nb, slots[:2], streams[:2], first=3)))
    outs_last, first_ev, _ = b.last
    verify_against_oracle(pr, local, outs_last, pool[first_ev:first_ev + CFG1_BATCH], cal, (0, 31, 63))
    b.release_all(slots[:2])
    D1, N1 = r["dc"][0] / (nb * CFG1_BATCH), r["dc"][1] / (nb * CFG1_BATCH)
    out["configs[1]"] = {"what": f"{CFG1_BATCH}-event batches through pr_acquire_batch, 2 in flight, device-resident, {nb} batches",
                         **chain_entry(nb * CFG1_BATCH, r["dc"][0], t, meanW, D1, N1, cal.n_modules, peak)}
    # one event at a time, one stream: the latency of a single pr_acquire -> pr_produce
    b.run_single(inp, 512, 64, slots[:1], streams[:1])
    t, _ = b.timed(streams[:1], lambda: b.run_single(inp, 512, 400, slots[:1], streams[:1], first=64))
    out["configs[1]"]["single_event_latency_us"] = t / 400 * 1e6
    # ---- configs[2] exactly as worded: 64 events, one pr_acquire each on its own stream, 8 in flight (A25), C++ host threads
    c2 = {}
    pr.run_streams(slots, streams, inp, 256, n_threads=1)                     # warm-up of the 8 slots
    st0 = b.p.stats()
    for nthr in (1, 2, 4):
        reps, best = 5, None
        for rep in range(reps):
            d = pr.run_streams(slots, streams, inp, 64 * 40, n_threads=nthr, first=64 * rep, spans=(rep == reps - 1))
            if best is None or d["wall_s"] < best["wall_s"]:
                best = {k: v for k, v in d.items() if not k.startswith("t_")}
            last = d
        sp = sorted(zip(last["t_start_ns"].tolist(), last["t_end_ns"].tolist()))
        busy_ns = sum(t1 - t0 for t0, t1 in sp)
        wall_ns = max(t1 for _, t1 in sp) - min(t0 for t0, _ in sp)
        ent = chain_entry(best["events"], best["digis"], best["wall_s"], meanW, D1, N1, cal.n_modules, peak)
        ent.update({"host_threads": nthr, "events": best["events"], "us_per_event": best["wall_s"] / best["events"] * 1e6,
                    "acquire_host_us_median": best["acquire_us_median"], "acquire_host_us_p99": best["acquire_us_p99"],
                    "mean_events_in_flight_on_device": busy_ns / max(wall_ns, 1),
                    "consecutive_events_overlapping": sum(1 for a, c in zip(sp, sp[1:]) if c[0] < a[1]) / max(len(sp) - 1, 1)})
        c2[f"threads_{nthr}"] = ent
    st1 = b.p.stats()
    t, _ = b.timed(streams, lambda: b.run_single(inp, 512, 64 * 20, slots, streams))
    c2["python_loop_events_per_s"] = 64 * 20 / t
    c2["new_cudaMalloc_in_timed_region"] = st1["device_pool"]["backend_allocs"] - st0["device_pool"]["backend_allocs"]
    c2["what"] = ("one pr_acquire / pr_produce / pr_release per event, slot = stream = event mod 8 (A25), device-resident inputs, "
                  "issued by C++ host threads (libpixreco_driver.so); wall clock from the first acquire to the last produce")
    best_thr = max((k for k in c2 if k.startswith("threads_")), key=lambda k: c2[k]["events_per_s"])
    out["configs[2]"] = {**{k: v for k, v in c2[best_thr].items()}, "best": best_thr, **c2}
    b.close()
    # ---- configs[0]: the tiny event, one at a time and 8 streams
    cal = wl.make_calib(0)
    pool = make_pool(wl, 0, 64)
    meanW0 = float(np.mean([e.n_words for e in pool]))
    b = Bench(torch, pr, local, cal)
    inp = b.inputs(b.upload(pool), pr.PR_MEM_DEVICE, 0)
    slots = [b.p.slot() for _ in range(STREAMS_IN_FLIGHT)]
    streams = [torch.cuda.Stream(device=local) for _ in range(STREAMS_IN_FLIGHT)]
    b.run_single(inp, 64, 64, slots[:1], streams[:1])
    r = {}
    t, _ = b.timed(streams[:1], lambda: r.update(dc=b.run_single(inp, 64, 400, slots[:1], streams[:1])))
    pr.run_streams(slots, streams, inp, 256, n_threads=2)
    d = pr.run_streams(slots, streams, inp, 64 * 40, n_threads=2)
    D0, N0 = r["dc"][0] / 400, r["dc"][1] / 400
    out["configs[0]"] = {"what": "1 tiny event per pr_acquire; `events_per_s` = 8 streams in flight from 2 C++ host threads; latency = one event at a time",
                         **chain_entry(d["events"], d["digis"], d["wall_s"], meanW0, D0, N0, cal.n_modules, peak),
                         "single_event_latency_us": t / 400 * 1e6}
    b.close()
    # ---- configs[4]: clustering stress, one event per pr_acquire, 2 in flight; 16 events (4 distinct ones, cycled)
    cal = wl.make_calib(4)
    pool = make_pool(wl, 4, 4)
    meanW4 = float(np.mean([e.n_words for e in pool]))
    b = Bench(torch, pr, local, cal)
    inp = b.inputs(b.upload(pool), pr.PR_MEM_DEVICE, 0)
    slots = [b.p.slot() for _ in range(2)]
    streams = [torch.cuda.Stream(device=local) for _ in range(2)]
    b.run_single(inp, 4, 4, slots, streams)
    r = {}
    t, _ = b.timed(streams, lambda: r.update(dc=b.run_single(inp, 4, 16, slots, streams)))
    D4, N4 = r["dc"][0] / 16, r["dc"][1] / 16
    out["configs[4]"] = {"what": "16 events (4 distinct, cycled), one pr_acquire per event, 2 in flight, device-resident",
                         **chain_entry(16, r["dc"][0], t, meanW4, D4, N4, cal.n_modules, peak)}
    # one of them against the oracle
    s = slots[0]
    s.acquire(b._keep[0][0][:pool[0].n_words], b._keep[0][1][:pool[0].n_words], stream=streams[0])
    while s.query() == pr.PR_NOT_READY:
        pass
    outs = (pr.pr_output * 1)()
    pr.lib().pr_produce_batch(s.ptr, outs, 1)
    verify_against_oracle(pr, local, outs, pool[:1], cal, (0,))
    s.release()
    b.close()
    return out


def run_only(args):
    """A few lone launches of one config's shape (for ncu captures of HBM-sized launches)."""
    import torch
    from paper_2004_04334_b200 import pixreco as pr, workloads as wl
    config, n_ev, batch = {"configs1": (1, CFG1_BATCH, True), "configs3": (3, HEAD_BATCH, True), "configs4": (4, 1, False)}[args.only]
    cal = wl.make_calib(config)
    pool = make_pool(wl, config, n_ev)
    b = Bench(torch, pr, 0, cal, flags=pr.PR_FLAG_KERNEL_TIMING)
    inp = b.inputs(b.upload(pool), pr.PR_MEM_DEVICE, 0)
    slots, streams = [b.p.slot()], [torch.cuda.Stream(device=0)]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda:0")
    for r in range(args.reps):
        flush.fill_(r)
        torch.cuda.synchronize(0)
        if batch:
            b.run_batches(inp, n_ev, n_ev, 1, slots, streams); b.release_all(slots)
        else:
            b.run_single(inp, n_ev, 1, slots, streams)
    st = b.p.stats()
    print(json.dumps({"config": args.only, "launches": args.reps, "unpack_ms": st["unpack_ms"] / st["timed_acquires"],
                      "cluster_ms": st["cluster_ms"] / st["timed_acquires"], "finalize_ms": st["finalize_ms"] / st["timed_acquires"]}), flush=True)
    b.close()


def main():
    args = parse()
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.only:
        run_only(args)
        return
    run_ours(args, rank, world)


if __name__ == "__main__":
    main()
