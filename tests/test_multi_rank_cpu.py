"""N>1 path on CPU (gloo, world_size 2): bench.py shards by giving every rank its own events and
aggregates timing as max-over-ranks; there is no data-path collective (events are
independent units).  This covers that host logic without a GPU."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys, json
    sys.path.insert(0, %r)
    import numpy as np, torch, torch.distributed as dist
    from paper_2004_04334_b200 import workloads as wl
    import bench
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    # every rank draws its own events (weak scaling): disjoint event indices
    n_pool = 4
    pool = bench.make_pool(wl, 0, n_pool, first_event=rank * n_pool)
    sig = np.array([int(e.words.astype(np.uint64).sum()) for e in pool], dtype=np.int64)
    allsig = [torch.zeros(n_pool, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(allsig, torch.from_numpy(sig))
    flat = torch.cat(allsig).tolist()
    assert len(set(flat)) == len(flat), "ranks must process disjoint events"
    # timing aggregation: value = all ranks' events / max-over-ranks time
    t = torch.tensor([0.5 + rank], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    assert float(t.item()) == 0.5 + (world - 1)
    value = world * 64 / float(t.item())
    dist.barrier()
    if rank == 0:
        print(json.dumps({"value": value, "world": world}))
    dist.destroy_process_group()
""") % ROOT


def test_two_ranks_disjoint_events_and_max_time():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import tempfile
    with tempfile.NamedTemporaryFile("w", suffix=".py", delete=False) as f:
        f.write(WORKER)
        path = f.name
    try:
        out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                              "--master-addr", "127.0.0.1", "--master-port", str(port), path],
                             env=env, capture_output=True, text=True, timeout=300)
        assert out.returncode == 0, out.stderr[-2000:]
        line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
        import json
        d = json.loads(line)
        assert d["world"] == 2 and abs(d["value"] - 2 * 64 / 1.5) < 1e-9
    finally:
        os.unlink(path)


def test_reference_arm_prints_contract_line_only_on_rank0():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                         env=env, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2", "--warmup", "1"],
                         env=env, capture_output=True, text=True, timeout=300)
    import json
    d = json.loads(out.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["unit"] == "events/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
