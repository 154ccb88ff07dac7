"""The N > 1 plumbing of bench.py (barrier + max over ranks, rank-0 reporting, per-rank seeds), run as two gloo processes
on CPU.  No GPU and no product kernels are involved.  The data path itself shards the events over the ranks and sums the
ranks' accumulators once per iteration (paper_1502_07478_b200/sharding.py; its host logic is tests/test_sharding_gloo.py)."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import bench

    r = bench.Ranks("gloo", None)
    assert (r.world, r.rank) == (world, rank)
    r.barrier()
    slow = r.max(1.0 + rank)                       # the slowest replica sets the time
    agg = r.aggregate(1000.0, 0.5 * (1 + rank))     # units of all ranks / slowest time
    seeds = r.seed(7)
    r.close()
    out.put((rank, slow, agg, seeds))


def test_two_rank_timing_reduce_and_seeds():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[1] for g in got] == [2.0, 2.0]
    assert [g[2] for g in got] == [pytest.approx(2 * 1000.0 / 1.0)] * 2
    assert [g[3] for g in got] == [7, 8]


def test_reference_arm_prints_only_on_rank_zero(tmp_path):
    """bench.py --impl reference under two ranks: rank 0 prints one JSON line, rank 1 exits 0 without work."""
    import json
    import subprocess

    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    outs = []
    for rank in (1, 0):
        e = dict(env, RANK=str(rank), LOCAL_RANK=str(rank))
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                            "--warmup", "0", "--workload", "cfg1"], env=e, capture_output=True, text=True, timeout=300)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    assert outs[0] == ""
    line = json.loads(outs[1].splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "events/s"
