"""Event sharding over ranks, host side, on CPU: the partition of the event list and the
orchestration of paper_1502_07478_b200.sharding.ShardedMlem (begin / accumulate per rank, one sum all-reduce of the
accumulator, finalise on every rank) run as two gloo processes.  The CUDA kernels cannot run here, so the per-rank
engine is a stand-in built on the oracle (test infrastructure); what is under test is the sharding logic - that the
shards tile the events, that the collective touches the right buffer, and that every rank ends with the image one
process computes over all events.  The device side of the same path is tests/test_round2_gpu.py."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shards_tile_the_event_list():
    from paper_1502_07478_b200.sharding import shard_range

    for n in (0, 1, 7, 100, 10_000_019):
        for world in (1, 2, 3, 8):
            cuts = [shard_range(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


class OracleEngine:
    """CPU stand-in for the binding: the accumulator of Eq. 3, acc(i) = sum_j P(e_j|i) / denominator_j, recovered from the
    oracle's iteration on rho_in (rho_out = rho_in * acc where s > 0)."""

    def __init__(self, oracle):
        import torch

        self.oracle, self.torch = oracle, torch

    def begin(self, geom, rho_in):
        self.geom, self.rho_in = geom, rho_in.numpy().astype(np.float64)
        n_y, n_z = geom[4], geom[5]
        self.acc = self.torch.zeros(n_y * n_z, dtype=self.torch.float64)

    def accumulate(self, events):
        out, _, _ = self.oracle.mlem_iterate(events.numpy(), *self.geom, self.rho_in.reshape(self.geom[4], self.geom[5]))
        r = self.rho_in.ravel()            # where rho_in = 0 the accumulator does not matter (rho_out = 0 there)
        self.acc += self.torch.from_numpy(np.divide(out.ravel(), r, out=np.zeros_like(r), where=r > 0))

    def accumulator(self):
        return self.acc

    def end(self, rho_in, rho_out):
        rho_out.copy_(rho_in.double() * self.acc)

    def sync(self):
        pass


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    import oracle
    from paper_1502_07478_b200 import synth
    from paper_1502_07478_b200.sharding import ShardedMlem, shard_range

    dist.init_process_group("gloo")
    cfg = synth.CONFIGS["cfg1"]
    geom = (cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel)
    events = synth.config_events(cfg, n=3001)                       # every rank draws the same list and takes its shard
    lo, hi = shard_range(len(events), rank, world)
    sm = ShardedMlem(dist, mode="nccl", engine=OracleEngine(oracle))     # "nccl" = all-reduce of the accumulator (gloo here)
    rho = torch.ones(cfg.n_y * cfg.n_z, dtype=torch.float64)
    out = torch.empty_like(rho)
    sm.reconstruct(torch.from_numpy(events[lo:hi]), geom, rho, out, 2)
    dist.destroy_process_group()
    return rank, lo, hi, out.numpy().reshape(cfg.n_y, cfg.n_z)


def _entry(rank, world, port, q):
    q.put(_worker(rank, world, port))


def test_two_ranks_reconstruct_what_one_process_does(oracle):
    import torch.multiprocessing as mp

    from paper_1502_07478_b200 import synth

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_entry, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg = synth.CONFIGS["cfg1"]
    events = synth.config_events(cfg, n=3001)
    want, _, _ = oracle.reconstruct(events, cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel, 2)
    assert (got[0][1], got[0][2], got[1][1], got[1][2]) == (0, 1500, 1500, 3001)
    for _, _, _, img in got:
        assert np.max(np.abs(img - want)) <= 1e-12 * want.max()
    assert (got[0][3] == got[1][3]).all()                            # every rank holds the same image


def test_single_rank_needs_no_process_group(oracle):
    import torch

    from paper_1502_07478_b200 import synth
    from paper_1502_07478_b200.sharding import ShardedMlem

    cfg = synth.CONFIGS["cfg1"]
    geom = (cfg.R, cfg.L, cfg.sigma_z, cfg.sigma_dl, cfg.n_y, cfg.n_z, cfg.pixel)
    events = synth.config_events(cfg, n=500)
    sm = ShardedMlem(None, engine=OracleEngine(oracle))
    assert (sm.world, sm.rank) == (1, 0)
    rho = torch.ones(cfg.n_y * cfg.n_z, dtype=torch.float64)
    out = sm.iterate(torch.from_numpy(events), geom, rho, torch.empty_like(rho))
    want, _, _ = oracle.mlem_iterate(events, *geom, np.ones((cfg.n_y, cfg.n_z)))
    assert np.max(np.abs(out.numpy().reshape(cfg.n_y, cfg.n_z) - want)) <= 1e-12 * want.max()


# ---- p2p mode: the decision to re-map a peer is taken from data every rank has -------------------------
class HandleEngine:
    """Stand-in for the cudaIpc side of the p2p mode: a "handle" names (rank, allocation generation); opening one gives a
    token.  Records what ShardedMlem opens, closes and passes to the finalise."""

    def __init__(self, rank):
        self.rank, self.generation, self.log, self.finalised_with = rank, 0, [], []

    def begin(self, geom, rho_in):
        pass

    def accumulate(self, events):
        pass

    def accumulator(self):
        return ("acc", self.rank, self.generation)

    def sync(self):
        pass

    def ipc_export(self, acc):
        return b"%d:%d" % (acc[1], acc[2])

    def ipc_open(self, handle):
        self.log.append(("open", handle))
        return ("mapped", handle)

    def ipc_close(self, peer):
        self.log.append(("close", peer[1]))

    def own_peer(self, acc):
        return acc

    def end_peers(self, rho_in, rho_out, peers):
        self.finalised_with.append(list(peers))


def _remap_worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist

    from paper_1502_07478_b200.sharding import ShardedMlem

    dist.init_process_group("gloo")
    eng = HandleEngine(rank)
    sm = ShardedMlem(dist, mode="p2p", engine=eng)
    for it in range(4):
        if it == 2 and rank == 1:
            eng.generation = 1          # rank 1 alone lost its workspace (jpet_release, a grown grid) between iterations
        sm.iterate(None, None, None, None)
    sm.close()
    dist.destroy_process_group()
    q.put((rank, eng.log, eng.finalised_with))


def test_p2p_remap_is_decided_collectively():
    """Rank 1's accumulator is re-allocated after two iterations, rank 0's is not.  Both must keep entering the same
    collectives (no hang), rank 0 must drop its stale mapping of rank 1 and open the new one exactly once, and rank 1 must
    not re-open rank 0's."""
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_remap_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=120) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, log0, fin0), (_, log1, fin1) = got
    assert log0 == [("open", b"1:0"), ("close", b"1:0"), ("open", b"1:1"), ("close", b"1:1")]
    assert log1 == [("open", b"0:0"), ("close", b"0:0")]
    assert fin0 == [[("acc", 0, 0), ("mapped", b"1:0")]] * 2 + [[("acc", 0, 0), ("mapped", b"1:1")]] * 2
    assert fin1 == [[("mapped", b"0:0"), ("acc", 1, 0)]] * 2 + [[("mapped", b"0:0"), ("acc", 1, 1)]] * 2
