"""Event sharding of an MLEM iteration over the GPUs of one node.

The paper's CPU scheme - "each thread writes to its own copy of rho_new ... added at the end of the iteration"
 - lifted to devices: events are independent given w = s*rho, so every rank (one process per GPU) runs
jpet_mlem_begin + jpet_mlem_accumulate over its own shard into its private accumulator (<= 1 MB), the accumulators are
summed, and every rank runs the pointwise finalise.  Two ways to sum:

  "p2p"   the sum is fused into the finalise kernel: every rank maps its peers' accumulators once (cudaIpc handles
          exchanged through torch.distributed) and jpet_mlem_end_peers reads all of them over NVLink in rank order, so all
          ranks get bit-identical images.  Two host-side collectives per iteration order the accumulators' life cycle:
          an all-gather of the ranks' current handles once every accumulator is written (it is the "all written before any
          is read" barrier, and it makes the decision to re-map a peer the same on every rank - a rank whose workspace was
          re-allocated is seen by all the others, none waits alone in a collective), and a barrier after the finalise
          (all read before any is zeroed again).  Scaling beyond one GPU is unmeasured.
  "nccl"  one in-place NCCL all-reduce (sum) of the accumulator view, then the plain jpet_mlem_end.

This module only orchestrates calls of the C-ABI binding (or of another object with the same five methods: the
world-size-2 gloo test on CPU passes an engine built on the oracle); it does none of the method's arithmetic.
"""
from __future__ import annotations


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous shard [lo, hi) of n events for `rank` of `world`: sizes differ by at most one, shards tile [0, n)."""
    if world < 1 or not 0 <= rank < world or n < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, n >= 0")
    return n * rank // world, n * (rank + 1) // world


class _BindingEngine:
    """The CUDA path: the binding's calls on the current device and stream."""

    def __init__(self):
        import paper_1502_07478_b200 as jp

        self.jp = jp

    def begin(self, geom, rho_in):
        self.jp.jpet_mlem_begin(*geom, rho_in)

    def accumulate(self, events):
        self.jp.jpet_mlem_accumulate(events)

    def accumulator(self):
        return self.jp.jpet_mlem_accumulator()

    def end(self, rho_in, rho_out):
        self.jp.jpet_mlem_end(rho_in, rho_out)

    def end_peers(self, rho_in, rho_out, peers):
        self.jp.jpet_mlem_end_peers(rho_in, rho_out, peers)

    def sync(self):
        import torch

        torch.cuda.current_stream().synchronize()

    def ipc_export(self, acc) -> bytes:
        return self.jp.jpet_ipc_export(acc.data_ptr())

    def ipc_open(self, handle: bytes):
        return self.jp.jpet_ipc_open(handle)

    def ipc_close(self, peer) -> None:
        self.jp.jpet_ipc_close(peer)

    def own_peer(self, acc):
        return acc.data_ptr()


class ShardedMlem:
    """One MLEM iteration (Eq. 3) over events sharded across the ranks of a torch.distributed process group."""

    def __init__(self, dist=None, mode: str = "nccl", engine=None):
        if mode not in ("nccl", "p2p"):
            raise ValueError("mode must be 'nccl' or 'p2p'")
        self.dist = dist if (dist is not None and dist.is_initialized() and dist.get_world_size() > 1) else None
        self.world = self.dist.get_world_size() if self.dist else 1
        self.rank = self.dist.get_rank() if self.dist else 0
        self.mode = mode
        self.engine = engine if engine is not None else _BindingEngine()
        self._handles = None          # per rank: the handle its current mapping was opened from (own rank: exported)
        self._peers = None            # all ranks' accumulators in rank order: own pointer, peer mappings
        self._opened = {}             # rank -> mapping this process opened (and must close)

    # ---- peer mappings (p2p mode) ----------------------------------------------------------------------------------
    def _exchange_handles(self, acc):
        """Collective, every iteration: all ranks publish the handle of their current accumulator; every rank re-opens
        exactly the peers whose handle differs from the one its mapping came from.  Whether anything is re-mapped is thus
        decided from data all ranks share - a rank whose workspace was released and re-allocated (another pointer, or the
        same pointer with a new allocation behind it: the handle differs) cannot leave the others waiting in a collective
        it never enters, and no stale mapping survives.  Called after this rank's accumulator is complete, it is also the
        barrier before the peers' accumulators are read."""
        e = self.engine
        handles = [None] * self.world
        self.dist.all_gather_object(handles, e.ipc_export(acc))
        peers = []
        for r, h in enumerate(handles):
            if r == self.rank:
                peers.append(e.own_peer(acc))
                continue
            if self._handles is None or self._handles[r] != h:
                if r in self._opened:
                    e.ipc_close(self._opened.pop(r))
                self._opened[r] = e.ipc_open(h)
            peers.append(self._opened[r])
        self._handles, self._peers = handles, peers

    def close(self):
        for p in self._opened.values():
            self.engine.ipc_close(p)
        self._opened, self._peers, self._handles = {}, None, None

    # ---- the iteration ---------------------------------------------------------------------------------------------
    def iterate(self, events_shard, geom, rho_in, rho_out):
        """events_shard: this rank's events [n_r, 3]; geom = (R, L, sigma_z, sigma_dl, n_y, n_z, pixel); rho_in must hold the
        same image on every rank; rho_out receives the same image on every rank."""
        e = self.engine
        e.begin(geom, rho_in)
        e.accumulate(events_shard)
        if self.world == 1:
            e.end(rho_in, rho_out)
        elif self.mode == "nccl":
            self.dist.all_reduce(e.accumulator(), op=self.dist.ReduceOp.SUM)
            e.end(rho_in, rho_out)
        else:
            e.sync()                          # this rank's accumulator is complete ...
            self._exchange_handles(e.accumulator())      # ... and, past this collective, so is every other rank's
            e.end_peers(rho_in, rho_out, self._peers)
            e.sync()
            self.dist.barrier()               # every rank has read every accumulator: the next begin may zero them
        return rho_out

    def reconstruct(self, events_shard, geom, rho_init, rho_out, n_iter: int):
        """n_iter sharded iterations; rho_init and rho_out may be the same tensor."""
        cur = rho_init
        for _ in range(n_iter):
            self.iterate(events_shard, geom, cur, rho_out)
            cur = rho_out
        if n_iter == 0 and rho_out is not rho_init:
            rho_out.copy_(rho_init)
        return rho_out
