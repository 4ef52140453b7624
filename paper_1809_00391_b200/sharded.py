"""Bunch-sharded tracking over several GPUs (mbt_shard in include/mbt.h): opt-in, one process per
GPU, torch.distributed for the one collective a turn needs.  PLUMBING ONLY: every step of the method runs in the library's
kernels; this module allocates the exchange buffer (a torch tensor), and per turn calls

    mbt_shard_turn_begin  ->  all_gather_into_tensor(exchange)  ->  mbt_shard_turn_end

on one CUDA stream.  The default path of the repository is one GPU (BASELINE north_star: "no sharding, no collectives").

Validation status: the turn halves are checked on one GPU with the all-gather EMULATED by copies (tests/test_gpu_sharded.py)
and the partition / layout logic over two gloo ranks on CPU (tests/test_shard_host.py).  The in-place NCCL
all_gather_into_tensor below has not yet run on more than one GPU (no multi-GPU box was available to this build).
"""
from __future__ import annotations

from . import mbt


def exchange_layout(n_bunches: int, world: int, n_lr: int):
    """(rows per rank, doubles per rank, doubles in all): rank r's source phasors a[b][r'] of its bunches
    [r * rows, r * rows + count) sit in its chunk of the buffer; rows beyond the fill are padding."""
    rows = -(-n_bunches // world)
    per_rank = rows * n_lr * 2
    return rows, per_rank, world * per_rank


class ShardedTracker:
    """One rank of a bunch-sharded run.  `group`: a torch.distributed process group (None: the default one);
    collectives run on the current CUDA stream, which is also the stream the library enqueues on."""

    def __init__(self, cfg, rank=None, world=None, group=None, device=None, log_capacity_turns=0, all_gather=None):
        import torch
        import torch.distributed as dist
        self._torch, self._dist, self._group = torch, dist, group
        self.rank = dist.get_rank(group) if rank is None else int(rank)
        self.world = dist.get_world_size(group) if world is None else int(world)
        if device is None:
            device = torch.cuda.current_device()
        self.device = torch.device("cuda", device)
        n_lr = sum(1 for r in cfg["wake"]["resonators"] if r["flags"] & 2)
        m = len(cfg["fill"]["buckets"])
        self.rows, self.per_rank, total = exchange_layout(m, self.world, n_lr)
        assert total == mbt.shard_exchange_doubles(m, self.world, n_lr)
        self.stream = torch.cuda.Stream(self.device)   # the library's kernels and the collective are ordered on this stream
        # The exchange buffer is zero-filled ON that stream: torch streams do not wait for the default stream, so a fill
        # enqueued there could land after the first turn's source phasors had been written.
        with torch.cuda.stream(self.stream):
            self.exchange = torch.zeros(max(total, 2), dtype=torch.float64, device=self.device)
        self._own = self.exchange[self.rank * self.per_rank:(self.rank + 1) * self.per_rank]
        self._all_gather = all_gather   # test hook: a callable(exchange tensor, own slice) replacing the collective
        self.tracker = mbt.Tracker(cfg, log_capacity_turns=log_capacity_turns, stream=self.stream.cuda_stream, device=device,
                                   shard=dict(rank=self.rank, world=self.world, d_exchange=self.exchange.data_ptr() if n_lr else None))
        self.n_lr = n_lr

    def track(self, n_turns: int):
        with self._torch.cuda.stream(self.stream):
            for _ in range(int(n_turns)):
                self.tracker.shard_turn_begin()
                if self.n_lr and self.world > 1:
                    if self._all_gather is not None:
                        self._all_gather(self.exchange, self._own)
                    else:   # in place: this rank's chunk of the output is its input
                        self._dist.all_gather_into_tensor(self.exchange[:self.world * self.per_rank], self._own, group=self._group)
                self.tracker.shard_turn_end()

    def close(self):
        self.tracker.close()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()
