"""Bunch sharding: the host logic that needs no GPU -- the partition of the fill over the ranks
(mbt_shard_range), the layout of the exchange buffer, and, over a world_size-2 gloo group, that the all-gather of the
ranks' source phasors rebuilds the single-rank array, so that the per-bunch phasor gather of DESIGN.md 7.2 -- written
out here in numpy -- gives every rank the phasors P[b][r] of its bunches bit for bit as a single rank computes them."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_range_partitions_the_fill():
    from paper_1809_00391_b200 import build, mbt
    build.build()
    for m in (1, 2, 3, 5, 22, 363, 484, 1000):
        for world in (1, 2, 3, 4, 7, 8):
            chunk = -(-m // world)
            seen = []
            for rank in range(world):
                first, count = mbt.shard_range(m, world, rank)
                assert first == min(rank * chunk, m) and 0 <= count <= chunk
                seen += list(range(first, first + count))
            assert seen == list(range(m))                       # every bunch exactly once, in order
            assert mbt.shard_exchange_doubles(m, world, 3) == world * chunk * 3 * 2
    with pytest.raises(mbt.MbtError):
        mbt.shard_range(5, 2, 2)
    from paper_1809_00391_b200 import sharded
    assert sharded.exchange_layout(363, 8, 2) == (46, 46 * 2 * 2, 8 * 46 * 2 * 2)


def _phasors(a, buckets, lam, t_rf, first, count):
    """P[b][r] = sum_{j < b} a[j][r] exp(lam_r (s_b - s_j) T_rf) for the bunches [first, first + count) (no history)."""
    out = np.zeros((count, a.shape[1]), dtype=np.complex128)
    for i in range(count):
        b = first + i
        for j in range(b):                                       # fixed order: bit-identical wherever it is evaluated
            out[i] += a[j] * np.exp(lam * ((buckets[b] - buckets[j]) * t_rf))
    return out


def _rank_main(rank, world, port, m, n_lr, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1809_00391_b200 import mbt, sharded
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(7)                                # the same on every rank: the single-rank truth
    a_all = rng.standard_normal((m, n_lr)) + 1j * rng.standard_normal((m, n_lr))
    buckets = np.sort(rng.choice(484, size=m, replace=False))
    lam = -1.0e6 * (1 + np.arange(n_lr)) + 1j * 7.5e9 * (1 + np.arange(n_lr))
    rows, per_rank, total = sharded.exchange_layout(m, world, n_lr)
    first, count = mbt.shard_range(m, world, rank)
    buf = torch.zeros(total, dtype=torch.float64)
    own = buf[rank * per_rank:(rank + 1) * per_rank]
    mine = np.zeros((rows, n_lr, 2))
    mine[:count, :, 0] = a_all[first:first + count].real          # what mbt_shard_turn_begin writes: this rank's rows
    mine[:count, :, 1] = a_all[first:first + count].imag
    own.copy_(torch.from_numpy(mine.ravel()))
    dist.all_gather_into_tensor(buf, own.clone())                 # the collective of ShardedTracker.track
    g = buf.numpy().reshape(world * rows, n_lr, 2)
    a_gathered = g[:m, :, 0] + 1j * g[:m, :, 1]
    ok_layout = bool(np.array_equal(a_gathered, a_all))           # global row j of the buffer is bunch j
    p_sharded = _phasors(a_gathered, buckets, lam, 2.0e-9, first, count)
    p_single = _phasors(a_all, buckets, lam, 2.0e-9, 0, m)[first:first + count]
    q.put((rank, ok_layout, bool(np.array_equal(p_sharded, p_single)), count))
    dist.destroy_process_group()


@pytest.mark.parametrize("m,n_lr", [(5, 2), (363, 2), (484, 3)])
def test_gloo_world2_exchange_rebuilds_single_rank_phasors(m, n_lr):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    import socket
    with socket.socket() as sk:                                   # a free port of this host
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, m, n_lr, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == [0, 1]
    assert all(r[1] and r[2] for r in res), res
    assert sum(r[3] for r in res) == m
