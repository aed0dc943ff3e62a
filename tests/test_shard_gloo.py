"""Multi-rank host logic on CPU (gloo, world_size 2): member sharding needs no data-path collective; the
diagnostic gather and the max-over-ranks timing reduction are the only exchanges."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

from paper_2306_12739_b200 import inputs, shard


def test_member_range_partitions():
    for E in (1, 2, 5, 16, 64, 257):
        for world in (1, 2, 3, 4, 8):
            got = [m for r in range(world) for m in shard.member_range(E, r, world)]
            assert got == list(range(E))
            sizes = [len(shard.member_range(E, r, world)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.member_range(4, 2, 2)


def _worker(rank, world, port, E, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = inputs.CONFIGS[1].with_E(E)
    mine = shard.member_range(E, rank, world)
    st = inputs.make_state(cfg, mine)                 # every rank generates only its own members
    rows = np.stack([np.full(6, float(e)) + np.arange(6) * 0.01 for e in mine]) if len(mine) else np.zeros((0, 6))
    allrows = shard.gather_rows(rows, E, 6)
    tmax = shard.max_over_ranks(1.0 + rank)
    if rank == 0:
        q.put((allrows, tmax, st["vhat"].shape[0]))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("E", [5, 8])
def test_two_rank_gather(E):
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, E, q)) for r in range(2)]
    for p in procs:
        p.start()
    allrows, tmax, n0 = q.get(timeout=120)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert allrows.shape == (E, 6)
    assert np.allclose(allrows[:, 0], np.arange(E)) and np.allclose(allrows[:, 5], np.arange(E) + 0.05)
    assert tmax == 2.0
    assert n0 == len(shard.member_range(E, 0, 2))


def test_sharded_members_equal_unsharded_inputs():
    cfg = inputs.CONFIGS[1].with_E(5)
    full = inputs.make_state(cfg)
    parts = [inputs.make_state(cfg, shard.member_range(5, r, 2)) for r in range(2)]
    assert np.array_equal(np.concatenate([p["vhat"] for p in parts]), full["vhat"])
