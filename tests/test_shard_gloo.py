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


# ------------------------------------------------------------------------------------------------ coupled ensemble (row f2)
def ens_count(cfg):
    """Doubles in the exchange buffer of a coupled ensemble (include/dns.h, dns_plan_set_exchange)."""
    return 2 * (3 * cfg.Ny * (cfg.Nz - 1) + cfg.Ny * (3 * cfg.Nz // 2))


def _coupled_worker(rank, world, port, E, q):
    """What a rank of a sharded coupled ensemble does at the exchange point of a stage, on the host: the sums over ITS
    members of the kx = 0 plane of the nonlinear vector go into the exchange buffer, shard.allreduce_sum_ (the callable
    the binding hands to dns_plan_set_exchange) sums it over the ranks, and the result is divided by E_total."""
    import torch
    import torch.distributed as dist
    from oracle.dns_oracle import Oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = inputs.Config(1, inputs.COUETTE, 400.0, 5.0, 3.0, 12, 13, 12, E, 0.02, 1, 0.2, 0, box=2)
    mine = shard.member_range(E, rank, world)
    st = inputs.make_state(cfg, mine)
    o = Oracle(*inputs.plan_args(cfg, E=len(mine)))
    o.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    Nu, Nv, Nw, _, _ = o.advection(o.v, o.eta, o.U, o.W)
    Nh = np.stack([o.to_spectral(f)[:, 0].sum(axis=0).T for f in (Nu, Nv, Nw)])      # [3][Ny][nkz] local sums
    buf = torch.zeros(ens_count(cfg), dtype=torch.float64)
    buf[:2 * Nh.size] = torch.from_numpy(np.ascontiguousarray(Nh).view(np.float64).ravel())
    shard.allreduce_sum_(buf)                                                         # the exchange step
    mean = (buf[:2 * Nh.size].numpy().view(np.complex128).reshape(Nh.shape)) / E
    if rank == 0:
        q.put(mean)
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_coupled_exchange_equals_the_unsharded_ensemble_mean():
    from oracle.dns_oracle import Oracle
    E = 5
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_coupled_worker, args=(r, 2, port, E, q)) for r in range(2)]
    for p in procs:
        p.start()
    mean = q.get(timeout=180)
    for p in procs:
        p.join(timeout=180)
        assert p.exitcode == 0
    cfg = inputs.Config(1, inputs.COUETTE, 400.0, 5.0, 3.0, 12, 13, 12, E, 0.02, 1, 0.2, 0, box=2)
    st = inputs.make_state(cfg)
    o = Oracle(*inputs.plan_args(cfg))
    o.set_state(st["vhat"], st["etahat"], st["U00"], st["W00"])
    Nu, Nv, Nw, _, _ = o.advection(o.v, o.eta, o.U, o.W)
    ref = np.stack([o.to_spectral(f)[:, 0].mean(axis=0).T for f in (Nu, Nv, Nw)])
    assert np.abs(mean - ref).max() < 1e-14 * np.abs(ref).max()
