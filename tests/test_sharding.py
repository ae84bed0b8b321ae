"""N > 1: energies are sharded over ranks with no data-path collective.
Covered on CPU with a world_size-2 gloo group: the shards are disjoint, equally sized, their union is
one uniform grid, and the per-rank quadrature weights sum to the dense trapezoid rule, so that an
all-reduce of per-rank densities equals the single-rank density of the dense grid."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2602_03438_b200 import workloads as W


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = W.shard_energies(W.make_workload(1, n_blocks=3, block_size=4, n_energy=6), rank, world)
    e = torch.from_numpy(wl.energies.copy())
    w = torch.from_numpy(wl.weights.copy())
    es = [torch.empty_like(e) for _ in range(world)]
    dist.all_gather(es, e)
    # stand-in for the density all-reduce: sum_E w_E f(E) with f = E^2 + 1 over the local shard
    part = (w * (e ** 2 + 1)).sum().reshape(1)
    dist.all_reduce(part)
    if rank == 0:
        q.put((torch.stack(es).numpy(), float(part)))
    dist.barrier()
    dist.destroy_process_group()


def test_energy_sharding_world2_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    shards, total = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert shards.shape == (2, 6)
    union = np.sort(shards.reshape(-1))
    assert np.allclose(union, np.linspace(-1.0, 1.0, 12))
    assert len(np.unique(union)) == 12
    dense = np.linspace(-1.0, 1.0, 12)
    ref = float((W.trapezoid_weights(dense) * (dense ** 2 + 1)).sum())
    assert abs(total - ref) < 1e-13


def test_single_rank_is_identity():
    wl = W.make_workload(0)
    assert W.shard_energies(wl, 0, 1) is wl
