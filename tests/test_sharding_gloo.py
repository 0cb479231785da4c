"""Multi-process (gloo, world size 2, CPU) test of the N > 1 path: replicas sharded with replica_offset, no data-path
collective, max-over-ranks timing, observables gathered in global replica order.  The compute stand-in is the oracle
(tests may call it); what is under test is the sharding logic bench.py uses on N GPUs."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2304_01772_b200 import sharding, workloads


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, batch, L, seed, n_sweeps, out_dir):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        off = sharding.replica_offset(rank, batch)
        beta = np.linspace(0.3, 0.6, batch)            # every rank runs the same recipe on its own replicas
        lat = oracle.init(batch, L, seed=seed, replica_offset=off)
        oracle.sweep(lat, beta, 1.0, 0.0, seed=seed, n_sweeps=n_sweeps, replica_offset=off)
        E, M = oracle.ising_observables(lat)
        Eg, Mg = sharding.gather_observables(torch.from_numpy(np.asarray(E, dtype=np.int64)),
                                             torch.from_numpy(np.asarray(M, dtype=np.int64)))
        slowest = sharding.max_over_ranks(10.0 + rank)
        sharding.barrier()
        if rank == 0:
            np.savez(os.path.join(out_dir, "gathered.npz"), E=Eg.numpy(), M=Mg.numpy(), slowest=slowest,
                     global_batch=sharding.global_batch(world, batch))
    finally:
        dist.destroy_process_group()


def test_two_ranks_equal_one_process(tmp_path, oracle_mod):
    world, batch, L, seed, n = 2, 3, 16, 21, 5
    mp.spawn(_worker, args=(world, _free_port(), batch, L, seed, n, str(tmp_path)), nprocs=world, join=True)
    got = np.load(tmp_path / "gathered.npz")
    assert int(got["global_batch"]) == world * batch
    assert float(got["slowest"]) == 11.0                      # max over ranks
    # the same replicas in one process: global replica g = rank * batch + b runs beta[b]
    beta = np.tile(np.linspace(0.3, 0.6, batch), world)
    lat = oracle_mod.init(world * batch, L, seed=seed)
    oracle_mod.sweep(lat, beta, 1.0, 0.0, seed=seed, n_sweeps=n)
    E, M = oracle_mod.ising_observables(lat)
    assert np.array_equal(got["E"], E) and np.array_equal(got["M"], M)


def test_offsets_partition_the_global_batch():
    for world, batch in [(1, 64), (2, 64), (4, 7), (8, 1024)]:
        seen = []
        for r in range(world):
            off = sharding.replica_offset(r, batch)
            seen.extend(range(off, off + batch))
        assert seen == list(range(sharding.global_batch(world, batch)))
    with pytest.raises(ValueError):
        sharding.replica_offset(-1, 4)
    assert sharding.max_over_ranks(3.5) == 3.5                # no process group: identity
    w = workloads.config(2)
    assert sharding.global_batch(8, w.batch) == 512
