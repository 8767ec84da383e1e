"""N > 1 path on CPU: two gloo ranks shard one batch, each computes its shard (the oracle stands in for the
kernels -- tests may call it), results are gathered in global order and the job reduction (max time, summed
counts) is checked.  The path has no data-path collective."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import sable_synth as S
from paper_2606_07099_b200.sharding import gather_rows, reduce_job, shard_range
from util import oracle_Y


def test_shard_range_partitions_exactly():
    for batch in (0, 1, 7, 64, 257):
        for world in (1, 2, 3, 8):
            cuts = [shard_range(batch, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == batch
            assert all(cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


def _worker(rank, world, port, batch, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    net = S.make_network(1)
    Y = oracle_Y(net)
    ps, qs, vs = S.make_scenarios(net, batch=batch)
    lo, hi = shard_range(batch, rank, world)
    res = oracle.nr_batch(Y, net.bus_type, ps[lo:hi], qs[lo:hi], vs[lo:hi], tol=1e-8, max_it=20, method=0, n_threads=1)
    vm = gather_rows(torch.from_numpy(res["vm"]), batch)
    it = gather_rows(torch.from_numpy(res["iterations"]), batch)
    secs, conv, solves = reduce_job(0.5 + rank, int(res["converged"].sum()), hi - lo)
    if rank == 0:
        q.put((vm.numpy(), it.numpy(), secs, conv, solves))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharded_solve_matches_single_process():
    batch, world = 13, 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, batch, q)) for r in range(world)]
    for p in procs:
        p.start()
    vm, it, secs, conv, solves = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    net = S.make_network(1)
    ps, qs, vs = S.make_scenarios(net, batch=batch)
    ref = oracle.nr_batch(oracle_Y(net), net.bus_type, ps, qs, vs, tol=1e-8, max_it=20, method=0)
    assert np.array_equal(vm, ref["vm"]) and np.array_equal(it, ref["iterations"])
    assert secs == 1.5 and conv == int(ref["converged"].sum()) and solves == batch
