"""Host-side logic of the N > 1 bench path (replicas only, no data-path
collective): every rank times its own replica, the job value is the particles of ALL ranks divided
by the MAX over ranks of the time.  Covered here with two gloo ranks on CPU."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import bench


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rmax, rsum = bench.make_reducers(world, torch.device("cpu"))
    ms_local, n_local = (100.0, 1000) if rank == 0 else (250.0, 3000)      # the slow rank sets the time
    ms, total = bench.aggregate(ms_local, n_local, world, rmax, rsum)
    launches = rsum(7 + rank)
    q.put((rank, ms, total, launches))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregation_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, total, launches in got:
        assert ms == 250.0 and total == 4000.0 and launches == 15.0
    # whole-job value: units of all ranks / max time
    evals = 2 * 5
    assert got[0][2] * evals / (got[0][1] * 1e-3) == pytest.approx(4000 * 10 / 0.25)


def test_single_rank_reducers_are_identity():
    rmax, rsum = bench.make_reducers(1, None)
    assert bench.aggregate(12.5, 42, 1, rmax, rsum) == (12.5, 42.0)
