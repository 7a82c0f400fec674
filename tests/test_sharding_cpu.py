"""Host-side logic of the Morton-range sharding (include/sph.h "sharding"), on CPU:
the partition (sph_partition: host only, no device call) and the in-place all-gather the binding hands to the library
(paper_1604_03290_b200.all_gather_slices), run by two and three gloo ranks on CPU tensors laid out like the library's
rate arrays.  The kernels of the sharded path are covered on the GPU by tests/test_gpu_parity.py::test_sharded_*."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import paper_1604_03290_b200 as P


@pytest.mark.parametrize("n,world", [(100, 3), (3_999_794, 8), (64, 4), (33, 2), (5, 8), (4416, 2), (65_536, 64)])
def test_partition_covers_the_sorted_order_in_warp_aligned_slices(n, world):
    parts = [P.sph_partition(n, world, r) for r in range(world)]
    slices = {sl for _, _, sl in parts}
    assert len(slices) == 1
    sl = slices.pop()
    assert sl % 32 == 0 and sl * world >= n and sl * world <= n + 32 * world      # fits the padded rate arrays
    assert parts[0][0] == 0 and parts[-1][1] == n
    for r, (lo, hi, _) in enumerate(parts):
        assert lo == min(n, r * sl) and lo <= hi <= n
        assert (lo % 32 == 0 or lo == n) and (hi % 32 == 0 or hi == n)                         # warp groups never straddle two ranks
        if r:
            assert lo == parts[r - 1][1]                                          # contiguous, disjoint
    with pytest.raises(P.SphError):
        P.sph_partition(n, world, world)
    with pytest.raises(P.SphError):
        P.sph_partition(n, 65, 0)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, n, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi, sl = P.sph_partition(n, world, rank)
    # two "rate arrays" as the library lays them out: world * slice elements, FP64 and int32, every rank fills its own slice
    full_d = np.arange(world * sl, dtype=np.float64) * 0.5 + 1.0
    full_i = np.arange(world * sl, dtype=np.int32) * 3 - 7
    d = np.full(world * sl, np.nan)
    i = np.full(world * sl, -1, np.int32)
    d[rank * sl:rank * sl + (hi - lo)] = full_d[lo:hi]
    i[rank * sl:rank * sl + (hi - lo)] = full_i[lo:hi]
    td, ti = torch.from_numpy(d).view(torch.uint8), torch.from_numpy(i).view(torch.uint8)
    P.all_gather_slices([td, ti], [8 * sl, 4 * sl], rank)
    ok = bool(np.array_equal(d[:n], full_d[:n]) and np.array_equal(i[:n], full_i[:n]))
    q.put((rank, ok, lo, hi))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,n", [(2, 1000), (3, 4416)])
def test_all_gather_of_rate_slices_gloo(world, n):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_main, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok for _, ok, _, _ in got)
    assert got[0][2] == 0 and got[-1][3] == n
