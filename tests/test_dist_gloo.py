"""N > 1 path on the CPU: two gloo ranks shard the batch with no data-path collective; only the barrier and the
max-over-ranks / sum-over-ranks reductions of bench.py communicate."""
import os
import socket

import pytest
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_items, q):
    import torch.distributed as dist
    from paper_2307_12585_b200 import dist as fdist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert fdist.env_world() == (rank, world, rank)
        mine = fdist.shard_range(n_items, world, rank)
        fdist.barrier()
        ms = 10.0 + 5.0 * rank                       # stand-in for this rank's device time
        worst = fdist.max_over_ranks(ms)
        total = fdist.sum_over_ranks(len(mine))
        q.put((rank, list(mine), worst, total))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_items", [1024, 7, 1])
def test_two_ranks_partition_and_reduce(n_items):
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_items, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    items = out[0][1] + out[1][1]
    assert items == list(range(n_items))                          # ordered partition, nothing lost or doubled
    assert abs(len(out[0][1]) - len(out[1][1])) <= 1
    assert all(o[2] == 15.0 for o in out)                         # max over ranks
    assert all(o[3] == float(n_items) for o in out)               # whole-job units


def test_shard_range_properties():
    from paper_2307_12585_b200.dist import shard_range
    for n in (0, 1, 5, 1024):
        for world in (1, 2, 3, 8):
            parts = [list(shard_range(n, world, r)) for r in range(world)]
            assert sum(parts, []) == list(range(n))
            assert max(map(len, parts)) - min(map(len, parts)) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)
