"""N > 1 path of bench.py on CPU: two gloo ranks run the timing protocol (barrier, max over ranks of the elapsed time,
sum over ranks of the units processed) that the replicas use; there is no data-path collective to test."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2607_06021_b200 import replicas as R
    assert R.env_world() == (rank, rank, world)
    dist = R.init("gloo")
    R.barrier(dist)
    local_ms = 10.0 * (rank + 1)              # rank 1 is the slow one
    units = 100.0 + rank
    agg = R.throughput(dist, local_ms, units)
    R.barrier(dist)
    # a batch of 5 independent problems split over the ranks; per-problem integers collected in problem order
    lo, hi = R.shard(5, rank, world)
    agg["shard"] = (lo, hi)
    agg["ranks_of_batch"] = R.gather_ints(dist, [100 * rank + p for p in range(lo, hi)], 5)
    q.put((rank, agg))
    dist.destroy_process_group()


def test_two_rank_aggregate_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        assert res[r]["ms"] == 20.0                       # max over ranks
        assert res[r]["units"] == 201.0                   # whole-job units
        assert abs(res[r]["per_s"] - 201.0 / 0.020) < 1e-9
        assert res[r]["ranks_of_batch"] == [0, 1, 2, 103, 104]     # rank 0 solved problems 0-2, rank 1 problems 3-4
    assert res[0]["shard"] == (0, 3) and res[1]["shard"] == (3, 5)


def test_shard_covers_every_problem_once():
    from paper_2607_06021_b200 import replicas as R
    for nprob in (0, 1, 2, 7, 8, 64, 1000):
        for world in (1, 2, 3, 8):
            blocks = [R.shard(nprob, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == nprob
            assert all(blocks[r][1] == blocks[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in blocks]
            assert max(sizes) - min(sizes) <= 1
    assert R.gather_ints(None, [4, 5], 2) == [4, 5]


def test_single_process_defaults():
    from paper_2607_06021_b200 import replicas as R
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert R.env_world() == (0, 0, 1)
    assert R.init("gloo") is None
    assert R.aggregate(None, 5.0, 7.0) == (5.0, 7.0)
