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


def test_single_process_defaults():
    from paper_2607_06021_b200 import replicas as R
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert R.env_world() == (0, 0, 1)
    assert R.init("gloo") is None
    assert R.aggregate(None, 5.0, 7.0) == (5.0, 7.0)
