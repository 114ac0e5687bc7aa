"""N>1 host logic on CPU: world_size-2 gloo run of the sharding and max-over-ranks timing helpers."""
import os
import socket

import torch.multiprocessing as mp

from paper_2104_12922_b200 import shard


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, ws, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(ws), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    r, lr, w = shard.init("gloo")
    shard.barrier()
    mine = [shard.batch_index(s, r, w, first=5) for s in range(4)]
    mx = shard.max_over_ranks(10.0 + r)
    sm = shard.sum_over_ranks(1.0 + r)
    shard.barrier()
    q.put((r, mine, mx, sm))
    import torch.distributed as dist
    dist.destroy_process_group()


def test_two_rank_sharding_and_timing_reduction():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    idx = res[0][1] + res[1][1]
    assert sorted(idx) == list(range(5, 13))          # disjoint and dense over ranks and steps
    assert all(r[2] == 11.0 for r in res)              # max over ranks
    assert all(r[3] == 3.0 for r in res)               # sum over ranks


def test_single_process_defaults():
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert shard.world() == (0, 0, 1)
    assert shard.max_over_ranks(3.5) == 3.5
    assert [shard.batch_index(s, 0, 1) for s in range(3)] == [0, 1, 2]
