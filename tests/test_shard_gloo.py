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
    mine = [shard.batch_index(s, r, w, 4, first=5) for s in range(4)]
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
    assert res[0][1] == [5, 6, 7, 8] and res[1][1] == [9, 10, 11, 12]   # contiguous per rank
    assert all(r[2] == 11.0 for r in res)              # max over ranks
    assert all(r[3] == 3.0 for r in res)               # sum over ranks


def test_single_process_defaults():
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert shard.world() == (0, 0, 1)
    assert shard.max_over_ranks(3.5) == 3.5
    assert [shard.batch_index(s, 0, 1, 3) for s in range(3)] == [0, 1, 2]
    assert not shard.under_torchrun()


def test_contiguous_ranges_partition_the_index_space():
    for world, per in ((1, 7), (2, 5), (8, 13)):
        seen = []
        for r in range(world):
            start, n = shard.batch_range(r, world, per, first=11)
            seen += list(range(start, start + n))
            assert [shard.batch_index(s, r, world, per, first=11) for s in range(per)] == list(range(start, start + n))
        assert seen == list(range(11, 11 + world * per))


def test_launch_cmd_is_the_contract_line():
    cmd = shard.launch_cmd(4, "bench.py", ["--gpus", "4", "--steps", "9"], 29123)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29123"
    assert cmd[-5:] == ["bench.py", "--gpus", "4", "--steps", "9"]


def test_spawner_starts_n_ranks(tmp_path):
    """`bench.py --gpus N` outside torchrun re-executes itself as N ranks through shard.respawn_under_torchrun; here the
    same spawner starts a 2-rank gloo job on the CPU."""
    import json
    worker = os.path.join(os.path.dirname(os.path.abspath(__file__)), "shard_worker.py")
    rc = shard.respawn_under_torchrun(2, worker, [str(tmp_path), "6"], require_gpus=False)
    assert rc == 0
    recs = [json.load(open(tmp_path / f"rank{r}.json")) for r in range(2)]
    assert [r["world"] for r in recs] == [2, 2]
    assert recs[0]["range"] == [3, 6] and recs[1]["range"] == [9, 6]
    assert all(r["max"] == 2.5 and r["sum"] == 2.0 for r in recs)


def test_spawner_refuses_more_ranks_than_devices():
    import pytest
    with pytest.raises(SystemExit):
        shard.respawn_under_torchrun(4096, "bench.py", [])          # no node has that many CUDA devices
