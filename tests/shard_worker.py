"""Rank body of tests/test_shard_gloo.py::test_spawner_starts_n_ranks (run under torchrun by shard.respawn_under_torchrun)."""
import json
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2104_12922_b200 import shard  # noqa: E402

if __name__ == "__main__":
    out_dir, per_rank = sys.argv[1], int(sys.argv[2])
    assert shard.under_torchrun()
    r, lr, w = shard.init("gloo")
    shard.barrier()
    rec = {"rank": r, "world": w, "range": list(shard.batch_range(r, w, per_rank, first=3)),
           "max": shard.max_over_ranks(1.5 + r), "sum": shard.sum_over_ranks(1.0)}
    with open(os.path.join(out_dir, f"rank{r}.json"), "w") as f:
        json.dump(rec, f)
    shard.barrier()
    import torch.distributed as dist
    if dist.is_initialized():
        dist.destroy_process_group()
