"""Worker of test_world_size_2_sharding_over_gloo: the N>1 logic of bench.py on CPU (gloo)."""
import os
import sys

import torch
import torch.distributed as dist

sys.path.insert(0, os.environ["PHS_ROOT"])
import bench  # noqa: E402

dist.init_process_group("gloo")
r, n = dist.get_rank(), dist.get_world_size()
mine = bench.shard_instances(64 * n + 1, r, n)
assert mine == list(range(mine[0], mine[0] + len(mine))), "blocks must be contiguous (seed = instance index)"
cnt = torch.tensor([len(mine)], dtype=torch.int64)
dist.all_reduce(cnt)
ms = torch.tensor([10.0 + r], dtype=torch.float64)
dist.all_reduce(ms, op=dist.ReduceOp.MAX)
allm = [None] * n
dist.all_gather_object(allm, mine)
assert sorted(sum(allm, [])) == list(range(64 * n + 1))
assert cnt.item() == 64 * n + 1 and ms.item() == 10.0 + n - 1
# each rank builds the host tables of ITS block only; seeds follow the global instance index
from paper_2505_01616_b200 import binding as B  # noqa: E402
from paper_2505_01616_b200 import workloads as W  # noqa: E402
w = W.cfg3(batch=2 * n)
blk = bench.shard_instances(w.batch, r, n)
sim = B.Sim.from_workload(w, instances=(blk[0], len(blk)))
ref = B.Sim.from_workload(w)
for i, g in enumerate(blk):
    assert all((a == b).all() for a, b in zip(sim.paths(i), ref.paths(g)))
dist.destroy_process_group()
print("ok", r)
