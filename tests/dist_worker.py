"""Worker of tests/test_dist.py: one rank of a world-size-2 gloo job that goes through the N > 1 plumbing of
bench.py (paper_2601_14301_b200/dist.py): sharding, per-rank seeds, max-over-ranks timing, summed units."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import numpy as np

from paper_2601_14301_b200 import dist as D
from paper_2601_14301_b200 import inputs


def main():
    rank, local_rank, world = D.init("gloo")
    wl = inputs.WORKLOADS["cfg1"]
    lo, hi = D.shard_range(1001, rank, world)
    m = inputs.markers(wl, n=64, seed=D.rank_seed(wl.seed, rank))
    D.barrier()
    # rank r "processes" (r + 1) * 100 units in (r + 1) seconds and launches 3 + r kernels
    agg = D.aggregate((rank + 1) * 100.0, float(rank + 1), {"launches": 3 + rank})
    # row f1 across ranks: every rank projects its shard of the markers (here with the oracle, on the CPU), one all-reduce
    import oracle
    import torch
    o = oracle.from_workload(wl, inputs)
    o.set_modes(wl.modes)
    mm = inputs.markers(wl, n=1001, seed=77)
    part = torch.from_numpy(o.scatter(mm["R"][lo:hi], mm["Z"][lo:hi], mm["phi"][lo:hi], mm["vpar"][lo:hi]))
    total = D.allreduce_sum_(part.clone()).numpy()
    whole = o.scatter(mm["R"], mm["Z"], mm["phi"], mm["vpar"])
    scatter_err = float(np.abs(total - whole).max() / np.abs(whole).max())
    out = {"rank": rank, "scatter_err": scatter_err, "world": world, "lo": lo, "hi": hi, "agg": agg,
           "checksum": float(np.sum(m["R"])), "max_all": D.reduce_max(float(rank)), "sum_all": D.reduce_sum(float(rank))}
    with open(os.path.join(sys.argv[1], f"rank{rank}.json"), "w") as f:
        json.dump(out, f)
    D.barrier()


if __name__ == "__main__":
    main()
