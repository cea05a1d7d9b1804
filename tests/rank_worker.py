"""Worker of tests/test_multirank.py: one of WORLD_SIZE processes on the CPU (gloo), launched by torchrun.

Exercises the host logic of bench.py's N > 1 path without a GPU: rank environment, an independent replica
per rank (own seed, no data-path collective), barrier, max-over-ranks timing, whole-job rate, rank 0 reports.
"""
import json
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import bench  # noqa: E402


def main():
    out_dir = sys.argv[1]
    world, rank, local = bench.rank_env()
    dist.init_process_group("gloo")
    assert dist.get_world_size() == world and dist.get_rank() == rank
    c = bench._workload(2048, rank, 3)                 # this rank's replica of the workload recipe
    fake_ms = 10.0 * (rank + 1)                        # stands in for this rank's device-side time
    dist.barrier()
    ms = bench.max_over_ranks(fake_ms, world, torch.device("cpu"))
    rate = bench.job_rate(world, c["N"], ms)
    # target sharding: one common ensemble, every rank owns N / world rows and gathers the rest
    import paper_1212_2934_b200 as ff            # import only: no library call, no GPU
    common = bench._workload(2048, 0, 3)
    full = torch.from_numpy(common["pos"])
    n_loc = common["N"] // world
    mine = full[rank * n_loc:(rank + 1) * n_loc].clone()
    gathered = bench.gather_particles(mine, world)
    gb, ge = ff.shard_groups(common["N"], world, rank)
    rec = {"rank": rank, "world": world, "local": local, "ms": ms, "rate": rate, "N": c["N"],
           "pos_sum": float(np.asarray(c["pos"], np.float64).sum()),
           "gather_ok": bool(torch.equal(gathered, full)), "groups": [gb, ge]}
    with open(os.path.join(out_dir, "rank%d.json" % rank), "w") as fh:
        json.dump(rec, fh)
    if rank == 0:
        print(json.dumps({"value": rate, "n_gpus": world}))
    dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
