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
    # the moments travel while the tree is built: begin / end pair around independent work
    mom_full = torch.from_numpy(common["mom"])
    pending = bench.gather_particles_begin(mom_full[rank * n_loc:(rank + 1) * n_loc].clone(), world)
    busy = float(gathered.double().sum())                        # stands in for ff_build_tree(p_all)
    mom_gathered = bench.gather_particles_end(pending)
    gb, ge = ff.shard_groups(common["N"], world, rank)
    gb64, ge64 = ff.shard_groups(common["N"], world, rank, 64)
    # the "strong" block of the JSON line from (fake) device times: one GPU 20 ms, sharded step 12.5 ms
    strong = bench.strong_block(world, common["N"], 20.0, bench.max_over_ranks(12.5 - rank, world, torch.device("cpu")),
                                0.5, 9.0, {"walk": 9.0})
    rec = {"rank": rank, "world": world, "local": local, "ms": ms, "rate": rate, "N": c["N"],
           "pos_sum": float(np.asarray(c["pos"], np.float64).sum()),
           "gather_ok": bool(torch.equal(gathered, full)) and bool(torch.equal(mom_gathered, mom_full)) and busy == busy,
           "groups": [gb, ge], "groups64": [gb64, ge64], "strong": strong}
    with open(os.path.join(out_dir, "rank%d.json" % rank), "w") as fh:
        json.dump(rec, fh)
    if rank == 0:
        print(json.dumps({"value": rate, "n_gpus": world, "scaling": "weak", "strong": strong}))
    dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
