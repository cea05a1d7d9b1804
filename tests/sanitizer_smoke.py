"""Smoke-sized pass over every kernel of libff.so, meant to be run under compute-sanitizer:

    compute-sanitizer --tool memcheck  python tests/sanitizer_smoke.py
    compute-sanitizer --tool racecheck python tests/sanitizer_smoke.py

or, where compute-sanitizer is not available, against the CHECKED build of the library (every kernel compiled with its
device-side index and bound checks, FF_CHECK in csrc/ff_internal.cuh; a failed check makes the next ff_get_timings /
ff_get_counters call return FF_ERR_CHECK with the source line):

    FF_CHECKED=1 python tests/sanitizer_smoke.py

Covers ff_build_tree, ff_eval_bh (N_leaf 1, 2 and 4, ragged N, counters on and off, W = 32 and 64, cell order 0 and 1),
ff_eval_bh_range,
ff_eval_direct (split and unsplit grids), ff_eval_bh_host and ff_step with Lennard-Jones pairs + walls, Barnes-Hut
and all-pairs.  The hazards it is there for: the walk's shared-memory ring, stack and parked-cell queue are ordered
by __syncwarp only, the sort's look-back by volatile status words (the paper's own build relies on atomics used as
locks).  Prints one line per case; the summaries are kept in profiles/.

    FF_CHECKED=1 python tests/sanitizer_smoke.py --full

runs the tree build and the walk (counters off and on, W = 32 and 64, N_leaf 1 and 8, cell order 0 and 1) over
configs 3 and 4 of BASELINE.json at their full size N = 2^20, i.e. with the walk's stack, ring and parked-cell queue
at the depth the bench reaches (the bounds checked: stack <= 1024, ring <= 128, parked <= 64 entries).
"""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import numpy as np
import torch

import ffgen
import paper_1212_2934_b200 as ff


def main():
    for N, nleaf, group, order in ((3000, 1, 32, 0), (4097, 4, 32, 0), (33, 1, 32, 0), (2500, 1, 64, 0), (2100, 2, 32, 1)):
        c = ffgen.config(1, N=N)
        pos, mom = torch.from_numpy(c["pos"]).cuda(), torch.from_numpy(c["mom"]).cuda()
        ctx = ff.FFContext(N, 0.5, nleaf=nleaf, counters=True)
        if group != 32:
            ctx.set_option(ff.FF_OPT_GROUP, group)
        if order:
            ctx.set_option(ff.FF_OPT_CELL_ORDER, order)
        ctx.build_tree(pos)
        H, F = ctx.eval_bh(pos, mom)
        ctx.set_option(ff.FF_OPT_COUNTERS, 0)
        H2, F2 = torch.full_like(H, float("nan")), torch.full_like(F, float("nan"))
        g = ff.shard_groups(N, 2, 0, group)[1]
        ctx.eval_bh_range(pos, mom, H2, F2, 0, g)
        ctx.eval_bh_range(pos, mom, H2, F2, g, -1)
        Hd, Fd = ctx.eval_direct(pos, mom)
        Hh, Fh = np.empty_like(c["pos"]), np.empty_like(c["pos"])
        ctx.eval_bh_host(c["pos"], c["mom"], Hh, Fh)
        L = float(c["pos"].max()) + 1.0
        for all_pairs in (0, 1):
            p = ff.ff_step_params()
            p.dtau, p.gamma_d, p.gamma_r = 1e-3, 1.0, 1.0
            p.lj_epsilon, p.lj_sigma, p.lj_cutoff = 1.0, 1.0, 2.5
            p.noise_d, p.noise_r, p.seed = 0.05, 0.05, 3
            p.wall_epsilon, p.wall_sigma = 1.0, 0.5
            for a in range(3):
                p.wall_lo[a], p.wall_hi[a] = -1.0, L
            p.all_pairs = all_pairs
            x, u = pos.clone(), mom.clone()
            v, w = torch.zeros_like(pos), torch.zeros_like(pos)
            for s in range(2):
                ctx.step(x, v, u, w, p, s)
        torch.cuda.synchronize()
        ctx.timings()                                      # raises FFError if a device-side check failed (checked build)
        same = bool(torch.equal(H, H2) and torch.equal(F, F2))
        print("N=%d nleaf=%d W=%d order=%d: ranges compose=%s, BH vs direct rel L2 %.3e, finite=%s"
              % (N, nleaf, group, order, same, float((H - Hd).norm() / Hd.norm()), bool(torch.isfinite(x).all())))
        assert same
    print("library: %s; no device-side error flag was raised" % ("CHECKED build (FF_CHECK compiled in)"
                                                               if os.environ.get("FF_CHECKED") == "1" else "release build"))


def full():
    for cfg in (3, 4):
        c = ffgen.config(cfg)
        N = len(c["pos"])
        pos, mom = torch.from_numpy(c["pos"]).cuda(), torch.from_numpy(c["mom"]).cuda()
        for nleaf, group, order in ((1, 32, 0), (1, 64, 0), (8, 32, 0), (1, 32, 1), (8, 32, 1)):
            ctx = ff.FFContext(N, c["theta"], nleaf=nleaf)
            if group != 32:
                ctx.set_option(ff.FF_OPT_GROUP, group)
            if order:
                ctx.set_option(ff.FF_OPT_CELL_ORDER, order)
            ctx.build_tree(pos)
            H, F = ctx.eval_bh(pos, mom)
            ctx.set_option(ff.FF_OPT_COUNTERS, 1)
            H2, F2 = ctx.eval_bh(pos, mom)
            torch.cuda.synchronize()
            cnt = ctx.counters()                           # raises FFError if a device-side check failed
            ctx.timings()
            print("config %d N=%d nleaf=%d W=%d order=%d: counters %s, finite=%s, counting variant identical=%s"
                  % (cfg, N, nleaf, group, order, cnt, bool(torch.isfinite(H).all() and torch.isfinite(F).all()),
                     bool(torch.equal(H, H2) and torch.equal(F, F2))))
            assert bool(torch.isfinite(H).all() and torch.isfinite(F).all())
            ctx.close()
            del ctx
    print("full size: %s; no device-side error flag was raised" % ("CHECKED build (FF_CHECK compiled in)"
                                                                 if os.environ.get("FF_CHECKED") == "1" else "release build"))


if __name__ == "__main__":
    full() if "--full" in sys.argv else main()
