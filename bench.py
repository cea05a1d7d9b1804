#!/usr/bin/env python
"""bench.py -- the headline measurement of BASELINE.json:

    dipole field+force particle-evals/s & ms/step at N = 2^20, theta = 0.5; FP32-pipe % of peak

One "step" = one pass of the whole hot path: ff_build_tree
(bounding box, Morton keys, radix sort, octree) + ff_eval_bh (cell moments, tree walk, scatter to
caller order) on config 3 (1 048 576 hard-sphere dipoles, volume fraction 0.1, isotropic moments),
inputs resident in HBM.  Prints ONE JSON line (see the driver contract in the task statement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n N] [--quick]

N > 1: launched under torchrun, one rank per GPU.  The headline line is weak scaling: every rank runs an
independent replica of the workload with its own seed (the paper averages over independent realisations,
PAPER.md:243), no data-path collective.  The same invocation then also measures the target-sharded path of
SURVEY.md 8(e) on ONE common ensemble (all-gather of pos and mom per step, redundant tree, every rank walks a
Morton-contiguous slice of the groups) and reports it in the "strong" block of the line.
--impl reference: the fp64 oracle (oracle/), as it stands, on the host cores of this box.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "dipole field+force particle-evals/s (Barnes-Hut step: sort+build+moments+walk), N=2^20, theta=0.5"
UNIT = "particle-evals/s"
FLOP_PER_INTERACTION = 60.0      # SURVEY.md 8(d)'s algorithmic figure per h+f pair term (the tensor form of ff_pair.cuh
                                 # executes 25 FFMA x 2 + 11 FMUL = 61 per interaction, + 1 MUFU.RSQ)
FP32_LANES_PER_SM = 128
# algorithmic bytes per particle of the HBM-bound phases (DESIGN.md section 5 / SURVEY.md 8(d))
ALG_BYTES = {"bbox_keys": 12 + 12 + 4, "sort": 4 * 16 + 4 + 12 + 16, "build": 26 + 16 * 0.39, "moments": 12 + 16 + 122}
# dram__bytes_read.sum + dram__bytes_write.sum of one ff_k_walk launch at config 3, from the
# `ncu --set full` capture summarised in profiles/r2_walk_full.md (a capture, not a measurement of this run)
WALK_DRAM_TRAFFIC_BYTES = 108625920   # 86.91 MB read + 21.72 MB written
WALK_DRAM_TRAFFIC_SOURCE = "ncu --set full capture of ff_k_walk<32,0,0,0> at commit 4ffcb26, profiles/r2_walk_full.md"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return json.load(fh), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def started(self):
        return self.proc is not None

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()

    def summary(self, t0, t1):
        """Median, minimum and count of the SM-clock samples taken between the wall-clock times t0 and t1, and every
        throttle reason seen in them.  The sampler keeps running (stop() ends it)."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_min_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in list(self.rows):
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                if t0 - 0.05 <= ts <= t1 + 0.15:
                    sm.append(float(f[0]))
                    mx.append(float(f[1]))
                    for nm, v in zip(names, f[3:7]):
                        if v.lower().startswith("active"):
                            reasons.add(nm)
            except ValueError:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_min_mhz": min(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm), "reasons": sorted(reasons)}


def _workload(n, seed, cfg=3):
    """Config `cfg` of BASELINE.json (default 3, the one the metric is quoted on); n overrides its size."""
    import ffgen
    c = ffgen.config(cfg, seed=seed, N=n)
    return c


# ---- rank plumbing (one process per GPU; tests/test_multirank.py drives these with gloo on the CPU) ----
def rank_env():
    """(world, rank, local_rank) from the torchrun environment; (1, 0, 0) for a plain launch."""
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def max_over_ranks(ms, world, device):
    """A time measured on each rank's device -> the slowest rank's time (the job finishes with its last rank)."""
    import torch
    t = torch.tensor([float(ms)], device=device, dtype=torch.float64)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_particles(local, world):
    """Target sharding: every rank owns N / world particles and needs all of them as sources.
    One all-gather per array and step (12 B per particle and array); the tree is then built redundantly."""
    if world == 1:
        return local
    import torch
    import torch.distributed as dist
    parts = [torch.empty_like(local) for _ in range(world)]
    dist.all_gather(parts, local.contiguous())
    return torch.cat(parts, dim=0)


def gather_particles_begin(local, world):
    """The same all-gather without waiting for it: returns a handle for gather_particles_end, so that the caller can
    enqueue independent work (the tree build needs the positions only) while the moments are still on the wire."""
    if world == 1:
        return (local, None, None)
    import torch
    import torch.distributed as dist
    parts = [torch.empty_like(local) for _ in range(world)]
    work = dist.all_gather(parts, local.contiguous(), async_op=True)
    return (None, parts, work)


def gather_particles_end(handle):
    import torch
    local, parts, work = handle
    if parts is None:
        return local
    work.wait()                        # NCCL: makes the current stream wait for the collective; gloo: blocks the host
    return torch.cat(parts, dim=0)


def strong_block(world, n, ms_one_gpu, ms_sharded, gather_ms, walk_ms, phases):
    """The target-sharded measurement as it appears in the JSON line: ONE ensemble of n particles on
    `world` GPUs.  efficiency = (time one GPU needs for the whole ensemble / world) / time of the sharded step."""
    return {"scaling": "strong", "n_gpus": world, "N": n, "ms_per_step": ms_sharded,
            "value": n / (ms_sharded * 1e-3), "unit": UNIT, "allgather_ms": gather_ms, "walk_ms_max_over_ranks": walk_ms,
            "one_gpu_ms_per_step": ms_one_gpu, "efficiency_vs_one_gpu": (ms_one_gpu / world) / ms_sharded,
            "phases_ms_rank0": phases,
            "sharding": "targets: one ensemble, all-gather of pos then mom per step (the mom gather overlaps the tree "
                        "build), redundant tree on every rank, each rank walks a Morton-contiguous slice of the groups"}


def job_rate(world, units_per_rank, ms):
    """Whole-job throughput: every rank processed `units_per_rank` units (weak scaling, independent replicas,
    no data-path collective) in `ms`, the max over ranks."""
    return world * units_per_rank / (ms * 1e-3)


GROUP_W = 32      # targets per walk group (FF_OPT_GROUP / the oracle's W) of the headline, in BOTH arms
NLEAF = 1         # leaf capacity of the headline, in both arms


def _config_dict(c, world):
    """The `config` object of the JSON line.  One function for the product arm and the reference arm, so that the two
    lines carry the same keys and values for the same workload."""
    return {"workload": _describe(c), "N": c["N"], "theta": c["theta"], "group": GROUP_W, "nleaf": NLEAF,
            "l2": "GPU arm: flushed between timed steps (512 MB memset); CPU reference arm: not applicable",
            "replicas": world, "sharding": "independent replicas, no collective"}


def _describe(c):
    kind = {1: "hard-sphere dipoles (d=1), phi=0.05, isotropic unit moments",
            2: "hard-sphere dipoles (d=1), phi=0.1, von Mises-Fisher moments about +z (kappa=5)",
            3: "hard-sphere dipoles (d=1), phi=0.1, isotropic unit moments",
            4: "straight head-to-tail chains of 32 touching spheres within 15 deg of z, moments along the chain",
            5: "hard-sphere dipoles (d=1), phi=0.2, isotropic unit moments"}[c["config"]]
    return ("config %d of BASELINE.json: N=%d %s, theta=%g, group rule W=%d, tree rebuilt every step, H and F"
            % (c["config"], c["N"], kind, c["theta"], GROUP_W))


def _oracle_step(c, groups, nthreads=0):
    """One oracle pass on a bounded sample: full tree + moments, walk of `groups` only.
    Returns (t_build, t_moments, t_walk)."""
    import oracle
    t0 = time.perf_counter()
    t = oracle.Tree(c["pos"])
    t1 = time.perf_counter()
    t.moments(c["mom"])
    t2 = time.perf_counter()
    t.eval(c["theta"], GROUP_W, groups=groups, nthreads=nthreads)
    t3 = time.perf_counter()
    return t1 - t0, t2 - t1, t3 - t2


def _oracle_rate(c, n_groups_sample, nthreads=0):
    """Whole-job particle-evals/s of the oracle from a bounded sample of the walk groups (all of them if the sample
    covers them: then nothing is extrapolated)."""
    N = c["N"]
    n_groups = (N + 31) // 32
    if n_groups_sample >= n_groups:
        groups = np.arange(n_groups)
    else:
        groups = np.random.default_rng(0).choice(n_groups, n_groups_sample, replace=False)
    tb, tm, tw = _oracle_step(c, groups, nthreads)
    full = tb + tm + tw * n_groups / len(groups)
    return N / full, dict(t_build_s=tb, t_moments_s=tm, t_walk_sample_s=tw, groups=int(len(groups)),
                          step_s=full, measured_s=tb + tm + tw)


REFERENCE_MAX_GROUPS = 32768     # every group of the one-million configs; a bounded sample only beyond that (config 5)


def run_reference(args):
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    c = _workload(args.n, 0, args.config)
    cores = oracle.max_threads()
    n_groups = (c["N"] + 31) // 32
    sample = min(n_groups, REFERENCE_MAX_GROUPS)
    for _ in range(args.warmup):
        _oracle_rate(c, sample)
    t0 = time.perf_counter()
    steps = [_oracle_rate(c, sample)[1] for _ in range(args.steps)]
    wall = time.perf_counter() - t0
    step_s = float(np.mean([d["step_s"] for d in steps]))
    value = c["N"] / step_s
    if sample == n_groups:
        desc = ("fp64 oracle (oracle/ff_oracle.c), every step complete and timed as it runs: tree build + cell moments "
                "over all N, walk of all %d groups of 32 targets (nothing extrapolated)" % n_groups)
    else:
        desc = ("fp64 oracle (oracle/ff_oracle.c), per step: full tree build + cell moments over all N, walk of %d sampled "
                "groups of 32 targets, walk time extrapolated to all %d groups" % (sample, n_groups))
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * step_s, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config_dict(c, args.gpus),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "wall_s": wall, "measured_s_per_step": float(np.mean([d["measured_s"] for d in steps])),
    }
    print(json.dumps(out))


def _rel_errs(x, ref, floor):
    e = np.linalg.norm(x - ref, axis=1) / np.maximum(np.maximum(np.linalg.norm(ref, axis=1), floor), 1e-300)
    return e


def _parity_block(Hg, Fg, Ho, Fo, Qo, tol=1e-4):
    """Per-particle relative L2 error of (H, F) against the oracle under the two metrics of DESIGN.md section 6, and
    how the gate moves with the constant kappa of the term-scale floor Q_k / kappa."""
    out = {"targets": int(len(Ho)), "tolerance": tol,
           "metric": "|x_k - ref_k| / max(|ref_k|, Q_k / 8) against the fp64 oracle's Barnes-Hut (same theta, W = 32)"}
    for name, x, ref, q in (("H", Hg, Ho, Qo[:, 0]), ("F", Fg, Fo, Qo[:, 1])):
        e = _rel_errs(x, ref, q / 8.0)
        survey = _rel_errs(x, ref, 1e-3 * np.sqrt((np.linalg.norm(ref, axis=1) ** 2).mean()))
        out[name] = {"max": float(e.max()), "p99": float(np.quantile(e, 0.99)), "median": float(np.median(e)),
                     "global_rel_l2": float(np.linalg.norm(x - ref) / np.linalg.norm(ref)),
                     "max_by_kappa": {str(k): float(_rel_errs(x, ref, q / k).max()) for k in (4, 8, 16)},
                     "max_survey_metric_no_Q": float(survey.max())}
    return out


def _md_parity(ff, ctx, snap, kw, theta, seed):
    """Config 3's MD run: the oracle re-evaluated on the GPU's OWN state at one step.  From a copy of
    the snapshot the GPU takes one deterministic ff_step (noise off); on sampled groups of that state the oracle gives
    Barnes-Hut h, f (same theta, W = 32), the Lennard-Jones force of Eq. 13 and the Euler-Maruyama update
    (oracle/md_step.py); compared are the increments, which is where the arithmetic of the step sits."""
    import torch
    from scipy.spatial import cKDTree

    import oracle
    from oracle.md_step import lj_force, md_step
    x0, v0, u0, w0 = [t.cpu().numpy() for t in snap]
    N = len(x0)
    q = ff.ff_step_params()
    q.dtau, q.gamma_d, q.gamma_r = kw["dtau"], kw["gamma_d"], kw["gamma_r"]
    for a in range(3):
        q.h_ext[a] = kw["h_ext"][a]
    q.lj_epsilon, q.lj_sigma, q.lj_cutoff = kw["lj"]
    xs, vs, us, ws = [t.clone() for t in snap]
    ctx.step(xs, vs, us, ws, q, 0)
    torch.cuda.synchronize()
    v1, w1 = vs.cpu().numpy().astype(np.float64), ws.cpu().numpy().astype(np.float64)
    otree = oracle.Tree(x0)
    otree.moments(u0)
    n_groups = (N + 31) // 32
    sel = np.random.default_rng(seed).choice(n_groups, min(32, n_groups), replace=False)
    Ho, Fo, _, Qo = otree.eval(theta, 32, groups=sel, scale=True)
    _, operm = otree.keys()
    rows = np.unique(operm[(sel[:, None] * 32 + np.arange(32)[None, :]).ravel().clip(max=N - 1)])
    # Eq. 13 for the sampled targets: the sources handed to the oracle are a superset of everything inside the
    # cut-off (a k-d tree query with a 1 % wider radius; input selection only), the rest contributes exactly zero
    xd = x0.astype(np.float64)
    near = cKDTree(xd).query_ball_point(xd[rows], kw["lj"][2] * 1.01)
    sub = np.unique(np.concatenate([np.asarray(n_, dtype=np.int64) for n_ in near] + [rows]))
    fsr = lj_force(xd[sub], kw["lj"][0], kw["lj"][1], kw["lj"][2], chunk=64, targets=np.searchsorted(sub, rows))
    _, vr, _, wr = md_step(x0[rows], v0[rows], u0[rows], w0[rows], Ho[rows], Fo[rows], kw["dtau"], kw["gamma_d"],
                           kw["gamma_r"], kw["h_ext"], fsr)
    dt, ulp = kw["dtau"], 2.0 ** -24
    # increments recovered from fp32 states carry the representation error 2^-24 |v1| / dtau of the stored result,
    # whatever the forces are: subtracted before the relative gate (as in tests/test_gpu_step.py)
    acc_g, acc_r = (v1[rows] - v0[rows]) / dt, (vr - v0[rows]) / dt
    scale = np.maximum(np.maximum(np.linalg.norm(acc_r, axis=1), Qo[rows, 1] / 8.0), np.linalg.norm(fsr, axis=1) / 8.0)
    e_acc = np.maximum(np.linalg.norm(acc_g - acc_r, axis=1) - ulp * np.linalg.norm(v1[rows], axis=1) / dt, 0.0) / scale
    tq_g, tq_r = (w1[rows] - w0[rows]) / dt, (wr - w0[rows]) / dt
    tscale = np.maximum(np.linalg.norm(tq_r, axis=1), 2.5 * Qo[rows, 0] / 8.0)
    e_tq = np.maximum(np.linalg.norm(tq_g - tq_r, axis=1) - ulp * np.linalg.norm(w1[rows], axis=1) / dt, 0.0) / tscale
    return {"targets": int(len(rows)), "velocity_increment_max_err": float(e_acc.max()),
            "angular_velocity_increment_max_err": float(e_tq.max()),
            "max_lj_force": float(np.linalg.norm(fsr, axis=1).max())}


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_1212_2934_b200 as ff

    world, rank, local = rank_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    # headline: an independent realisation per rank (weak scaling, no data-path collective)
    c = _workload(args.n, rank, args.config)
    N, theta = c["N"], c["theta"]
    pos_h = torch.from_numpy(c["pos"]).pin_memory()
    mom_h = torch.from_numpy(c["mom"]).pin_memory()
    pos, mom = pos_h.to(dev), mom_h.to(dev)
    H, F = torch.empty_like(pos), torch.empty_like(pos)
    ctx = ff.FFContext(N, theta, device=dev, timing=True)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def step():
        ctx.build_tree(pos)
        ctx.eval_bh(pos, mom, H, F)

    sampler = ClockSampler(local)          # one nvidia-smi sampler (20 ms period) for the whole run, rank 0 only
    t_run0 = time.time()

    def timed(step_fn, steps, sample_clocks):
        """W >= 3 untimed steps, then `steps` steps timed on the device (CUDA events around each, L2 flushed before
        each and outside the timed region), barrier + synchronize on both sides, max over ranks."""
        for _ in range(max(args.warmup, 3)):
            flush.zero_()
            step_fn()
        torch.cuda.synchronize()
        ctx.timings()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        if sample_clocks and rank == 0 and not sampler.started():
            sampler.start()                                # keeps running until the line is printed (whole-run clocks)
            time.sleep(0.25)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        ph = {k: 0.0 for k in ff.PHASES}
        l0 = ctx.launch_count()
        t_wall0 = time.time()
        for i in range(steps):
            flush.zero_()                                  # evict the previous step from L2 (not timed)
            ev[i][0].record()
            step_fn()
            ev[i][1].record()
            ev[i][1].synchronize()
            for k, v in ctx.timings().items():
                ph[k] += v
        torch.cuda.synchronize()
        t_wall1 = time.time()
        n_launch = ctx.launch_count() - l0
        if world > 1:
            dist.barrier()
        ms = [a.elapsed_time(b) for a, b in ev]
        total = max_over_ranks(sum(ms), world, dev)
        clk = sampler.summary(t_wall0, t_wall1) if (sample_clocks and rank == 0) else None
        return total / steps, ms, {k: v / steps for k, v in ph.items()}, n_launch, clk

    # interaction counts of this workload (separate, untimed run of the counting kernel variant)
    ctx.set_option(ff.FF_OPT_COUNTERS, 1)
    step()
    n_cell, n_part, n_mac = ctx.counters()
    ctx.set_option(ff.FF_OPT_COUNTERS, 0)
    interactions = n_cell + n_part

    ms_per_step, step_ms, phases, launches, clocks = timed(step, args.steps, True)
    value = job_rate(world, N, ms_per_step)
    Hg, Fg = H.cpu().numpy().astype(np.float64), F.cpu().numpy().astype(np.float64)     # results of the timed steps

    # ---- N > 1: the target-sharded path on ONE common ensemble, in the same invocation
    strong = None
    if world > 1 and N % world == 0:
        c0 = c if rank == 0 else _workload(args.n, 0, args.config)
        rows = slice(rank * (N // world), (rank + 1) * (N // world))
        pos_local = torch.from_numpy(c0["pos"][rows.start:rows.stop]).to(dev)
        mom_local = torch.from_numpy(c0["mom"][rows.start:rows.stop]).to(dev)
        g_begin, g_end = ff.shard_groups(N, world, rank)
        Hs, Fs = torch.empty_like(pos), torch.empty_like(pos)

        def step_sharded():
            p_all = gather_particles(pos_local, world)             # the tree build needs the positions only ...
            pending = gather_particles_begin(mom_local, world)     # ... the moments travel under it
            ctx.build_tree(p_all)
            m_all = gather_particles_end(pending)
            ctx.eval_bh_range(p_all, m_all, Hs, Fs, g_begin, g_end)

        ms_strong, _, ph_strong, _, _ = timed(step_sharded, args.steps, False)
        # the exchange alone
        g0e, g1e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        dist.barrier()
        g0e.record()
        for _ in range(args.steps):
            gather_particles(pos_local, world)
            gather_particles(mom_local, world)
        g1e.record()
        g1e.synchronize()
        gather_ms = max_over_ranks(g0e.elapsed_time(g1e) / args.steps, world, dev)
        walk_ms = max_over_ranks(ph_strong["walk"], world, dev)
        strong = strong_block(world, N, ms_per_step, ms_strong, gather_ms, walk_ms, ph_strong)

    # ---- end to end through the C ABI with host buffers (H2D + step + D2H of every step inside the timed region).
    # ff_eval_bh_host_async pipelines successive steps: uploads, compute and downloads run on three streams with
    # double-buffered staging, so the copies of one step overlap the compute of its neighbours.  Two result
    # buffers alternate on the host so that a step's download never lands in a buffer still being checked.
    H_h = [torch.empty((N, 3), dtype=torch.float32).pin_memory() for _ in range(2)]
    F_h = [torch.empty((N, 3), dtype=torch.float32).pin_memory() for _ in range(2)]
    for i in range(2):
        ctx.eval_bh_host(pos_h, mom_h, H_h[i], F_h[i])
    e2e_steps = max(3, args.steps)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(e2e_steps):
        flush[:192 << 20].zero_()                      # evict the previous step from the 126 MB L2 (inside the timed region here)
        ctx.eval_bh_host_async(pos_h, mom_h, H_h[i & 1], F_h[i & 1])
    ctx.host_sync()
    e1.record()
    e1.synchronize()
    e2e_ms = e0.elapsed_time(e1)
    # the same call, one step at a time (upload, compute, download strictly in sequence): what a loop pays whose next
    # input depends on the previous result
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(5):
        ctx.eval_bh_host(pos_h, mom_h, H_h[0], F_h[0])
    e2e_serial_ms = max_over_ranks((time.perf_counter() - t0) * 1e3 / 5, world, dev)
    H_h, F_h = H_h[0], F_h[0]
    e2e_value = job_rate(world, N, max_over_ranks(e2e_ms, world, dev) / e2e_steps)
    checksum = float(H_h.double().abs().sum() + F_h.double().abs().sum())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the walk): plain FP32 ALU work
    peaks, peak_src = _peaks()
    sm_max = float(clocks["sm_max_mhz"] or peaks.get("sm_max_mhz", 1965.0))
    num_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peak_tflops = num_sms * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    walk_ms = phases["walk"]
    achieved = interactions * FLOP_PER_INTERACTION / (walk_ms * 1e-3) / 1e12
    probes = {name: max(ctx.measure_probe(kind, 1 << 13) for _ in range(2))
              for name, kind in (("ffma", ff.FF_PROBE_FFMA), ("ffma2_three_register_pairs", ff.FF_PROBE_FFMA2_PAIRS),
                                 ("ffma2_reused_operand", ff.FF_PROBE_FFMA2_REUSE),
                                 ("ffma2_scalar_operand", ff.FF_PROBE_FFMA2_SCALAR), ("eval_loop", ff.FF_PROBE_EVAL),
                                 ("eval_loop_scalar", ff.FF_PROBE_EVAL_SCALAR), ("eval_loop_hybrid", ff.FF_PROBE_EVAL_HYBRID))}
    roofline = {
        "bound": "alu", "kernel": "ff_k_walk", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": achieved / peak_tflops, "traffic": WALK_DRAM_TRAFFIC_BYTES, "traffic_source": WALK_DRAM_TRAFFIC_SOURCE,
        "peak_source": "nominal: %d SMs x 128 FP32 lanes x 2 flop x %.0f MHz (clocks.max.sm); MEASURED_PEAKS.json (%s) "
                       "holds no FP32 figure; the probes below are measured in this run (ff_measure_probe)"
                       % (num_sms, sm_max, peak_src),
        "measured_fma_peak_tflops": probes["ffma"], "frac_of_measured_fma": achieved / probes["ffma"],
        "measured_packed_ffma2_tflops": {k: probes[k] for k in ("ffma2_three_register_pairs", "ffma2_reused_operand",
                                                                "ffma2_scalar_operand")},
        "eval_loop_tflops": probes["eval_loop"], "eval_loop_ceiling_frac": probes["eval_loop"] / peak_tflops,
        "frac_of_eval_loop_ceiling": achieved / probes["eval_loop"],
        # the same 36 operations per interaction in the two other encodings (csrc/ff_probe.cu): all scalar FFMA / FMUL,
        # and packed except for the twelve three-register-pair FFMA2 (as 24 scalar FFMA).  If neither beats
        # eval_loop_tflops the packed encoding is the fastest form of this arithmetic on this part.
        "eval_loop_scalar_tflops": probes["eval_loop_scalar"], "eval_loop_hybrid_tflops": probes["eval_loop_hybrid"],
        "interactions_per_launch": interactions, "flop_per_interaction": FLOP_PER_INTERACTION,
        "kernel_ms": walk_ms, "kernel_share_of_step": walk_ms / ms_per_step,
        "interactions_per_s": interactions / (walk_ms * 1e-3),
        # FP32-pipe occupancy by the interaction arithmetic alone = interactions x 36 FP32 lane-ops
        # (18 packed instructions of two lanes' worth each) / (time x SMs x 128 lanes x clock)
        "fp32_lane_ops_per_interaction": 36,
        "fp32_lane_occupancy_by_interactions": interactions * 36.0 / (walk_ms * 1e-3 * num_sms * FP32_LANES_PER_SM * sm_max * 1e6),
        "note": "25 of the 36 FP32 instructions per interaction are FMAs, so a saturated FP32 pipe reads 0.85; the "
                "register file feeds a packed instruction two register words per lane and cycle, so packed FMAs with "
                "three register-pair operands issue every 3 cycles (ffma2_three_register_pairs; 12 of the 36), which "
                "caps this instruction mix at eval_loop_ceiling_frac: the evaluation loop of the walk run alone",
    }
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    # algorithmic bytes per particle of the HBM-bound phases (DESIGN.md / SURVEY.md 8(d))
    alg_bytes = ALG_BYTES
    hbm_phases = {k: {"ms": phases[k], "achieved_gbs": alg_bytes[k] * N / (phases[k] * 1e-3) / 1e9,
                      "frac_of_hbm_peak": alg_bytes[k] * N / (phases[k] * 1e-3) / 1e9 / hbm}
                  for k in alg_bytes if phases[k] > 0}

    extras = {}
    if not args.quick and N <= (1 << 21):                  # the N^2 kernel takes minutes beyond that
        # GPU direct all-pairs on the same workload (a8), once; and the BH-vs-all-pairs error vs theta
        torch.cuda.synchronize()
        ctx.timings()
        Hd, Fd = ctx.eval_direct(pos, mom)
        torch.cuda.synchronize()
        d_ms = ctx.timings()["direct"]
        pairs = float(N) * (N - 1)
        extras["gpu_direct"] = {"ms": d_ms, "pair_interactions_per_s": pairs / (d_ms * 1e-3),
                                "tflops": pairs * FLOP_PER_INTERACTION / (d_ms * 1e-3) / 1e12,
                                "frac_of_fp32_peak": pairs * FLOP_PER_INTERACTION / (d_ms * 1e-3) / 1e12 / peak_tflops,
                                "frac_of_eval_loop_ceiling": pairs * FLOP_PER_INTERACTION / (d_ms * 1e-3) / 1e12 / probes["eval_loop"],
                                "flop_per_pair": FLOP_PER_INTERACTION, "speedup_bh_over_direct": d_ms / ms_per_step}
        # the oracle's all-pairs sum on a sample of targets (all sources), on the host cores: the GPU result of those
        # targets is checked against it, and its rate extrapolated to all N targets is the CPU all-pairs baseline
        # the paper's Table 1 compares with (there: one core, single precision)
        import oracle as _oracle
        rng = np.random.default_rng(1)
        tsel = np.sort(rng.choice(N, size=min(N, 1024), replace=False)).astype(np.int64)
        t0 = time.perf_counter()
        Ha, Fa, Qa = _oracle.allpairs(c["pos"], c["mom"], targets=tsel, scale=True)
        t_ap = time.perf_counter() - t0
        Hs, Fs = Hd[torch.from_numpy(tsel).to(dev)].cpu().numpy(), Fd[torch.from_numpy(tsel).to(dev)].cpu().numpy()
        pd = _parity_block(Hs, Fs, Ha, Fa, Qa, tol=1e-5)
        extras["gpu_direct"].update({
            "max_err_vs_oracle_allpairs": {"H": pd["H"]["max"], "F": pd["F"]["max"], "targets": int(len(tsel)),
                                           "tolerance": 1e-5, "H_survey_metric_no_Q": pd["H"]["max_survey_metric_no_Q"],
                                           "F_survey_metric_no_Q": pd["F"]["max_survey_metric_no_Q"]},
            "cpu_allpairs_oracle": {"pairs_per_s": len(tsel) * (N - 1) / t_ap, "cores": _oracle.max_threads(),
                                    "extrapolated_s_per_eval": t_ap * N / len(tsel),
                                    "sample": "%d targets x all sources, fp64" % len(tsel)}})
        errs = {}
        ctx.build_tree(pos)          # (the host calls above built their tree from the staging copy of the positions)
        for th in (0.3, 0.5, 0.7):
            ctx.set_option(ff.FF_OPT_THETA, th)
            Hb, Fb = ctx.eval_bh(pos, mom)
            errs[str(th)] = {"H_rel_l2": float((Hb - Hd).double().norm() / Hd.double().norm()),
                             "F_rel_l2": float((Fb - Fd).double().norm() / Fd.double().norm())}
        ctx.set_option(ff.FF_OPT_THETA, theta)
        extras["bh_vs_allpairs_error"] = {"reference": "GPU direct kernel (ff_eval_direct)", "by_theta": errs}
        # the group width (reading Q2 of DESIGN.md): W = 64 at the same theta -- more interactions, smaller error
        ctx.set_option(ff.FF_OPT_GROUP, 64)
        ctx.set_option(ff.FF_OPT_COUNTERS, 1)
        ctx.build_tree(pos)
        Hb, Fb = ctx.eval_bh(pos, mom)
        c64 = ctx.counters()
        ctx.set_option(ff.FF_OPT_COUNTERS, 0)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(5):
            ctx.build_tree(pos)
            ctx.eval_bh(pos, mom, Hb, Fb)
        b.record()
        b.synchronize()
        w64 = ctx.timings()["walk"]
        ctx.set_option(ff.FF_OPT_GROUP, 32)
        extras["group_width_64"] = {
            "ms_per_step": a.elapsed_time(b) / 5, "walk_ms": w64, "interactions_per_target": (c64[0] + c64[1]) / N,
            "walk_tflops": (c64[0] + c64[1]) * FLOP_PER_INTERACTION / (w64 * 1e-3) / 1e12,
            "frac_of_fp32_peak": (c64[0] + c64[1]) * FLOP_PER_INTERACTION / (w64 * 1e-3) / 1e12 / peak_tflops,
            "H_rel_l2_vs_allpairs": float((Hb - Hd).double().norm() / Hd.double().norm()),
            "F_rel_l2_vs_allpairs": float((Fb - Fd).double().norm() / Fd.double().norm()),
            "note": "FF_OPT_GROUP = 64 at theta = %g, L2 not flushed; W = 32 is the headline" % theta}

        # better cells at equal cost: bucket leaves and the first-order cell term, alone and together
        variants = {}
        for nleaf_v, order_v, th in ((1, 0, 0.5), (1, 1, 0.5), (8, 0, 0.5), (8, 1, 0.5), (1, 1, 0.6), (8, 1, 0.6),
                                     (1, 0, 0.7), (1, 1, 0.7), (8, 1, 0.7), (1, 0, 0.4)):
            ctx.set_option(ff.FF_OPT_NLEAF, nleaf_v)
            ctx.set_option(ff.FF_OPT_CELL_ORDER, order_v)
            ctx.set_option(ff.FF_OPT_THETA, th)
            ctx.set_option(ff.FF_OPT_COUNTERS, 1)
            ctx.build_tree(pos)
            Hb, Fb = ctx.eval_bh(pos, mom)
            cv = ctx.counters()
            ctx.set_option(ff.FF_OPT_COUNTERS, 0)
            ctx.timings()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(5):
                ctx.build_tree(pos)
                ctx.eval_bh(pos, mom, Hb, Fb)
            b.record()
            b.synchronize()
            variants["nleaf=%d order=%d theta=%g" % (nleaf_v, order_v, th)] = {
                "ms_per_step": a.elapsed_time(b) / 5, "walk_ms": ctx.timings()["walk"],
                "cell_terms_per_target": cv[0] / N, "particle_terms_per_target": cv[1] / N,
                "H_rel_l2_vs_allpairs": float((Hb - Hd).double().norm() / Hd.double().norm()),
                "F_rel_l2_vs_allpairs": float((Fb - Fd).double().norm() / Fd.double().norm())}
        ctx.set_option(ff.FF_OPT_NLEAF, 1)
        ctx.set_option(ff.FF_OPT_CELL_ORDER, 0)
        ctx.set_option(ff.FF_OPT_THETA, theta)
        extras["cell_variants"] = {"by_variant": variants,
                                   "note": "config 3, L2 not flushed; order=1 adds the first-order cell term "
                                           "(FF_OPT_CELL_ORDER), nleaf=8 bucket leaves (FF_OPT_NLEAF); errors are global "
                                           "relative L2 against the GPU all-pairs result"}

        # the same recipe at smaller sizes (device-resident, L2 not flushed): how the step scales with N
        sweep = {}
        for n_small in (1 << 10, 1 << 12, 1 << 14, 1 << 16, 1 << 18):
            if n_small >= N:
                continue
            cs = _workload(n_small, rank, args.config)
            ps, ms_ = torch.from_numpy(cs["pos"]).to(dev), torch.from_numpy(cs["mom"]).to(dev)
            cx = ff.FFContext(n_small, theta, device=dev)
            for _ in range(3):
                cx.build_tree(ps); cx.eval_bh(ps, ms_)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(10):
                cx.build_tree(ps); cx.eval_bh(ps, ms_)
            b.record(); b.synchronize()
            bh_ms = a.elapsed_time(b) / 10
            cx.eval_direct(ps, ms_)
            a.record()
            for _ in range(3):
                cx.eval_direct(ps, ms_)
            b.record(); b.synchronize()
            ap_ms = a.elapsed_time(b) / 3
            # one MD step (ff_step: fields + Lennard-Jones + Euler-Maruyama) with either algorithm
            md = {}
            for name, flag in (("md_step_bh_ms", 0), ("md_step_allpairs_ms", 1)):
                q = ff.ff_step_params()
                q.dtau, q.gamma_d, q.gamma_r = 1e-3, 1.0, 1.0
                q.lj_epsilon, q.lj_sigma, q.lj_cutoff = 1.0, 1.0, 2.5
                q.all_pairs = flag
                xs, us = ps.clone(), ms_.clone()
                vs, ws = torch.zeros_like(ps), torch.zeros_like(ps)
                cx.step(xs, vs, us, ws, q, 0)
                reps = 10 if (flag == 0 or n_small <= (1 << 16)) else 2
                a.record()
                for r in range(reps):
                    cx.step(xs, vs, us, ws, q, 1 + r)
                b.record(); b.synchronize()
                md[name] = a.elapsed_time(b) / reps
            sweep[str(n_small)] = {"bh_ms_per_step": bh_ms, "allpairs_ms_per_eval": ap_ms,
                                   "particle_evals_per_s": n_small / (bh_ms * 1e-3), **md}
            del cx
        # the paper's Table 1 has the same crossover: all-pairs wins for N ~ 10^3, Barnes-Hut above
        extras["size_sweep"] = sweep

        # config 3 as BASELINE.json states it: 100 MD steps (ff_step: tree rebuilt, H and F by Barnes-Hut,
        # Lennard-Jones force, Euler-Maruyama update, dtau = 0.001 as in PAPER.md:200), per-phase timing.  The state
        # is snapshotted before steps 0, 50 and 99 (outside the timed segments) and the oracle re-evaluated on those
        # states afterwards.
        kw = {"dtau": 1e-3, "gamma_d": 1.0, "gamma_r": 1.0, "h_ext": (0.0, 0.0, 0.5), "lj": (1.0, 1.0, 2.5),
              "noise": (0.05, 0.05)}
        prm = ff.ff_step_params()
        prm.dtau, prm.gamma_d, prm.gamma_r = kw["dtau"], kw["gamma_d"], kw["gamma_r"]
        prm.h_ext[0], prm.h_ext[1], prm.h_ext[2] = kw["h_ext"]
        prm.lj_epsilon, prm.lj_sigma, prm.lj_cutoff = kw["lj"]
        prm.noise_d, prm.noise_r, prm.seed = kw["noise"][0], kw["noise"][1], 1
        x, u = pos.clone(), mom.clone()
        v, w = torch.zeros_like(pos), torch.zeros_like(pos)
        for s_ in range(3):
            ctx.step(x, v, u, w, prm, s_)
        torch.cuda.synchronize()
        ctx.timings()
        md_steps, snaps, md_total = 100, {}, 0.0
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for lo_, hi_ in ((0, 50), (50, 99), (99, 100)):
            snaps[lo_] = tuple(t.clone() for t in (x, v, u, w))
            torch.cuda.synchronize()
            e0.record()
            for s_ in range(lo_, hi_):
                ctx.step(x, v, u, w, prm, 3 + s_)
            e1.record()
            torch.cuda.synchronize()
            md_total += e0.elapsed_time(e1)
        md_ms = md_total / md_steps
        last = ctx.timings()
        md_par = {str(k): _md_parity(ff, ctx, snaps[k], kw, theta, 11 + k) for k in sorted(snaps)}
        del snaps
        extras["md_100_steps"] = {
            "ms_per_step": md_ms, "particle_steps_per_s": N / (md_ms * 1e-3), "steps": md_steps,
            "phases_ms_last_step": last, "finite": bool(torch.isfinite(x).all() and torch.isfinite(u).all()),
            "params": {"dtau": kw["dtau"], "gamma_d": kw["gamma_d"], "gamma_r": kw["gamma_r"], "h_ext": list(kw["h_ext"]),
                       "lj": list(kw["lj"]), "noise": list(kw["noise"])},
            "parity": {"by_step": md_par, "tolerance": 1e-4,
                       "max_err": max(max(d["velocity_increment_max_err"], d["angular_velocity_increment_max_err"])
                                      for d in md_par.values()),
                       "how": "state of the running simulation before steps 0, 50, 99 -> one deterministic ff_step on a "
                              "copy; velocity and angular-velocity increments against the oracle (Barnes-Hut at the same "
                              "theta and W, Eq. 13 pair sum, Euler-Maruyama update) on 32 sampled groups; metric and "
                              "tolerance of tests/test_gpu_step.py (DESIGN.md section 6)"},
            "note": "L2 not flushed between these steps (back-to-back MD steps, as in a simulation)"}

    # ---- the other full-size configs of BASELINE.json, timed the same way (L2 flushed, device resident): config 4
    # (chains: unbalanced tree, divergence) and config 5 (2^24 particles: the case where the O(N) phases are HBM bound)
    if not args.quick and args.config == 3 and args.n is None:
        for cfg_id, steps_c in ((4, 5), (5, 3)):
            cc = _workload(None, 0, cfg_id)
            Nc = cc["N"]
            pc, mc = torch.from_numpy(cc["pos"]).to(dev), torch.from_numpy(cc["mom"]).to(dev)
            Hc, Fc = torch.empty_like(pc), torch.empty_like(pc)
            cx = ff.FFContext(Nc, cc["theta"], device=dev, timing=True, counters=True)
            cx.build_tree(pc)
            cx.eval_bh(pc, mc, Hc, Fc)
            cnt = cx.counters()
            cx.set_option(ff.FF_OPT_COUNTERS, 0)
            for _ in range(2):
                cx.build_tree(pc); cx.eval_bh(pc, mc, Hc, Fc)
            torch.cuda.synchronize()
            cx.timings()
            phc, tot = {k: 0.0 for k in ff.PHASES}, 0.0
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for _ in range(steps_c):
                flush.zero_()
                a.record()
                cx.build_tree(pc); cx.eval_bh(pc, mc, Hc, Fc)
                b.record(); b.synchronize()
                tot += a.elapsed_time(b)
                for k, v_ in cx.timings().items():
                    phc[k] += v_
            phc = {k: v_ / steps_c for k, v_ in phc.items() if v_ > 0}
            inter = cnt[0] + cnt[1]
            extras["config%d" % cfg_id] = {
                "workload": _describe(cc), "ms_per_step": tot / steps_c, "particle_evals_per_s": Nc / (tot / steps_c * 1e-3),
                "phases_ms": phc, "interactions_per_target": inter / Nc,
                "walk_frac_of_fp32_peak": inter * FLOP_PER_INTERACTION / (phc["walk"] * 1e-3) / 1e12 / peak_tflops,
                "hbm_phases": {k: {"achieved_gbs": ALG_BYTES[k] * Nc / (phc[k] * 1e-3) / 1e9,
                                   "frac_of_hbm_peak": ALG_BYTES[k] * Nc / (phc[k] * 1e-3) / 1e9 / hbm} for k in ALG_BYTES},
                "finite": bool(torch.isfinite(Hc).all() and torch.isfinite(Fc).all())}
            del cx, pc, mc, Hc, Fc, cc

    # ---- parity of this very run at full size: the oracle's Barnes-Hut on sampled groups (DESIGN.md section 6 metric)
    import oracle
    otree = oracle.Tree(c["pos"])
    otree.moments(c["mom"])
    n_groups = (N + 31) // 32
    sel = np.random.default_rng(7).choice(n_groups, min(256, n_groups), replace=False)
    Ho, Fo, _, Qo = otree.eval(theta, 32, groups=sel, scale=True)
    _, operm = otree.keys()
    rows = operm[(sel[:, None] * 32 + np.arange(32)[None, :]).ravel().clip(max=N - 1)]
    rows = np.unique(rows)
    parity = _parity_block(Hg[rows], Fg[rows], Ho[rows], Fo[rows], Qo[rows])
    del otree

    # ---- the oracle timed beside it on this box's host cores (bounded sample)
    cores = oracle.max_threads()
    sample = 2048 if N >= (1 << 20) else max(1, min(2048, (N + 31) // 32))
    cpu_value, cpu_detail = _oracle_rate(c, sample)
    cpu_1, _ = _oracle_rate(c, max(1, sample // 8), nthreads=1)
    cpu_baseline = {"value": cpu_value, "unit": UNIT, "cores": cores, "kind": "oracle",
                    "sample": "full tree + moments over all N, walk of %d sampled groups (%d targets) extrapolated to all "
                              "groups" % (cpu_detail["groups"], cpu_detail["groups"] * 32),
                    "detail": cpu_detail, "single_thread_value": cpu_1}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": _config_dict(c, world),
        "clocks": clocks, "gpu_launches": int(launches), "launches_per_step": launches / args.steps,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 2 * N * 12, "d2h_bytes_per_step": 2 * N * 12,
                "steps": e2e_steps, "api": "ff_eval_bh_host_async + ff_host_sync (pinned host buffers, steps pipelined over three "
                                           "streams; a 192 MB L2 flush before every step is inside the timed region)",
                "dependent_calls_value": job_rate(world, N, e2e_serial_ms), "dependent_calls_ms": e2e_serial_ms,
                "which_models_what": "value: independent evaluations streamed through the host API (e.g. realisations of an "
                                     "ensemble, PAPER.md:243).  dependent_calls_value: ff_eval_bh_host one call at a time, "
                                     "what a loop pays whose next input depends on the last result.  An MD loop is of the "
                                     "second kind and should not cross PCIe at all: ff_step keeps the state resident "
                                     "(md_100_steps.ms_per_step)",
                "checksum": checksum},
        "roofline": roofline, "cpu_baseline": cpu_baseline, "parity_at_full_size": parity,
        "phases_ms": phases, "hbm_phases": hbm_phases,
        "counters": {"n_cell": n_cell, "n_particle": n_part, "n_mac_tests": n_mac,
                     "interactions_per_target": interactions / N},
        "step_ms_min_max": [min(step_ms), max(step_ms)],
    }
    if strong is not None:
        out["strong"] = strong
    out.update(extras)
    if rank == 0:
        # the same sampler over everything this invocation ran after the warm-up (timed steps, e2e, md_100_steps, the
        # other configs, the all-pairs run, the probes): sample count, median and minimum SM clock, reasons seen
        out["clocks"]["whole_run"] = sampler.summary(t_run0, time.time())
        sampler.stop()
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=None, help="particles (default: the size of the chosen config; config 3 = 2^20)")
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json config whose recipe is used (default 3, the one the metric is quoted on)")
    ap.add_argument("--quick", action="store_true", help="skip the direct kernel and the theta sweep")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
