#!/usr/bin/env python
"""bench.py -- the headline measurement of BASELINE.json:

    dipole field+force particle-evals/s & ms/step at N = 2^20, theta = 0.5; FP32-pipe % of peak

One "step" = one pass of the whole hot path: ff_build_tree
(bounding box, Morton keys, radix sort, octree) + ff_eval_bh (cell moments, tree walk, scatter to
caller order) on config 3 (1 048 576 hard-sphere dipoles, volume fraction 0.1, isotropic moments),
inputs resident in HBM.  Prints ONE JSON line (see the driver contract in the task statement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n N] [--quick]

N > 1: launched under torchrun, one rank per GPU; every rank runs an independent replica of the
workload with its own seed (the paper averages over independent realisations), no
data-path collective, "scaling": "weak".
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
FLOP_PER_INTERACTION = 60.0      # 21 FFMA x2 + 17 FADD/FMUL + 1 MUFU.RSQ per h+f pair term
FP32_LANES_PER_SM = 128
# dram__bytes_read.sum + dram__bytes_write.sum of one ff_k_walk launch at config 3, from the
# `ncu --set full` capture summarised in profiles/ (None until a capture exists)
WALK_DRAM_TRAFFIC_BYTES = 107508480   # 84.74 MB read + 22.76 MB written (profiles/r1_walk_full.md)


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
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.rows:
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
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


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


def job_rate(world, units_per_rank, ms):
    """Whole-job throughput: every rank processed `units_per_rank` units (weak scaling, independent replicas,
    no data-path collective) in `ms`, the max over ranks."""
    return world * units_per_rank / (ms * 1e-3)


def _describe(c):
    kind = {1: "hard-sphere dipoles (d=1), phi=0.05, isotropic unit moments",
            2: "hard-sphere dipoles (d=1), phi=0.1, von Mises-Fisher moments about +z (kappa=5)",
            3: "hard-sphere dipoles (d=1), phi=0.1, isotropic unit moments",
            4: "straight head-to-tail chains of 32 touching spheres within 15 deg of z, moments along the chain",
            5: "hard-sphere dipoles (d=1), phi=0.2, isotropic unit moments"}[c["config"]]
    return "config %d of BASELINE.json: N=%d %s, theta=%g" % (c["config"], c["N"], kind, c["theta"])


def _oracle_step(c, groups, nthreads=0):
    """One oracle pass on a bounded sample: full tree + moments, walk of `groups` only.
    Returns (t_build, t_moments, t_walk)."""
    import oracle
    t0 = time.perf_counter()
    t = oracle.Tree(c["pos"])
    t1 = time.perf_counter()
    t.moments(c["mom"])
    t2 = time.perf_counter()
    t.eval(c["theta"], 32, groups=groups, nthreads=nthreads)
    t3 = time.perf_counter()
    return t1 - t0, t2 - t1, t3 - t2


def _oracle_rate(c, n_groups_sample, nthreads=0):
    """Extrapolated whole-job particle-evals/s of the oracle from a bounded sample."""
    N = c["N"]
    n_groups = (N + 31) // 32
    groups = np.random.default_rng(0).choice(n_groups, min(n_groups_sample, n_groups), replace=False)
    tb, tm, tw = _oracle_step(c, groups, nthreads)
    full = tb + tm + tw * n_groups / len(groups)
    return N / full, dict(t_build_s=tb, t_moments_s=tm, t_walk_sample_s=tw, groups=int(len(groups)))


def run_reference(args):
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    c = _workload(args.n, 0, args.config)
    cores = oracle.max_threads()
    n_groups = (c["N"] + 31) // 32
    sample = min(n_groups, 1024)
    for _ in range(args.warmup):
        _oracle_rate(c, sample)
    t0 = time.perf_counter()
    rates = [_oracle_rate(c, sample)[0] for _ in range(args.steps)]
    wall = time.perf_counter() - t0
    value = float(np.mean(rates))
    desc = ("fp64 oracle (oracle/ff_oracle.c), per step: full tree build + cell moments over all N, walk of %d sampled "
            "groups of 32 targets, walk time extrapolated to all %d groups" % (sample, n_groups))
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * c["N"] / value, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": _describe(c) + ", group rule W=32", "N": c["N"], "theta": c["theta"]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "wall_s": wall,
    }
    print(json.dumps(out))


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

    sharded = args.shard == "targets" and world > 1
    # replicas: an independent realisation per rank; target sharding: ONE ensemble, every rank owns N / world rows
    c = _workload(args.n, 0 if sharded else rank, args.config)
    N, theta = c["N"], c["theta"]
    pos_h = torch.from_numpy(c["pos"]).pin_memory()
    mom_h = torch.from_numpy(c["mom"]).pin_memory()
    pos, mom = pos_h.to(dev), mom_h.to(dev)
    H, F = torch.empty_like(pos), torch.empty_like(pos)
    ctx = ff.FFContext(N, theta, device=dev, timing=True)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    if sharded:
        assert N % world == 0, "target sharding needs N divisible by the number of ranks"
        rows = slice(rank * (N // world), (rank + 1) * (N // world))
        pos_local, mom_local = pos[rows].clone(), mom[rows].clone()
        g_begin, g_end = ff.shard_groups(N, world, rank)

    def step():
        if sharded:
            p_all, m_all = gather_particles(pos_local, world), gather_particles(mom_local, world)
            ctx.build_tree(p_all)
            ctx.eval_bh_range(p_all, m_all, H, F, g_begin, g_end)
        else:
            ctx.build_tree(pos)
            ctx.eval_bh(pos, mom, H, F)

    # interaction counts of this workload (separate, untimed run of the counting kernel variant)
    ctx.set_option(ff.FF_OPT_COUNTERS, 1)
    step()
    n_cell, n_part, n_mac = ctx.counters()
    ctx.set_option(ff.FF_OPT_COUNTERS, 0)
    interactions = n_cell + n_part

    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        step()
    torch.cuda.synchronize()
    ctx.timings()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    phases = {k: 0.0 for k in ff.PHASES}
    l0 = ctx.launch_count()
    t_wall0 = time.time()
    for i in range(args.steps):
        flush.zero_()                                  # evict the previous step from L2 (not timed)
        ev[i][0].record()
        step()
        ev[i][1].record()
        ev[i][1].synchronize()
        for k, v in ctx.timings().items():
            phases[k] += v
    torch.cuda.synchronize()
    t_wall1 = time.time()
    launches = ctx.launch_count() - l0
    if world > 1:
        dist.barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = max_over_ranks(sum(step_ms), world, dev)
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    ms_per_step = total_ms / args.steps
    value = job_rate(1 if sharded else world, N, ms_per_step)     # sharded: the ranks share ONE ensemble of N
    phases = {k: v / args.steps for k, v in phases.items()}

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
    # the same call, one step at a time (upload, compute, download strictly in sequence)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(3):
        ctx.eval_bh_host(pos_h, mom_h, H_h[0], F_h[0])
    e2e_serial_ms = (time.perf_counter() - t0) * 1e3 / 3
    H_h, F_h = H_h[0], F_h[0]
    # (with --shard targets this stays the single-GPU host call of every rank: reported per GPU, not summed)
    e2e_value = job_rate(1 if sharded else world, N, max_over_ranks(e2e_ms, world, dev) / e2e_steps)
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
    fma_peak = ctx.measure_fp32_peak(1 << 14)
    roofline = {
        "bound": "alu", "kernel": "ff_k_walk", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": achieved / peak_tflops, "traffic": WALK_DRAM_TRAFFIC_BYTES,
        "peak_source": "nominal: %d SMs x 128 FP32 lanes x 2 flop x %.0f MHz (clocks.max.sm); MEASURED_PEAKS.json (%s) "
                       "holds no FP32 figure" % (num_sms, sm_max, peak_src),
        "measured_fma_peak_tflops": fma_peak, "frac_of_measured_fma": achieved / fma_peak,
        "interactions_per_launch": interactions, "flop_per_interaction": FLOP_PER_INTERACTION,
        "kernel_ms": walk_ms, "kernel_share_of_step": walk_ms / ms_per_step,
        "interactions_per_s": interactions / (walk_ms * 1e-3),
        # FP32-pipe occupancy by the interaction arithmetic alone = interactions x 38 FP32 lane-ops
        # (19 packed instructions of two lanes' worth each) / (time x SMs x 128 lanes x clock)
        "fp32_lane_ops_per_interaction": 38,
        "fp32_lane_occupancy_by_interactions": interactions * 38.0 / (walk_ms * 1e-3 * num_sms * FP32_LANES_PER_SM * sm_max * 1e6),
        "note": "21 of the 38 FP32 instructions per interaction are FMAs, so a saturated FP32 pipe reads 0.78; packed "
                "FFMA2 with three register-pair operands issues every 3 cycles (profiles/r1_walk_full.md), which caps "
                "this instruction mix near 0.60",
    }
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    # algorithmic bytes per particle of the HBM-bound phases (DESIGN.md / SURVEY.md 8(d))
    alg_bytes = {"bbox_keys": 12 + 12 + 4, "sort": 4 * 16 + 4 + 12 + 16, "build": 26, "moments": 12 + 16 + 122}
    hbm_phases = {k: {"ms": phases[k], "achieved_gbs": alg_bytes[k] * N / (phases[k] * 1e-3) / 1e9,
                      "frac_of_hbm_peak": alg_bytes[k] * N / (phases[k] * 1e-3) / 1e9 / hbm}
                  for k in alg_bytes if phases[k] > 0}

    extras = {}
    if not args.quick and not sharded and N <= (1 << 21):                  # the N^2 kernel takes minutes beyond that
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
        eH = float((np.linalg.norm(Hs - Ha, axis=1) / np.maximum(np.linalg.norm(Ha, axis=1), Qa[:, 0] / 8)).max())
        eF = float((np.linalg.norm(Fs - Fa, axis=1) / np.maximum(np.linalg.norm(Fa, axis=1), Qa[:, 1] / 8)).max())
        extras["gpu_direct"].update({
            "max_err_vs_oracle_allpairs": {"H": eH, "F": eF, "targets": int(len(tsel)), "tolerance": 1e-5},
            "cpu_allpairs_oracle": {"pairs_per_s": len(tsel) * (N - 1) / t_ap, "cores": _oracle.max_threads(),
                                    "extrapolated_s_per_eval": t_ap * N / len(tsel),
                                    "sample": "%d targets x all sources, fp64" % len(tsel)}})
        errs = {}
        for th in (0.3, 0.5, 0.7):
            ctx.set_option(ff.FF_OPT_THETA, th)
            Hb, Fb = ctx.eval_bh(pos, mom)
            errs[str(th)] = {"H_rel_l2": float((Hb - Hd).double().norm() / Hd.double().norm()),
                             "F_rel_l2": float((Fb - Fd).double().norm() / Fd.double().norm())}
        ctx.set_option(ff.FF_OPT_THETA, theta)
        extras["bh_vs_allpairs_error"] = {"reference": "GPU direct kernel (ff_eval_direct)", "by_theta": errs}

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
        # Lennard-Jones force, Euler-Maruyama update, dtau = 0.001 as in PAPER.md:200), per-phase timing
        prm = ff.ff_step_params()
        prm.dtau, prm.gamma_d, prm.gamma_r = 1e-3, 1.0, 1.0
        prm.h_ext[0], prm.h_ext[1], prm.h_ext[2] = 0.0, 0.0, 0.5
        prm.lj_epsilon, prm.lj_sigma, prm.lj_cutoff = 1.0, 1.0, 2.5
        prm.noise_d, prm.noise_r, prm.seed = 0.05, 0.05, 1
        x, u = pos.clone(), mom.clone()
        v, w = torch.zeros_like(pos), torch.zeros_like(pos)
        for s in range(3):
            ctx.step(x, v, u, w, prm, s)
        torch.cuda.synchronize()
        ctx.timings()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        md_steps = 100
        e0.record()
        for s in range(md_steps):
            ctx.step(x, v, u, w, prm, 3 + s)
        e1.record()
        torch.cuda.synchronize()
        md_ms = e0.elapsed_time(e1) / md_steps
        last = ctx.timings()
        extras["md_100_steps"] = {
            "ms_per_step": md_ms, "particle_steps_per_s": N / (md_ms * 1e-3), "steps": md_steps,
            "phases_ms_last_step": last, "finite": bool(torch.isfinite(x).all() and torch.isfinite(u).all()),
            "params": {"dtau": 1e-3, "gamma_d": 1.0, "gamma_r": 1.0, "h_ext": [0, 0, 0.5], "lj": [1.0, 1.0, 2.5],
                       "noise": [0.05, 0.05]},
            "note": "L2 not flushed between these steps (back-to-back MD steps, as in a simulation)"}

    # ---- parity of this very run at full size: the oracle's Barnes-Hut on sampled groups (DESIGN.md section 6 metric)
    import oracle
    otree = oracle.Tree(c["pos"])
    otree.moments(c["mom"])
    g_lo, g_hi = (g_begin, g_end) if sharded else (0, (N + 31) // 32)
    sel = g_lo + np.random.default_rng(7).choice(g_hi - g_lo, min(256, g_hi - g_lo), replace=False)
    Ho, Fo, _, Qo = otree.eval(theta, 32, groups=sel, scale=True)
    _, operm = otree.keys()
    rows = operm[(sel[:, None] * 32 + np.arange(32)[None, :]).ravel().clip(max=N - 1)]
    rows = np.unique(rows)
    Hg, Fg = H.cpu().numpy().astype(np.float64), F.cpu().numpy().astype(np.float64)

    def _errs(x, ref, q):
        e = np.linalg.norm(x - ref, axis=1) / np.maximum(np.linalg.norm(ref, axis=1), q / 8.0)
        return {"max": float(e.max()), "p99": float(np.quantile(e, 0.99)), "median": float(np.median(e)),
                "global_rel_l2": float(np.linalg.norm(x - ref) / np.linalg.norm(ref))}
    parity = {"targets": int(len(rows)), "tolerance": 1e-4,
              "H": _errs(Hg[rows], Ho[rows], Qo[rows, 0]), "F": _errs(Fg[rows], Fo[rows], Qo[rows, 1]),
              "metric": "|x_k - ref_k| / max(|ref_k|, Q_k / 8) against the fp64 oracle's Barnes-Hut (same theta, W = 32)"}
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
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if sharded else "weak",
        "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": _describe(c) + ", tree rebuilt every step, H and F",
                   "N": N, "theta": theta, "group": 32, "nleaf": 1, "l2": "flushed between timed steps (512 MB memset)",
                   "replicas": 1 if sharded else world,
                   "sharding": "targets: one ensemble, all-gather of pos and mom per step, redundant tree, each rank walks "
                               "a Morton-contiguous slice of the groups" if sharded else "independent replicas, no collective"},
        "clocks": clocks, "gpu_launches": int(launches), "launches_per_step": launches / args.steps,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 2 * N * 12, "d2h_bytes_per_step": 2 * N * 12,
                "steps": e2e_steps, "api": "ff_eval_bh_host_async + ff_host_sync (pinned host buffers, steps pipelined over three "
                                           "streams; a 192 MB L2 flush before every step is inside the timed region)",
                "one_step_at_a_time_ms": e2e_serial_ms, "checksum": checksum},
        "roofline": roofline, "cpu_baseline": cpu_baseline, "parity_at_full_size": parity,
        "phases_ms": phases, "hbm_phases": hbm_phases,
        "counters": {"n_cell": n_cell, "n_particle": n_part, "n_mac_tests": n_mac,
                     "interactions_per_target": interactions / N},
        "step_ms_min_max": [min(step_ms), max(step_ms)],
    }
    out.update(extras)
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
    ap.add_argument("--shard", default="replicas", choices=["replicas", "targets"],
                    help="N > 1: independent replicas per rank (default, weak scaling) or one ensemble with the "
                         "targets sharded over the ranks (all-gather of pos and mom per step, strong scaling)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
