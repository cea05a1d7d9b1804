"""world_size-2 test of bench.py's multi-rank host logic on the CPU (gloo), launched the way the driver
launches the GPU bench: python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(nproc, script_args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc),
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + script_args
    env = dict(os.environ, OMP_NUM_THREADS="2")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_two_rank_replicas_max_time_and_job_rate(tmp_path):
    r = _torchrun(2, [os.path.join(ROOT, "tests", "rank_worker.py"), str(tmp_path)])
    assert r.returncode == 0, r.stderr[-2000:]
    recs = [json.load(open(tmp_path / ("rank%d.json" % k))) for k in range(2)]
    assert [x["rank"] for x in recs] == [0, 1] and all(x["world"] == 2 for x in recs)
    # every rank sees the slowest rank's time, and the job rate counts the units of both replicas
    assert all(x["ms"] == 20.0 for x in recs)
    assert all(abs(x["rate"] - 2 * 2048 / 20e-3) < 1e-6 for x in recs)
    # independent replicas: same recipe and size, different seed
    assert recs[0]["N"] == recs[1]["N"] == 2048 and recs[0]["pos_sum"] != recs[1]["pos_sum"]
    # target sharding: the all-gather re-assembles the common ensemble on every rank, the group slices tile it
    assert all(x["gather_ok"] for x in recs)
    assert recs[0]["groups"] == [0, 32] and recs[1]["groups"] == [32, 64]
    assert recs[0]["groups64"] == [0, 16] and recs[1]["groups64"] == [16, 32]
    # exactly one JSON line, from rank 0, carrying both measurements: the weak-scaling headline and the "strong" block
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak"
    st = d["strong"]
    assert st["scaling"] == "strong" and st["n_gpus"] == 2 and st["N"] == 2048
    assert st["ms_per_step"] == 12.5                                   # max over ranks of (12.5, 11.5)
    assert abs(st["value"] - 2048 / 12.5e-3) < 1e-6                    # ONE ensemble: N, not world * N
    assert abs(st["efficiency_vs_one_gpu"] - (20.0 / 2) / 12.5) < 1e-12
    assert {"allgather_ms", "walk_ms_max_over_ranks", "one_gpu_ms_per_step", "phases_ms_rank0"} <= set(st)


def test_reference_arm_runs_on_rank_zero_only():
    r = _torchrun(2, [os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                      "--warmup", "0", "--config", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["n_gpus"] == 2
