"""CPU tests of bench.py's plumbing: the N>1 launch path (torchrun, gloo, world_size 2: barrier,
max-over-ranks, whole-job aggregation) and the --impl reference arm (the oracle on host cores)."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def torchrun(n, *bench_args):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n),
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.join(ROOT, "bench.py")] + list(bench_args)
    env = dict(os.environ, OMP_NUM_THREADS="2")
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    return [json.loads(l) for l in lines]


def test_world_size_2_gloo_aggregation():
    out = torchrun(2, "--gpus", "2", "--steps", "4", "--warmup", "3", "--dist-dry-run")
    assert len(out) == 1                                     # rank 0 alone prints
    line = out[0]
    # ranks pretend 10 ms and 20 ms: the job time is the max, the value counts both ranks' cells
    assert line["n_gpus"] == 2 and line["scaling"] == "weak"
    assert abs(line["ms_per_step"] - 20.0 / 4) < 1e-9
    assert abs(line["value"] - 1000 * 4 * 2 / 0.020 / 1e6) < 1e-9


def test_reference_arm_under_torchrun_prints_once():
    out = torchrun(2, "--gpus", "2", "--steps", "2", "--warmup", "1", "--impl", "reference", "--config", "1")
    assert len(out) == 1
    line = out[0]
    assert line["impl"] == "reference" and line["unit"] == "MLUPS" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["value"] == line["value"] and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["gpu_launches"] == 0


def test_aggregate_is_whole_job():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(1_000_000, 10, 8, 0.5) == 1_000_000 * 10 * 8 / 0.5 / 1e6
