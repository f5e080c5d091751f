"""The N>1 path of bench.py on CPU: two gloo ranks (replicas only) -- max over ranks of the
timed region, aggregate value, launch count summed; the --impl reference arm under torchrun (rank 0
alone works and prints, the other rank exits 0); and `bench.py --gpus N` starting its own N ranks."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def torchrun(args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port())] + args
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="2")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_replica_aggregation_two_gloo_ranks():
    out = torchrun([os.path.join("tests", "_dist_worker.py")])
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("RESULT ")]
    assert len(line) == 1
    r = json.loads(line[0][7:])
    assert r["ms_total"] == 140.0                  # the slowest rank bounds the region
    assert abs(r["ms_step"] - 7.0) < 1e-12
    assert abs(r["value"] - 0.0035) < 1e-15        # 2 replicas x 20 iterations in 0.140 s
    assert r["launches"] == 171


def test_reference_arm_under_torchrun_runs_on_rank0_only():
    out = torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "3", "--warmup", "1",
                    "--workload", "config1_4^4"])
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    r = json.loads(lines[0])
    assert r["impl"] == "reference" and r["unit"] == "s/iter" and r["value"] > 0
    assert r["cpu_baseline"]["kind"] == "oracle" and r["cpu_baseline"]["value"] == r["value"]
    assert r["e2e"] == {"value": r["value"], "unit": "s/iter", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert r["higher_is_better"] is False and r["n_gpus"] == 2


def bench_direct(args, timeout=300):
    """`python bench.py ...` as the driver calls it for N > 1 when it does not wrap it in torchrun itself"""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    env.update(CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="2")
    return subprocess.run([sys.executable, "bench.py"] + args, cwd=ROOT, env=env, capture_output=True, text=True,
                          timeout=timeout)


def test_gpus_n_starts_its_own_ranks():
    """--gpus 2 outside torchrun: bench.py re-executes itself under torch.distributed.run with 2 ranks.  The
    plumbing check is the part of that path that needs neither a GPU nor the library (gloo)."""
    out = bench_direct(["--gpus", "2", "--steps", "20", "--plumbing-check"])
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    r = json.loads(lines[0])
    assert r["n_gpus"] == 2 and r["plumbing_check"] is True
    assert r["ms_total"] == 20.0 and abs(r["value"] - 0.0005) < 1e-15 and r["launches"] == 201


def test_gpus_n_without_n_devices_fails_loudly():
    """never a line with fewer GPUs than asked: no devices here, so --gpus 2 must exit non-zero and print no JSON"""
    out = bench_direct(["--gpus", "2", "--quick", "--steps", "4", "--warmup", "3"])
    assert out.returncode != 0
    assert "needs 2 CUDA devices" in out.stderr
    assert not [l for l in out.stdout.splitlines() if l.startswith("{")]


def test_world_size_must_match_gpus():
    out = torchrun(["bench.py", "--gpus", "4", "--plumbing-check"])
    assert out.returncode != 0 and "WORLD_SIZE=2" in out.stderr
