"""The N > 1 launch path of bench.py on CPU: under torchrun with two processes the reference arm must run on rank 0 alone
and print exactly one JSON line (the all-reduce of the sharded build is covered by tests/test_shard_allreduce.py); the
flop model of the roofline is checked against hand counts."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_under_torchrun_two_ranks():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29731", os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--workload", "tiny",
           "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["workload"] == "tiny" and d["gpu_launches"] == 0


def test_flop_model_hand_counts():
    sys.path.insert(0, ROOT)
    import bench
    # (ss|ss): two Boys values (60 flop), no recursion, one E term each side: 60 + 2*(1 + 1 + 1)
    assert bench.flops_k(0, 0, 0, 0) == 66
    assert bench.flops_j(0, 0) == 62
    # eq 47-49 at L = 1: three multiplications
    assert bench.flops_base(1) == 66 + 3
    # K (pp|pp): h(2) = 10 Hermite functions, 33 non-zero E terms per pp pair, 9 x 9 components
    assert bench.flops_k(1, 1, 1, 1) == bench.flops_base(4) + 2 * (10 * 33 + 9 * 33 + 81)
    assert bench._eterms(2, 2) == 336 and bench._eterms(1, 1) == 33 and bench._eterms(0, 0) == 1
