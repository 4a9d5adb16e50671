"""N > 1 host logic on CPU: world_size 2, gloo, launched exactly as the driver launches bench.py."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def test_two_rank_gloo_max_over_ranks_and_aggregate():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "tests", "_gloo_worker.py")]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    line = [l for l in res.stdout.splitlines() if l.startswith("{")][-1]
    out = json.loads(line)
    assert out["world"] == 2
    assert out["ms"] == 15.0                              # max over ranks, not rank 0's 10 ms
    assert out["ok"] is False and out["ok2"] is True
    assert abs(out["value"] - 2 * 1000 * 3 * 4 / 15e-3) < 1e-6


def test_reference_arm_prints_contract_line():
    """bench.py --impl reference runs the oracle on the host cores and prints the JSON contract line."""
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                          "--workload", "small_1d2v_128^3"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    out = json.loads([l for l in res.stdout.splitlines() if l.startswith("{")][-1])
    assert out["impl"] == "reference" and out["cpu_baseline"]["kind"] == "oracle" and out["value"] > 0
    assert out["e2e"]["h2d_bytes_per_step"] == 0 and out["unit"] == "DOF-updates/s"
