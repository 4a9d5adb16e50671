"""N > 1 host logic on CPU: world_size 2, gloo, launched exactly as the driver launches bench.py."""
import json
import os
import socket
import subprocess
import sys

import pytest

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


def test_bench_gpus_2_starts_two_ranks_itself():
    """`python bench.py --gpus 2` without a torchrun environment starts the two ranks itself; the line says n_gpus = 2
    (reference arm: rank 0 alone runs the oracle, the other rank exits 0 without work)."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--workload", "small_1d2v_128^3"], capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # rank 0 only
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["impl"] == "reference"


def test_xslab_partition():
    sys.path.insert(0, ROOT)
    from paper_2202_13532_b200 import sharded
    assert sharded.slab_partition(64, 8) == [(8 * r, 8 * r + 8) for r in range(8)]
    parts = sharded.slab_partition(5, 2)
    assert parts == [(0, 2), (2, 5)]
    for N, w in ((7, 3), (64, 5), (3, 3)):
        p = sharded.slab_partition(N, w)
        assert p[0][0] == 0 and p[-1][1] == N and all(a[1] == b[0] for a, b in zip(p, p[1:])) and all(b > a for a, b in p)
    import pytest
    with pytest.raises(ValueError):
        sharded.slab_partition(2, 3)
    lo, hi = sharded.slab_bounds(0.0, 10.0, 5, 2, 5)
    assert (lo, hi) == (4.0, 10.0)


def test_xslab_world1_wraps_through_the_halo_planes():
    """world = 1: the periodic roll goes through exchange_faces -> halo planes; must equal the unsharded oracle."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import _xslab_worker as xw
    for sc in (True, False):
        err, part = xw.run_sharded(0, 1, self_consistent=sc)
        assert part == (0, 5) and err <= 1e-13, (sc, err)
    err, _ = xw.run_sharded(0, 1, self_consistent=False, bc0=1)
    assert err <= 1e-13


@pytest.mark.parametrize("transport", ["direct", "hoststaged"])
def test_xslab_two_rank_gloo_matches_unsharded_oracle(transport):
    """world = 2 over gloo, uneven slabs (2 + 3 x-elements): face-plane exchange + all-gather of rho; through TorchDistComm
    and through HostStagedComm (the transport of the two-processes-on-one-GPU test)."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "tests", "_xslab_worker.py"), transport]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-3000:]
    out = json.loads([l for l in res.stdout.splitlines() if l.startswith("{")][-1])
    assert out["world"] == 2 and out["parts"] == [[0, 2], [2, 5]]
    assert out["err_sc1_bc0"] <= 1e-13 and out["err_sc0_bc0"] <= 1e-13 and out["err_sc0_bc1"] <= 1e-13, out
