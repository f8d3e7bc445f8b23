"""N>1 launch path on CPU: world_size-2 gloo run of bench.py's rank logic, and the reference arm under torchrun."""
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


def _torchrun(script_args, timeout=600):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + script_args
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout)


def test_gloo_two_ranks_max_and_aggregate():
    r = _torchrun([os.path.join("tests", "helpers", "gloo_ranks.py")])
    assert r.returncode == 0, r.stderr[-2000:]
    rate = [l for l in r.stdout.splitlines() if l.startswith("RATE")]
    assert len(rate) == 1
    # 2 replicas x 81920 state-steps x 4 steps / 11 ms
    assert abs(float(rate[0].split()[1]) - 2 * 256 * 16 * 20 * 4 / 11e-3) < 1e-3


def test_gloo_two_ranks_k_sharded_step_host_logic():
    r = _torchrun([os.path.join("tests", "helpers", "gloo_sharded.py")])
    assert r.returncode == 0, r.stderr[-2000:]
    assert any(l.startswith("SHARDED_OK") for l in r.stdout.splitlines())


def test_reference_arm_under_torchrun_prints_one_line():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                   "--workload", "C0"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                      # rank 0 alone prints; the other rank exits 0 without work
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["n_gpus"] == 2
