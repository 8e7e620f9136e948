"""N>1 host logic on CPU: gloo, world_size 2 (the GPU path is replicas only -- DESIGN.md section 8)."""
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


def _torchrun(script_args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port())] + script_args
    env = dict(os.environ, OMP_NUM_THREADS="2")
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout, env=env)


def test_max_over_ranks_and_whole_job_rate(tmp_path):
    r = _torchrun([os.path.join(ROOT, "tests", "_gloo_worker.py"), str(tmp_path)])
    assert r.returncode == 0, r.stderr[-2000:]
    outs = [json.load(open(tmp_path / ("rank%d.json" % k))) for k in range(2)]
    for k, o in enumerate(outs):
        assert o["rank"] == k and o["world"] == 2
        assert o["max_ms"] == 15.0  # the slower rank decides
        assert abs(o["rate"] - 2 * 1000.0 / 0.015) < 1e-6  # units of ALL ranks / max time


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2", "--warmup", "1",
                   "--config", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["cpu_baseline"]["kind"] == "oracle"
