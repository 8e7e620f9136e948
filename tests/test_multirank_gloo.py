"""N>1 host logic on CPU over gloo: the max-over-ranks / whole-job arithmetic of the replica mode, the reference arm under
torchrun, and the face exchange of the T-slab mode (world sizes 2 and 3) -- DESIGN.md section 8."""
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


def _torchrun(script_args, timeout=300, nproc=2):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc), "--master-addr", "127.0.0.1",
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


import pytest  # noqa: E402


@pytest.mark.parametrize("world", [2, 3])
def test_slab_face_exchange_over_gloo(tmp_path, world):
    """A rank's face DOWN must arrive as the face_from_above of the rank below, its face UP as the face_from_below of the rank
    above (periodic ring in t).  world = 2 is the case where both neighbours are the same peer and message order does the
    matching."""
    r = _torchrun([os.path.join(ROOT, "tests", "_gloo_slab_worker.py"), str(tmp_path)], nproc=world)
    assert r.returncode == 0, r.stderr[-2000:]
    for k in range(world):
        o = json.load(open(tmp_path / ("slab_rank%d.json" % k)))
        assert o["world"] == world and o["up"] == (k + 1) % world and o["down"] == (k - 1) % world and o["t0"] == k * o["lt"]
        assert o["sent_intact"]
        assert o["above_min"] == o["above_max"] == 10 * ((k + 1) % world) + 1  # the face DOWN of the rank above
        assert o["below_min"] == o["below_max"] == 10 * ((k - 1) % world) + 2  # the face UP of the rank below
