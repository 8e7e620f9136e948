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
def test_slab_halo_exchange_over_gloo(tmp_path, world):
    """Each rank's ghost slices must end up holding the neighbouring rank's boundary slices (periodic ring in t).
    world = 2 is the case where both neighbours are the same peer and message order does the matching."""
    r = _torchrun([os.path.join(ROOT, "tests", "_gloo_slab_worker.py"), str(tmp_path)], nproc=world)
    assert r.returncode == 0, r.stderr[-2000:]
    for k in range(world):
        o = json.load(open(tmp_path / ("slab_rank%d.json" % k)))
        lt = o["lt"]
        assert o["world"] == world and o["up"] == (k + 1) % world and o["down"] == (k - 1) % world
        assert o["interior_ok"]
        # lower ghost = last interior slice (index lt) of the rank below; upper ghost = slice 1 of the rank above
        assert o["lo_min"] == o["lo_max"] == 10 * ((k - 1) % world) + lt
        assert o["hi_min"] == o["hi_max"] == 10 * ((k + 1) % world) + 1


def test_slab_geometry_and_message_plan():
    from paper_2301_03636_b200 import slab
    g = slab.SlabGeometry((8, 4, 4, 12), 3, 1)
    assert g.lt == 4 and g.t0 == 4 and g.local_dims == (8, 4, 4, 6) and (g.up, g.down) == (2, 0)
    assert g.slice_bytes("spinor", "f64", "soa", False) == 128 * 192
    assert g.slice_bytes("gauge", "f32", "aos", True) == 128 * 48 * 4
    assert [m[0] for m in slab.halo_messages(g)] == ["send", "send", "recv", "recv"]
    with pytest.raises(ValueError):
        slab.SlabGeometry((8, 4, 4, 10), 3, 0)  # L_T not divisible
    with pytest.raises(ValueError):
        slab.SlabGeometry((3, 3, 3, 4), 2, 0).slice_bytes("spinor", "f64", "soa", False)  # 27 sites per slice
    # in-process exchange (the single-GPU emulation) moves the same slices
    import torch
    world, nb = 3, 16
    geoms = [slab.SlabGeometry((2, 2, 2, 6), world, r) for r in range(world)]
    bufs = [torch.zeros((geoms[r].lt + 2) * nb, dtype=torch.uint8) for r in range(world)]
    for r in range(world):
        for k in range(1, geoms[r].lt + 1):
            bufs[r][k * nb:(k + 1) * nb] = 10 * r + k
    slab.exchange_halos_in_process(bufs, geoms, nb)
    for r in range(world):
        assert int(bufs[r][0]) == 10 * ((r - 1) % world) + geoms[r].lt and int(bufs[r][-1]) == 10 * ((r + 1) % world) + 1
    one = slab.SlabGeometry((2, 2, 2, 4), 1, 0)
    b = torch.arange(6 * nb, dtype=torch.uint8)
    ref = b.clone()
    assert slab.exchange_halos(b, one, nb) == []
    assert torch.equal(b[:nb], ref[4 * nb:5 * nb]) and torch.equal(b[5 * nb:], ref[nb:2 * nb])
