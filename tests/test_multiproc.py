"""N > 1 plumbing of bench.py on CPU (world_size 2, gloo): the path is single-GPU by specification, N ranks run N
independent replicas ("replicas only") and only the timing is combined -- max over ranks."""
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


def _torchrun(script_args, timeout=240, nproc=2, out_dir=None):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc), "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port())] + script_args
    env = dict(os.environ, OMP_NUM_THREADS="1")
    if out_dir is not None:
        env["AGATE_MP_OUT"] = str(out_dir)
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def _rank_files(out_dir, prefix, world):
    return [json.load(open(os.path.join(out_dir, f"{prefix}{r}.json"))) for r in range(world)]


def test_max_over_ranks_and_aggregate_rate_gloo(tmp_path):
    res = _torchrun([os.path.join("tests", "mp", "rank_helper.py")], out_dir=tmp_path)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = _rank_files(tmp_path, "rank", 2)            # one file per rank (shared stdout can interleave lines)
    assert sorted(l["rank"] for l in lines) == [0, 1]
    for l in lines:
        assert l["world"] == 2 and l["ms_max"] == 15.0                  # the slower rank sets the time
        assert abs(l["rate"] - 1000 * 2 * 4 / 15e-3) < 1e-6             # both replicas' zones count


def test_reference_arm_under_torchrun_prints_one_line():
    res = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "1"])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads(l) for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                              # rank 0 alone runs and prints
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


import pytest


@pytest.mark.parametrize("world", [2, 3])
def test_slab_halo_exchange_schedule_gloo(tmp_path, world):
    """NEXT-4: every rank receives exactly the two planes below and above its slab (wrapped when periodic, none at an
    open end), for uneven splits and for two ranks that are each other's neighbour on both faces; the v_max
    all-reduce returns the maximum."""
    res = _torchrun([os.path.join("tests", "mp", "slab_helper.py")], nproc=world, out_dir=tmp_path)
    assert res.returncode == 0, res.stderr[-2000:]
    outs = _rank_files(tmp_path, "slab_rank", world)
    for o in outs:
        assert o["world"] == world and o["vmax"] == 1.0 + 0.25 * (world - 1)
        assert len(o["cases"]) == 3
        for c in o["cases"]:
            assert c["ok"], c


def test_slab_split_and_neighbours():
    from paper_2503_20899_b200 import slab
    assert slab.split(10, 3) == [(0, 4), (4, 3), (7, 3)]
    assert slab.split(512, 8)[-1] == (448, 64)
    with pytest.raises(ValueError):
        slab.split(5, 3)
    assert slab.neighbours(0, 4, True) == (3, 1) and slab.neighbours(3, 4, True) == (2, 0)
    assert slab.neighbours(0, 4, False) == (None, 1) and slab.neighbours(3, 4, False) == (2, None)
    assert slab.neighbours(0, 1, True) == (0, 0) and slab.neighbours(0, 1, False) == (None, None)
