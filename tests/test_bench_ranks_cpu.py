"""Host logic of `bench.py --gpus N` on CPU: world_size-2 gloo process group -> barrier, max over
ranks of the per-rank time, whole-job value, distinct replica seeds; and the reference arm under a
2-rank launch (rank 0 alone works, the other rank exits 0 without output).  DESIGN.md section 9."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch
    import bench
    synced = []
    grp = bench.RankGroup(rank, world, backend="gloo", device=torch.device("cpu"), sync=lambda: synced.append(1))
    grp.barrier()
    ms = grp.max_over_ranks(10.0 * (rank + 1))          # rank r "measured" 10 (r+1) ms
    grp.barrier()
    out[rank] = (ms, bench.whole_job_value(world, 64 * 64, 5, ms), bench.replica_seed(13, rank), len(synced))
    grp.close()


def test_rank_group_gloo_world2():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for r in (0, 1):
        ms, value, seed, nsync = res[r]
        assert ms == 20.0                                  # the slowest rank's time, on every rank
        assert value == pytest.approx(2 * 64 * 64 * 5 / 20e-3)
        assert seed == 13 + r
        assert nsync == 2
    assert res[0][2] != res[1][2]


def test_single_rank_group_is_local():
    sys.path.insert(0, ROOT)
    import bench
    grp = bench.RankGroup(0, 1)
    grp.barrier()
    assert grp.max_over_ranks(3.5) == 3.5
    grp.close()


def test_reference_arm_rank1_exits_quietly():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_rank0_line():
    env = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["metric"] == "SW spin updates/s" and line["higher_is_better"] is True
