"""Host-side logic of bench.py that needs no GPU: the replicas-only aggregation over ranks (gloo,
world_size 2), the oracle crop sampler, and the --impl reference arm's JSON contract."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sys.path.insert(0, ROOT)
    import bench
    # rank r "measured" (10 + 5 r) ms for 1000 (r + 1) units
    ms, units = bench.aggregate(10.0 + 5.0 * rank, 1000 * (rank + 1), world, dist, None)
    dist.barrier()
    q.put((rank, ms, units))
    dist.destroy_process_group()


def test_aggregate_max_time_total_units_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, units in res:
        assert ms == 15.0 and units == 3000.0      # max over ranks, sum of units: value = 3000 / 15 ms


def test_aggregate_single_rank_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(3.5, 42, 1) == (3.5, 42)


def test_crop_config_is_a_dense_corner():
    sys.path.insert(0, ROOT)
    import bench
    from paper_1911_07045_b200 import workloads as wl
    c = wl.make_replica("5p")
    s = bench.crop_config(c, 20)
    assert (s["Lx"], s["Ly"], s["Lz"]) == (20, 20, 20) and s["q"].shape == (5, 8000)
    q3 = c["q"].reshape(5, c["Lz"], c["Ly"], c["Lx"])[:, :20, :20, :20]
    assert np.array_equal(s["q"].reshape(5, 20, 20, 20), q3)
    assert s["mask"].sum() == 400                   # the z = 0 wall layer of the crop


def test_reference_arm_json_contract():
    """bench.py --impl reference runs the oracle on host cores and prints the contract's line"""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "1",
                          "--steps", "2", "--warmup", "1", "--ref-crop", "16"], capture_output=True, text=True,
                         timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "site-updates/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["dtype"] == "f64" and line["vs_baseline"] is None


def test_reference_arm_nonzero_rank_is_silent():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "1",
                          "--steps", "1", "--warmup", "1", "--ref-crop", "8"], capture_output=True, text=True,
                         timeout=300, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
