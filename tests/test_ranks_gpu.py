"""The one-rank-per-process driver of the z-slab decomposition ("each processing unit
is assigned to one of these subregions" and halo sites are communicated every step), actually run by several
processes: parallel.fire_minimize_rank on 2 and 3 ranks, each rank its own process with its own CUDA context on the one
GPU, gloo transport with host-staged halo packages and reduction rows (no kernel ever waits on another process: every
wait is a host wait inside gloo).  Gathered Q after 60 steps must match the ORACLE to 1e-8 and be bit-identical to the
same-process C group driver lq_slabs_fire_minimize (same sweeps, same rank-ordered reduction); velocities and the
schedule scalars are checked too.  The NCCL transport (staging="device") shares every line of the driver but the
buffer placement; it needs one GPU per rank and stays unmeasured on hardware."""
import os
import socket

import numpy as np
import pytest

from paper_1911_07045_b200 import parallel, workloads as wl

pytestmark = pytest.mark.gpu
TOL_Q = 1e-8
STEPS = 60

CASES = {
    "replica4": lambda: wl.make_replica("4"),      # periodic one-constant lattice: recompute sweep, one halo round per step
    "replica3": lambda: wl.make_replica("3"),      # L1+L2+L3, walls + colloid: stored force + fix-up, two halo rounds
    "replica5p": lambda: wl.make_replica("5p"),    # masked one-constant, Eq. 14 + 15 anchoring at the outer slab faces
}


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _rank_worker(rank, world, port, name, integrator, outdir):
    import torch
    import torch.distributed as dist
    from paper_1911_07045_b200 import binding as lq
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        lq.load()
        c = CASES[name]()
        z0, nz = parallel.split_z(c["Lz"], world)[rank]
        ctx = parallel.make_slab(lq, c, z0, nz)
        if rank == world - 1:                        # one rank on a stream of its own: the driver must follow it
            side = torch.cuda.Stream()
            lq.lq_set_stream(ctx, side.cuda_stream)
        rep = parallel.fire_minimize_rank(lq, ctx, parallel.DistComm(dist, rank, world), STEPS, 0.0,
                                          dict(c["fire"], integrator=integrator), staging="host")
        np.savez(os.path.join(outdir, "rank%d.npz" % rank), q=lq.lq_get_Q(ctx), v=lq.lq_get_velocity(ctx),
                 scal=np.array([rep["steps"], rep["dt"], rep["alpha"], rep["Fmax"], rep["P"], rep["sweep_launches"]]))
        lq.lq_destroy(ctx)
    finally:
        dist.destroy_process_group()


def _gather(parts, c, key):
    arrs = [p[key].reshape(5, -1, c["Ly"], c["Lx"]) for p in parts]
    return np.ascontiguousarray(np.concatenate(arrs, axis=1)).reshape(5, -1)


@pytest.mark.parametrize("name,world,integrator", [("replica4", 2, 0), ("replica3", 3, 0), ("replica5p", 2, 0),
                                                   ("replica4", 3, 1)])
def test_rank_per_process_vs_oracle_and_group_driver(name, world, integrator, oracle_mod, tmp_path):
    import torch
    import torch.multiprocessing as mp
    assert torch.cuda.is_available()
    from paper_1911_07045_b200 import binding as lq, build
    build.build()
    lq.load()
    c = CASES[name]()
    fire = dict(c["fire"], integrator=integrator)
    ctx = mp.get_context("spawn")
    port = _free_port()
    procs = [ctx.Process(target=_rank_worker, args=(r, world, port, name, integrator, str(tmp_path))) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(timeout=600)
        assert p.exitcode == 0, "rank process failed or hung (exit code %r)" % (p.exitcode,)
    parts = [np.load(os.path.join(str(tmp_path), "rank%d.npz" % r)) for r in range(world)]
    q, v = _gather(parts, c, "q"), _gather(parts, c, "v")
    # the oracle knows nothing of sub-domains or processes
    o = oracle_mod.Oracle(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"],
                          mask=c["mask"], kind=c["kind"], W=c["W"], axis=c["axis"])
    qref, rref, vref = o.fire(c["q"], STEPS, 0.0, fire, variant=1, return_v=True)
    assert np.abs(q - qref).max() <= TOL_Q, "%s x%d: Q err %.3e" % (name, world, np.abs(q - qref).max())
    assert np.abs(v - vref).max() <= 1e-7 * max(np.abs(vref).max(), 1e-3)
    for p in parts:                                   # every rank holds the same schedule
        assert p["scal"][0] == STEPS == rref["steps"]
        assert abs(p["scal"][1] - rref["dt"]) <= 1e-15 and abs(p["scal"][2] - rref["alpha"]) <= 1e-15
        assert np.array_equal(p["scal"][:5], parts[0]["scal"][:5])
    # the same-process group driver: identical kernels and reduction order -> identical bits
    ctxs = parallel.make_slabs(lq, c, world)
    rep = lq.lq_slabs_fire_minimize(ctxs, STEPS, 0.0, fire)
    assert np.array_equal(parallel.gather(lq.lq_get_Q, ctxs), q)
    assert np.array_equal(parallel.gather(lq.lq_get_velocity, ctxs), v)
    assert rep["dt"] == parts[0]["scal"][1] and rep["Fmax"] == parts[0]["scal"][3]
    if c["mask"] is not None:
        obj = c["mask"] == 1
        assert np.array_equal(q[:, obj], c["q"][:, obj]) and np.abs(v[:, obj]).max(initial=0.0) == 0.0
    for x in ctxs:
        lq.lq_destroy(x)


def test_bench_decomp_one_rank_nccl():
    """bench.py --decomp with one rank: the same driver with staging="device" -- NCCL process group, device halo
    packages, all_gather of the row, everything on the context's stream -- on the one GPU (the slab is the whole
    lattice and its halo wraps onto itself).  Checks the JSON contract of the decomposed arm."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        env.pop(k, None)
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--decomp", "--workload", "2", "--steps", "40",
                          "--warmup", "3", "--no-cpu-baseline", "--no-e2e", "--sustained-s", "0.2"],
                         capture_output=True, text=True, timeout=600, env=env, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["config"]["multi_gpu"] == "z-slabs" and line["scaling"] == "strong" and line["n_gpus"] == 1
    assert line["steps"] == 40 and line["value"] > 0 and line["gpu_launches"] >= 40
    assert line["config"]["n_simulated"] == 980000
    assert line["roofline"]["sustained"]["steps"] >= 40 and line["roofline"]["sustained"]["frac"] > 0
