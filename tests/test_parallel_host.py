"""Host-side rank logic of the z-slab decomposition on CPU: the partition, the slices with their
margins, and the comm layer (halo packages to both neighbours, rank-ordered all-gather of the reduction rows) over a
world-size-2 and -3 gloo group.  numpy planes stand in for the device buffers; no kernel runs here."""
import os
import socket

import numpy as np
import pytest

from paper_1911_07045_b200 import parallel


def test_split_and_neighbours():
    for Lz, n in ((72, 4), (50, 3), (100, 7), (16, 4)):
        parts = parallel.split_z(Lz, n)
        assert parts[0][0] == 0 and sum(nz for _, nz in parts) == Lz
        assert all(a[0] + a[1] == b[0] for a, b in zip(parts, parts[1:]))
        assert max(nz for _, nz in parts) - min(nz for _, nz in parts) <= 1 and min(nz for _, nz in parts) >= 4
    with pytest.raises(ValueError):
        parallel.split_z(15, 4)
    assert parallel.neighbours(0, 4) == (3, 1) and parallel.neighbours(3, 4) == (2, 0) and parallel.neighbours(0, 1) == (0, 0)


def test_slices_with_margin_wrap():
    Lx, Ly, Lz = 3, 2, 10
    a = np.arange(5 * Lz * Ly * Lx, dtype=np.float64).reshape(5, -1)
    s = parallel.slice_planes(a, (Lx, Ly, Lz), 7, 3, 3, (5,)).reshape(5, 9, Ly, Lx)
    full = a.reshape(5, Lz, Ly, Lx)
    assert np.array_equal(s[:, 3:6], full[:, 7:10])                  # own planes
    assert np.array_equal(s[:, :3], full[:, 4:7]) and np.array_equal(s[:, 6:], full[:, 0:3])   # margins wrap
    assert parallel.slice_planes(None, (Lx, Ly, Lz), 0, 4) is None


def test_combine_rows_is_rank_ordered():
    rows = np.array([[1.0, 2, 3, 0.5, 7, 0.1], [10.0, 20, 30, 0.7, 70, 0.9], [-1.0, 0, 1, 0.2, 0, 0.3]])
    t = parallel.combine_rows(rows)
    assert np.array_equal(t, [10.0, 22, 34, 0.7, 77, 0.9])


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, Lz, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        comm = parallel.DistComm(dist, rank, world)
        Lx, Ly = 4, 3
        dims = (Lx, Ly, Lz)
        glob = np.arange(5 * Lz * Ly * Lx, dtype=np.float64).reshape(5, Lz, Ly, Lx) + 0.25
        z0, nz = parallel.split_z(Lz, world)[rank]
        local = glob[:, z0:z0 + nz]
        # my boundary planes: low face z = 0, 1; high face z = nz-2, nz-1 (what lq_halo_export packs)
        to_lo = torch.from_numpy(np.ascontiguousarray(local[:, 0:2]).reshape(-1))
        to_hi = torch.from_numpy(np.ascontiguousarray(local[:, nz - 2:nz]).reshape(-1))
        from_lo, from_hi = torch.empty_like(to_lo), torch.empty_like(to_hi)
        comm.exchange(to_lo, to_hi, from_lo, from_hi)
        # ghost planes z = -2, -1 and nz, nz+1 must be the global lattice's (periodic) planes
        ext = parallel.slice_planes(glob.reshape(5, -1), dims, z0, nz, 2, (5,)).reshape(5, nz + 4, Ly, Lx)
        ok_halo = np.array_equal(from_lo.numpy().reshape(5, 2, Ly, Lx), ext[:, 0:2]) and \
            np.array_equal(from_hi.numpy().reshape(5, 2, Ly, Lx), ext[:, nz + 2:nz + 4])
        # reduction rows: all-gather in rank order, same combination on every rank
        row = torch.tensor([1.0 + rank, 2.0 * rank, 0.5, 0.1 * (rank + 1), 3.0, 0.01 * (world - rank)], dtype=torch.float64)
        rows = torch.zeros((world, 6), dtype=torch.float64)
        comm.allgather(row, rows)
        expect = np.array([[1.0 + r, 2.0 * r, 0.5, 0.1 * (r + 1), 3.0, 0.01 * (world - r)] for r in range(world)])
        ok_rows = np.array_equal(rows.numpy(), expect)
        tot = parallel.combine_rows(rows.numpy())
        out.put((rank, ok_halo, ok_rows, tot.tolist()))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,Lz", [(2, 9), (3, 14)])
def test_comm_layer_over_gloo(world, Lz):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, Lz, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(r[1] and r[2] for r in res)
    assert all(r[3] == res[0][3] for r in res)           # the same combined totals on every rank
