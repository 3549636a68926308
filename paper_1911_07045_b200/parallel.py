"""z-slab domain decomposition: the host-side rank logic.

No arithmetic of the method lives here: which planes belong to which rank, which neighbour a halo package goes to,
in which order the per-rank reduction rows are combined, and the step loop that strings the C-ABI pieces together
(``lq_fire_begin / lq_fire_step_local / halo export + import / lq_fire_step_finish / lq_fire_step_commit /
lq_fire_end``, include/lq.h).

Three drivers over the same pieces:
  * ``lq_slabs_fire_minimize`` (binding): N slabs of one process on one GPU, everything in C -- the measured path;
  * ``fire_minimize_emulated``: the per-rank pieces driven rank by rank in ONE process through a ``LocalComm``
    (how the transport-agnostic ABI is checked on the one B200 a lease has: no kernel ever waits on another);
  * ``fire_minimize_rank``: one rank per GPU over ``torch.distributed`` (NCCL device buffers; gloo for the CPU test
    of the comm layer).  Unmeasured on hardware: a lease has one GPU.
"""
from __future__ import annotations

import numpy as np


# ------------------------------------------------------------------ partition

def split_z(Lz: int, nranks: int, min_planes: int = 4):
    """[(z0, nz)] per rank: contiguous, balanced (sizes differ by at most one plane), every slab >= min_planes"""
    if nranks < 1 or Lz < nranks * min_planes:
        raise ValueError("cannot cut %d planes into %d slabs of >= %d planes" % (Lz, nranks, min_planes))
    base, extra = divmod(Lz, nranks)
    out, z = [], 0
    for r in range(nranks):
        nz = base + (1 if r < extra else 0)
        out.append((z, nz))
        z += nz
    return out


def neighbours(rank: int, nranks: int):
    """(rank below, rank above), periodic in the slab index (the lattice is index-periodic in z; walls are objects)"""
    return (rank - 1) % nranks, (rank + 1) % nranks


def slice_planes(a, dims, z0, nz, margin=0, lead=()):
    """planes z0-margin .. z0+nz+margin-1 (periodic wrap) of a dense array [*lead][Lz][Ly][Lx] given flat"""
    if a is None:
        return None
    Lx, Ly, Lz = dims
    zz = np.arange(z0 - margin, z0 + nz + margin) % Lz
    b = np.asarray(a).reshape(*lead, Lz, Ly, Lx)[..., zz, :, :]
    return np.ascontiguousarray(b).reshape(*lead, -1)


def combine_rows(rows):
    """rank-ordered combination of the per-rank rows (P, |F|^2, |v|^2, max|F|, |F0|^2, max|F0|): what the advance
    kernel computes on the device (sums left to right in rank order, maxima) -- used to check the all-gather path"""
    rows = np.asarray(rows, dtype=np.float64).reshape(-1, 6)
    tot = np.zeros(6)
    for r in rows:
        tot[0] += r[0]; tot[1] += r[1]; tot[2] += r[2]; tot[4] += r[4]
        tot[3] = max(tot[3], r[3]); tot[5] = max(tot[5], r[5])
    return tot


# ------------------------------------------------------------------ building the sub-domains

def make_slab(lq, c, z0, nz):
    """sub-domain context of workload dict ``c`` (workloads.py) for planes [z0, z0+nz): geometry with its 3-plane
    margin, local Q.  Ghost planes of Q still need a halo exchange."""
    dims = (c["Lx"], c["Ly"], c["Lz"])
    ctx = lq.lq_create_slab(c["Lx"], c["Ly"], c["Lz"], z0, nz, c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"])
    if c.get("mask") is not None:
        lq.lq_set_sites_ext(ctx, slice_planes(c["mask"], dims, z0, nz, 3), slice_planes(c.get("kind"), dims, z0, nz, 3),
                            slice_planes(c.get("W"), dims, z0, nz, 3), slice_planes(c.get("axis"), dims, z0, nz, 3, (3,)))
    lq.lq_set_Q(ctx, slice_planes(c["q"], dims, z0, nz, 0, (5,)))
    return ctx


def make_slabs(lq, c, nslabs):
    return [make_slab(lq, c, z0, nz) for z0, nz in split_z(c["Lz"], nslabs)]


def gather(fn, ctxs, ncomp=5, dtype=np.float64):
    """concatenate per-slab [ncomp][nz*Ly*Lx] arrays returned by fn(ctx) into the global [ncomp][N] array"""
    parts = [np.asarray(fn(c)).reshape(ncomp, c.Lz, c.Ly, c.Lx) for c in ctxs]
    return np.ascontiguousarray(np.concatenate(parts, axis=1)).reshape(ncomp, -1).astype(dtype, copy=False)


# ------------------------------------------------------------------ comm layers

class LocalComm:
    """all ranks live in this process: packages and rows are just handed over (emulation of the rank protocol)"""

    def __init__(self, nranks):
        self.n = nranks

    def exchange(self, sends):
        """sends[r] = (package for the rank below, package for the rank above) -> recvs[r] = (from below, from above)"""
        recvs = []
        for r in range(self.n):
            lo, hi = neighbours(r, self.n)
            recvs.append((sends[lo][1], sends[hi][0]))      # below sends me its HIGH face, above its LOW face
        return recvs

    def allgather(self, rows):
        return [np.stack(rows) if isinstance(rows[0], np.ndarray) else _stack(rows) for _ in range(self.n)]


def _stack(rows):
    import torch
    return torch.stack(list(rows))


class DistComm:
    """one rank per process over torch.distributed (NCCL with CUDA tensors; gloo with CPU tensors in the test)"""

    def __init__(self, dist, rank, world):
        self.dist, self.rank, self.world = dist, rank, world

    def exchange(self, to_lo, to_hi, from_lo, from_hi):
        """send my low-face package to the rank below and my high-face package to the rank above; receive theirs"""
        d = self.dist
        lo, hi = neighbours(self.rank, self.world)
        if self.world == 1:
            from_lo.copy_(to_hi)
            from_hi.copy_(to_lo)
            return
        ops = [d.P2POp(d.isend, to_lo, lo, tag=0), d.P2POp(d.isend, to_hi, hi, tag=1),
               d.P2POp(d.irecv, from_hi, hi, tag=0), d.P2POp(d.irecv, from_lo, lo, tag=1)]
        for w in d.batch_isend_irecv(ops):
            w.wait()

    def allgather(self, row, rows):
        """rows[world][6] <- every rank's row, in rank order"""
        self.dist.all_gather_into_tensor(rows.view(-1), row)


# ------------------------------------------------------------------ step loops over the C-ABI pieces

def _total_sweeps(max_steps, stored, euler):
    return max_steps + 1 if (stored or euler) else max(max_steps, 1)


def fire_minimize_emulated(lq, ctxs, max_steps, force_tol, params, stored=False, poll=100):
    """the rank protocol, all ranks in this process, one after the other (no kernel waits on another):
    step_local on every rank, all-gather of the rows, halo packages to both neighbours, commit on every rank"""
    import torch
    n = len(ctxs)
    comm = LocalComm(n)
    dev = torch.device("cuda")

    def halo_round(what):
        nb = [lq.lq_halo_bytes(c, what) // 8 for c in ctxs]
        sends = []
        for c, k in zip(ctxs, nb):
            lo, hi = torch.empty(k, dtype=torch.float64, device=dev), torch.empty(k, dtype=torch.float64, device=dev)
            lq.lq_halo_export(c, what, 0, lo)
            lq.lq_halo_export(c, what, 1, hi)
            sends.append((lo, hi))
        for c, (frm_lo, frm_hi) in zip(ctxs, comm.exchange(sends)):
            lq.lq_halo_import(c, what, 0, frm_lo)
            lq.lq_halo_import(c, what, 1, frm_hi)

    halo_round(lq.LQ_HALO_Q)
    for c in ctxs:
        lq.lq_fire_begin(c, max_steps, force_tol, params)
    euler = int(params.get("integrator", 0)) == 1
    rows = torch.zeros((n, 6), dtype=torch.float64, device=dev)
    total = _total_sweeps(max_steps, stored, euler)
    for s in range(total):
        for c in ctxs:
            lq.lq_fire_step_local(c)
        halo_round(lq.LQ_HALO_STATE)
        again = [lq.lq_fire_step_finish(c, rows[r]) for r, c in enumerate(ctxs)]
        for c in ctxs:
            lq.lq_fire_step_commit(c, rows)
        if any(again):
            halo_round(lq.LQ_HALO_STATE)
        if force_tol > 0.0 and (s + 1) % poll == 0 and lq.lq_fire_peek(ctxs[0])["converged"]:
            break
    reps = [lq.lq_fire_end(c) for c in ctxs]
    halo_round(lq.LQ_HALO_Q)
    return reps[0]


def fire_minimize_rank(lq, ctx, comm: DistComm, max_steps, force_tol, params, stored=False, poll=100):
    """one rank of the decomposed run (call on every rank): NCCL moves the halo packages and the 6-double rows.
    Unmeasured on hardware (one GPU per lease); the comm layer is covered by the gloo test."""
    import torch
    dev = torch.device("cuda", torch.cuda.current_device())

    def halo_round(what):
        k = lq.lq_halo_bytes(ctx, what) // 8
        to_lo, to_hi, from_lo, from_hi = (torch.empty(k, dtype=torch.float64, device=dev) for _ in range(4))
        lq.lq_halo_export(ctx, what, 0, to_lo)
        lq.lq_halo_export(ctx, what, 1, to_hi)
        torch.cuda.current_stream().synchronize()
        comm.exchange(to_lo, to_hi, from_lo, from_hi)
        lq.lq_halo_import(ctx, what, 0, from_lo)
        lq.lq_halo_import(ctx, what, 1, from_hi)

    halo_round(lq.LQ_HALO_Q)
    lq.lq_fire_begin(ctx, max_steps, force_tol, params)
    euler = int(params.get("integrator", 0)) == 1
    row = torch.zeros(6, dtype=torch.float64, device=dev)
    rows = torch.zeros((comm.world, 6), dtype=torch.float64, device=dev)
    # a second halo round per step is needed as soon as ANY rank's step has a fix-up launch: agree on it once
    row[0] = lq.lq_get_info(ctx, "has_fixup")
    comm.allgather(row, rows)
    again = bool(rows[:, 0].max().item() > 0)
    for s in range(_total_sweeps(max_steps, stored, euler)):
        lq.lq_fire_step_local(ctx)
        halo_round(lq.LQ_HALO_STATE)
        lq.lq_fire_step_finish(ctx, row)
        comm.allgather(row, rows)
        lq.lq_fire_step_commit(ctx, rows)
        if again:
            halo_round(lq.LQ_HALO_STATE)
        if force_tol > 0.0 and (s + 1) % poll == 0 and lq.lq_fire_peek(ctx)["converged"]:
            break
    rep = lq.lq_fire_end(ctx)
    halo_round(lq.LQ_HALO_Q)
    return rep
