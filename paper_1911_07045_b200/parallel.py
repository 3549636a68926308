"""z-slab domain decomposition: the host-side rank logic.

No arithmetic of the method lives here: which planes belong to which rank, which neighbour a halo package goes to,
in which order the per-rank reduction rows are combined, and the step loop that strings the C-ABI pieces together
(``lq_fire_begin / lq_fire_step_local / halo export + import / lq_fire_step_finish / lq_fire_step_commit /
lq_fire_end``, include/lq.h).

Three drivers over the same pieces:
  * ``lq_slabs_fire_minimize`` (binding): N slabs of one process on one GPU, everything in C -- the measured path;
  * ``fire_minimize_emulated``: the per-rank pieces driven rank by rank in ONE process through a ``LocalComm``
    (how the transport-agnostic ABI is checked on the one B200 a lease has: no kernel ever waits on another);
  * ``fire_minimize_rank``: one rank per process over ``torch.distributed``: NCCL with device buffers (one rank per
    GPU; unmeasured on hardware: a lease has one GPU) or gloo with host-staged packages (several processes sharing
    the one GPU: tests/test_ranks_gpu.py runs it against the oracle).
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
        # gloo matches by tag; NCCL ignores tags and matches the sends and receives of a pair of ranks in issue order.
        # With two ranks both neighbours are the same peer: the order below pairs my first send (low face) with its
        # first receive (its high ghost) and my second send with its second receive, which is what is wanted.
        ops = [d.P2POp(d.isend, to_lo, lo, tag=0), d.P2POp(d.isend, to_hi, hi, tag=1),
               d.P2POp(d.irecv, from_hi, hi, tag=0), d.P2POp(d.irecv, from_lo, lo, tag=1)]
        for w in d.batch_isend_irecv(ops):
            w.wait()

    def allgather(self, row, rows):
        """rows[world][6] <- every rank's row, in rank order"""
        self.dist.all_gather_into_tensor(rows.view(-1), row)


# ------------------------------------------------------------------ step loops over the C-ABI pieces

def ctx_torch_stream(ctx):
    """the context's CUDA stream as a torch stream.  The LQ_DEVICE halo / finish / commit calls only enqueue on that
    stream (include/lq.h, "Stream order"), so every torch op and every NCCL call that touches their buffers has to
    run with it as torch's current stream: NCCL orders its own stream against the current one on both sides."""
    import torch
    return torch.cuda.ExternalStream(ctx.stream) if ctx.stream else torch.cuda.default_stream()


class _HaloBuffers:
    """the four halo packages of one context (to / from the rank below and above), allocated ONCE at the size of the
    larger package (LQ_HALO_STATE) and handed out as views: nothing the enqueued copies or the transport still read
    can be recycled by torch's allocator between rounds.  host=True: pinned CPU tensors for a host-staged transport."""

    def __init__(self, lq, ctx, host):
        import torch
        self.k = {w: lq.lq_halo_bytes(ctx, w) // 8 for w in (lq.LQ_HALO_Q, lq.LQ_HALO_STATE)}
        kmax = max(self.k.values())
        kw = dict(dtype=torch.float64, device="cpu", pin_memory=True) if host else \
            dict(dtype=torch.float64, device=torch.device("cuda", torch.cuda.current_device()))
        self.bufs = [torch.empty(kmax, **kw) for _ in range(4)]

    def views(self, what):
        return [b[:self.k[what]] for b in self.bufs]          # to_lo, to_hi, from_lo, from_hi


def fire_minimize_emulated(lq, ctxs, max_steps, force_tol, params, poll=100):
    """the rank protocol, all ranks in this process, one after the other (no kernel waits on another):
    step_local on every rank, halo packages to both neighbours, all-gather of the rows, commit on every rank.
    All contexts must use one stream (as lq_slabs_fire_minimize demands): packages change hands between them."""
    import torch
    n = len(ctxs)
    if any(c.stream != ctxs[0].stream for c in ctxs):
        raise ValueError("fire_minimize_emulated: all contexts must use the same stream")
    comm = LocalComm(n)
    with torch.cuda.stream(ctx_torch_stream(ctxs[0])):
        hb = [_HaloBuffers(lq, c, host=False) for c in ctxs]

        def halo_round(what):
            sends = []
            for c, b in zip(ctxs, hb):
                to_lo, to_hi, _, _ = b.views(what)
                lq.lq_halo_export(c, what, 0, to_lo)
                lq.lq_halo_export(c, what, 1, to_hi)
                sends.append((to_lo, to_hi))
            for c, (frm_lo, frm_hi) in zip(ctxs, comm.exchange(sends)):
                lq.lq_halo_import(c, what, 0, frm_lo)
                lq.lq_halo_import(c, what, 1, frm_hi)

        halo_round(lq.LQ_HALO_Q)
        for c in ctxs:
            lq.lq_fire_begin(c, max_steps, force_tol, params)
        rows = torch.zeros((n, 6), dtype=torch.float64, device=torch.device("cuda", torch.cuda.current_device()))
        total = int(lq.lq_get_info(ctxs[0], "fire_sweeps_total"))
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
        torch.cuda.current_stream().synchronize()
    return reps[0]


def fire_minimize_rank(lq, ctx, comm: DistComm, max_steps, force_tol, params, poll=100, staging="device"):
    """one rank of the decomposed run (call on every rank).

    staging="device": NCCL moves the halo packages and the 6-double rows between device buffers.  Everything -- the
    library's enqueue-only LQ_DEVICE calls, torch's ops, NCCL -- runs with the context's stream as torch's current
    stream, so the run is stream-ordered end to end with no host synchronisation inside a step (only lq_fire_peek
    every `poll` steps when there is a force tolerance).
    staging="host": packages and rows go through pinned host buffers (the LQ_HOST calls synchronise the stream), for
    a transport without device support (gloo): how the protocol is run rank-per-process on the one GPU a lease has.
    Buffers are allocated once, before the step loop.  Returns this rank's report (Frms: lq_fire_end's note)."""
    import torch
    if staging not in ("device", "host"):
        raise ValueError("staging must be 'device' or 'host'")
    host = staging == "host"
    with torch.cuda.stream(ctx_torch_stream(ctx)):
        where = torch.device("cpu") if host else torch.device("cuda", torch.cuda.current_device())
        hb = _HaloBuffers(lq, ctx, host)
        row = torch.zeros(6, dtype=torch.float64, device=where)
        rows = torch.zeros((comm.world, 6), dtype=torch.float64, device=where)

        def halo_round(what):
            to_lo, to_hi, from_lo, from_hi = hb.views(what)
            lq.lq_halo_export(ctx, what, 0, to_lo)
            lq.lq_halo_export(ctx, what, 1, to_hi)
            comm.exchange(to_lo, to_hi, from_lo, from_hi)
            lq.lq_halo_import(ctx, what, 0, from_lo)
            lq.lq_halo_import(ctx, what, 1, from_hi)

        halo_round(lq.LQ_HALO_Q)
        lq.lq_fire_begin(ctx, max_steps, force_tol, params)
        # a second halo round per step is needed as soon as ANY rank's step has a fix-up launch: agree on it once
        row[0] = lq.lq_get_info(ctx, "has_fixup")
        comm.allgather(row, rows)
        again = bool(rows[:, 0].max().item() > 0)
        for s in range(int(lq.lq_get_info(ctx, "fire_sweeps_total"))):
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
        torch.cuda.current_stream().synchronize()
    return rep
