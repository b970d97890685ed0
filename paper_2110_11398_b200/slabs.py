"""x-slab domain decomposition of the near field over several GPUs.

The paper's parallel method (sec. 3.2): every node owns "a contiguous span of slabs" and, because
the near field reaches R cells, needs the particles of the R slabs beyond each end of its range from its x-neighbours;
sinks are owned, so nothing is reduced.  Here one process drives one GPU:

    parts = slab_partition(cpd, world, cost)                 # nf_slab_partition: contiguous ranges, balanced interaction cost
    first, nsl = parts[rank]
    local, n_own = halo_exchange(pos_owned, cpd, R, rank, world, parts, dist, LibrarySelector(plan))
    plan.set_sink_slabs(first, nsl); plan.bin(local); acc = plan.accel()[:n_own]
    cost = all_reduce(plan.slab_cost())                      # next step's partition

Everything that looks at particle data runs in the CUDA library (``nf_slab_histogram``, ``nf_slab_select``: which slab a
particle is in, the stable device-to-device compaction of what a peer needs); this module is host logic on slab INDICES
plus point-to-point transfers through ``torch.distributed`` (NCCL moves the CUDA tensors over NVLink).  The CPU tests
run the same exchange over gloo with a selector of their own.
"""
from __future__ import annotations

import torch

from . import binding as _b

__all__ = ["slab_partition", "needed_slabs", "needed_ranges", "LibrarySelector", "pack_for_peers", "halo_exchange"]


def slab_partition(cpd: int, world: int, cost=None) -> list[tuple[int, int]]:
    """Contiguous slab ranges (first, count), every rank at least one slab, minimising the largest range cost
    (``cost`` [cpd]: pair interactions per slab, ``Plan.slab_cost()`` summed over the ranks; None = equal costs)."""
    if not 1 <= world <= cpd:
        raise ValueError("need 1 <= world <= cpd")
    return _b.nf_slab_partition(cost, cpd, world)


def needed_slabs(first: int, count: int, cpd: int, R: int) -> set[int]:
    """Slabs a rank owning [first, first + count) reads as sources but does not own: R on either side, periodic."""
    own = {(first + i) % cpd for i in range(count)}
    halo = {(first - 1 - i) % cpd for i in range(R)} | {(first + count + i) % cpd for i in range(R)}
    return halo - own


def needed_ranges(need: set[int], owner: tuple[int, int], cpd: int) -> list[tuple[int, int]]:
    """The slabs of ``need`` that ``owner`` = (first, count) holds, as contiguous (first, count) runs in the owner's
    slab order (one or two runs: the lower and the upper end of its range)."""
    f, c = owner
    runs, start, length = [], None, 0
    for i in range(c):
        s = (f + i) % cpd
        if s in need:
            if start is None:
                start, length = s, 0
            length += 1
        elif start is not None:
            runs.append((start, length))
            start = None
    if start is not None:
        runs.append((start, length))
    return runs


class LibrarySelector:
    """Slab membership and compaction by the CUDA library (the cell rule of nf_bin, on the device)."""

    def __init__(self, plan):
        self.plan = plan

    def histogram(self, pos: torch.Tensor) -> list[int]:
        return self.plan.slab_histogram(pos)

    def select(self, pos: torch.Tensor, first: int, count: int, cap: int):
        return self.plan.slab_select(pos, first, count, cap, want_index=True)


def pack_for_peers(pos_owned: torch.Tensor, cpd: int, R: int, rank: int, world: int, parts, selector, payload=None):
    """What this rank sends: for every peer q the owned particles q needs as halo (``nf_slab_select`` per contiguous slab
    run, device to device, original relative order), and the payload rows that travel with them.  Returns (sends, pays)."""
    n_own = pos_owned.shape[0]
    first, cnt = parts[rank]
    hist = selector.histogram(pos_owned)                     # particles per slab, by the library's cell rule
    mine = {(first + i) % cpd for i in range(cnt)}
    if sum(hist[s] for s in mine) != n_own:
        raise ValueError("pos_owned holds particles outside this rank's slabs")
    sends, pays = [], []
    for q in range(world):
        chunks, pchunks = [], []
        if q != rank:
            need = needed_slabs(parts[q][0], parts[q][1], cpd, R)
            for f, c in needed_ranges(need, parts[rank], cpd):
                m = sum(hist[(f + i) % cpd] for i in range(c))
                if m:
                    sel, idx = selector.select(pos_owned, f, c, m)
                    chunks.append(sel)
                    if payload is not None:
                        pchunks.append(payload[idx])
        sends.append(torch.cat(chunks) if chunks else pos_owned[:0])
        if payload is not None:
            pays.append(torch.cat(pchunks) if pchunks else payload[:0])
    return sends, pays


def halo_exchange(pos_owned: torch.Tensor, cpd: int, R: int, rank: int, world: int, parts, dist, selector, payload=None):
    """One exchange step.  ``pos_owned`` [n_own][3] float32 holds the particles of this rank's slabs (any order);
    ``payload`` [n_own][k] (optional, e.g. masses) travels with the particles.
    Returns (pos_local, n_own) or (pos_local, payload_local, n_own): the owned particles first, then the halo particles
    received from the peers in rank order, each peer's in its original relative order.  ``world == 1``: nothing moves."""
    if cpd < 2 * R + 1:
        raise ValueError("cpd < 2R+1")
    n_own = pos_owned.shape[0]
    done = (lambda p, y: (p, n_own) if payload is None else (p, y, n_own))
    if world == 1 or dist is None:
        return done(pos_owned, payload)
    sends, pays = pack_for_peers(pos_owned, cpd, R, rank, world, parts, selector, payload)
    # sizes first (every rank learns what it will receive), then the particles, all point-to-point
    counts = torch.tensor([s.shape[0] for s in sends], dtype=torch.int64, device=pos_owned.device)
    table = [torch.zeros_like(counts) for _ in range(world)]
    dist.all_gather(table, counts)
    recvs = [torch.empty((int(table[q][rank]), 3), dtype=pos_owned.dtype, device=pos_owned.device) for q in range(world)]
    precv = [torch.empty((int(table[q][rank]), payload.shape[1]), dtype=payload.dtype, device=payload.device)
             for q in range(world)] if payload is not None else None
    ops = []
    for q in range(world):
        if q == rank:
            continue
        if sends[q].shape[0]:
            ops.append(dist.P2POp(dist.isend, sends[q].contiguous(), q))
            if payload is not None:
                ops.append(dist.P2POp(dist.isend, pays[q].contiguous(), q))
        if recvs[q].shape[0]:
            ops.append(dist.P2POp(dist.irecv, recvs[q], q))
            if payload is not None:
                ops.append(dist.P2POp(dist.irecv, precv[q], q))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    pos_local = torch.cat([pos_owned] + [recvs[q] for q in range(world) if q != rank], dim=0).contiguous()
    pay_local = torch.cat([payload] + [precv[q] for q in range(world) if q != rank], dim=0).contiguous() if payload is not None else None
    return done(pos_local, pay_local)
