"""x-slab domain decomposition of the near field over several GPUs.

The paper's parallel method (sec. 3.2): every node owns a contiguous range of x-slabs
and, because the near field reaches R cells, needs the particles of the R slabs beyond each end of its range
from its x-neighbours; sinks are owned, so nothing is reduced.  Here one process drives one GPU:

    first, nsl = slab_partition(cpd, world)[rank]
    local, n_own = halo_exchange(pos_owned, cpd, L, R, rank, world)      # one exchange step (P2P over NCCL / gloo)
    plan.set_sink_slabs(first, nsl); plan.bin(local); acc = plan.accel()[:n_own]

``halo_exchange`` is host logic plus point-to-point transfers through ``torch.distributed`` (NCCL moves the
CUDA tensors over NVLink; the CPU tests run it over gloo).  All the arithmetic of the path stays in the CUDA
library; this module only selects and ships whole particles.
"""
from __future__ import annotations

import torch

__all__ = ["slab_partition", "slab_of", "needed_slabs", "select_for_peer", "halo_exchange"]


def slab_partition(cpd: int, world: int) -> list[tuple[int, int]]:
    """Contiguous slab ranges (first, count), as equal as possible; every rank owns at least one slab."""
    if not 1 <= world <= cpd:
        raise ValueError("need 1 <= world <= cpd")
    base, extra = divmod(cpd, world)
    out, first = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((first, n))
        first += n
    return out


def slab_of(pos: torch.Tensor, cpd: int, L: float) -> torch.Tensor:
    """x index of the cell of every particle -- the float64 formula of the library (reading C6)."""
    s = torch.floor(pos[:, 0].to(torch.float64) * (float(cpd) / float(L))).to(torch.int64)
    return s.clamp_(0, cpd - 1)


def needed_slabs(first: int, count: int, cpd: int, R: int) -> set[int]:
    """Slabs a rank owning [first, first + count) reads as sources but does not own: R on either side, periodic."""
    own = {(first + i) % cpd for i in range(count)}
    halo = {(first - 1 - i) % cpd for i in range(R)} | {(first + count + i) % cpd for i in range(R)}
    return halo - own


def select_for_peer(pos_owned: torch.Tensor, slabs: torch.Tensor, peer_range: tuple[int, int], cpd: int, R: int) -> torch.Tensor:
    """The owned particles a peer needs as halo, in their original relative order (so that the peer's stable
    cell sort reproduces the order a whole-box plan would see inside every cell)."""
    need = needed_slabs(peer_range[0], peer_range[1], cpd, R)
    if not need:
        return pos_owned[:0]
    mask = torch.zeros(cpd, dtype=torch.bool, device=pos_owned.device)
    mask[torch.tensor(sorted(need), device=pos_owned.device)] = True
    return pos_owned[mask[slabs]].contiguous()


def halo_exchange(pos_owned: torch.Tensor, cpd: int, L: float, R: int, rank: int, world: int, dist=None):
    """One exchange step.  ``pos_owned`` [n_own][3] float32 holds the particles of this rank's slabs (any order);
    more columns travel with the particle (column 3 = mass for ``Plan.set_masses``: split the result into
    ``[:, :3].contiguous()`` and ``[:, 3].contiguous()``).
    Returns (pos_local, n_own): the owned particles first, then the halo particles received from the peers in
    rank order.  With ``world == 1`` (or ``dist is None``) nothing moves."""
    if cpd < 2 * R + 1:
        raise ValueError("cpd < 2R+1")
    n_own = pos_owned.shape[0]
    if world == 1 or dist is None:
        return pos_owned, n_own
    parts = slab_partition(cpd, world)
    slabs = slab_of(pos_owned, cpd, L)
    first, cnt = parts[rank]
    rel = (slabs - first) % cpd
    if n_own and int(rel.max()) >= cnt:
        raise ValueError("pos_owned holds particles outside this rank's slabs")
    sends = [select_for_peer(pos_owned, slabs, parts[q], cpd, R) if q != rank else pos_owned[:0] for q in range(world)]
    # sizes first (every rank learns what it will receive), then the particles, all point-to-point
    counts = torch.tensor([s.shape[0] for s in sends], dtype=torch.int64, device=pos_owned.device)
    table = [torch.zeros_like(counts) for _ in range(world)]
    dist.all_gather(table, counts)
    recvs = [torch.empty((int(table[q][rank]), pos_owned.shape[1]), dtype=pos_owned.dtype, device=pos_owned.device) for q in range(world)]
    ops = []
    for q in range(world):
        if q == rank:
            continue
        if sends[q].shape[0]:
            ops.append(dist.P2POp(dist.isend, sends[q], q))
        if recvs[q].shape[0]:
            ops.append(dist.P2POp(dist.irecv, recvs[q], q))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    pos_local = torch.cat([pos_owned] + [recvs[q] for q in range(world) if q != rank], dim=0).contiguous()
    return pos_local, n_own
