"""Slab decomposition of the box along x for several GPUs.

The path shards by space: U_i depends on the atoms within r_force of i, and the record P_ji that atom i gathers
depends on the neighbourhood of j, so rank r can finish every owned atom if it also holds the positions of all
atoms within 2 r_list of its slab ("halo").  Per step one exchange of boundary POSITIONS (an all-gather of the
atoms within 2 r_list of a slab face; nothing else crosses ranks), then the unchanged single-GPU calls
(md_build_neighbors / md_*_force) on the local system [owned | halo].  The local system lives in a frame whose x
axis is the slab plus its two halos plus a vacuum gap of r_list, so the library's periodic box never couples
the two halo edges (reading A15: a vacuum-padded box serves as the non-periodic case); y and z stay
periodic.  Halo atoms get incomplete forces, which are discarded.

This module holds only the host-side logic (who owns what, what is sent, where it lands); the arithmetic of the
method runs in the CUDA library.  It works on torch tensors on any device, so the exchange is covered by a
world-size-2 gloo test on CPU and the assembly by a single-GPU test that evaluates the slabs one after another.
"""
from __future__ import annotations

from dataclasses import dataclass

import torch


@dataclass
class SlabDomain:
    box: tuple          # global box (Lx, Ly, Lz)
    world: int
    rank: int
    r_list: float

    def __post_init__(self):
        self.w = self.box[0] / self.world
        self.halo = 2.0 * self.r_list
        self.lo = self.rank * self.w
        if self.world > 1 and self.w < 2.0 * self.halo:
            raise ValueError("slab narrower than 4 r_list: an atom could sit in both halos of a neighbour")
        self.local_box = (self.w + 2.0 * self.halo + 1.25 * self.r_list, self.box[1], self.box[2])

    # -- ownership -------------------------------------------------------------------------------------------
    def owner_of(self, x: torch.Tensor) -> torch.Tensor:
        return torch.clamp((x / self.w).floor().long(), 0, self.world - 1)

    def local_x(self, x: torch.Tensor) -> torch.Tensor:
        """x in the local frame: the slab starts at `halo`; the left halo is [0, halo), the right one
        [halo + w, 2 halo + w).  Periodic in the GLOBAL box, so a neighbour slab across x = 0 lands correctly."""
        return torch.remainder(x - self.lo + self.halo, self.box[0])

    # -- what this rank contributes to an exchange ---------------------------------------------------------------
    def boundary_mask(self, x_owned: torch.Tensor) -> torch.Tensor:
        """Owned atoms within `halo` of either face of the slab (they are somebody's halo)."""
        d = torch.remainder(x_owned - self.lo, self.box[0])
        return (d < self.halo) | (d >= self.w - self.halo)

    # -- what this rank keeps from an exchange -------------------------------------------------------------------
    def halo_mask(self, x_any: torch.Tensor, owner: torch.Tensor) -> torch.Tensor:
        """Of atoms owned by other ranks: those inside this rank's halos."""
        xl = self.local_x(x_any)
        return (owner != self.rank) & ((xl < self.halo) | ((xl >= self.halo + self.w) & (xl < 2.0 * self.halo + self.w)))


def all_gather_boundary(payload: torch.Tensor, group=None):
    """All-gather of per-rank boundary payloads [m_r, C] of different lengths: counts first, then the rows padded
    to the longest.  Returns the list of per-rank tensors.  The one collective of the decomposition."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    cnt = torch.tensor([payload.shape[0]], dtype=torch.int64, device=payload.device)
    cnts = [torch.zeros_like(cnt) for _ in range(world)]
    dist.all_gather(cnts, cnt, group=group)
    m = int(max(int(c) for c in cnts))
    pad = torch.zeros((m, payload.shape[1]), dtype=payload.dtype, device=payload.device)
    pad[:payload.shape[0]] = payload
    outs = [torch.zeros_like(pad) for _ in range(world)]
    dist.all_gather(outs, pad, group=group)
    return [o[:int(c)] for o, c in zip(outs, cnts)]


def boundary_payload(dom: SlabDomain, ids, x, y, z, extra=()):
    """Rows [id, x, y, z, *extra] of the owned atoms another rank may need."""
    m = dom.boundary_mask(x)
    cols = [ids[m].to(x.dtype), x[m], y[m], z[m]] + [e[m] for e in extra]
    return torch.stack(cols, dim=1)


def assemble_local(dom: SlabDomain, ids, x, y, z, contributions, extra=()):
    """Local system [owned | halo] in the local frame from this rank's owned atoms and the boundary payloads of
    all ranks (the list all_gather_boundary returns, or the same list built by hand in a single-process test).
    Returns dict(n_own, ids, x, y, z, extra=[...]) with halo atoms ordered by (source rank, payload order)."""
    hx, hy, hz, hid = [], [], [], []
    hextra = [[] for _ in extra]
    for src, pay in enumerate(contributions):
        if src == dom.rank or pay.shape[0] == 0:
            continue
        owner = torch.full((pay.shape[0],), src, dtype=torch.long, device=pay.device)
        keep = dom.halo_mask(pay[:, 1], owner)
        hid.append(pay[keep, 0].long()); hx.append(pay[keep, 1]); hy.append(pay[keep, 2]); hz.append(pay[keep, 3])
        for q in range(len(extra)):
            hextra[q].append(pay[keep, 4 + q])
    cat = lambda own, parts: torch.cat([own] + parts) if parts else own
    X = cat(x, hx)
    return {"n_own": int(x.shape[0]), "ids": cat(ids, hid), "x": dom.local_x(X), "y": cat(y, hy), "z": cat(z, hz),
            "extra": [cat(e, h) for e, h in zip(extra, hextra)]}


def split_owned(dom: SlabDomain, ids, x, *arrays):
    """The atoms of a global array set that this rank owns (used to set up a run and in tests)."""
    m = dom.owner_of(x) == dom.rank
    return [ids[m], x[m]] + [a[m] for a in arrays]
