"""Worker of tests/test_slab_cpu.py: run under torch.distributed.run with the gloo backend (CPU tensors).
Each rank owns one x-slab of the same seeded crystal, exchanges boundary atoms with the one collective of
paper_1610_03343_b200.slab and checks its local system against a brute-force selection from the global arrays."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import md_inputs as mi                                   # noqa: E402
from paper_1610_03343_b200 import slab                   # noqa: E402  (host logic only: no CUDA library is loaded)


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    s = mi.silicon_crystal(6, 0.05, 300.0, 77)
    n, box, r_list = s["n"], tuple(float(b) for b in s["box"]), 3.5
    G = {k: torch.from_numpy(s[k]) for k in ("x", "y", "z", "vx", "vy", "vz")}
    ids = torch.arange(n)
    dom = slab.SlabDomain(box, world, rank, r_list)
    for it in range(2):                                  # second round: after the atoms moved a little
        if it == 1:
            for k, v in (("x", "vx"), ("y", "vy"), ("z", "vz")):
                G[k] = torch.remainder(G[k] + 5.0 * G[v], box[0])
        own = slab.split_owned(dom, ids, G["x"], G["y"], G["z"], G["vx"])
        oid, ox, oy, oz, ovx = own
        assert int(torch.tensor([oid.numel()]).sum()) > 0
        pay = slab.boundary_payload(dom, oid, ox, oy, oz, extra=(ovx,))
        contributions = slab.all_gather_boundary(pay)
        loc = slab.assemble_local(dom, oid, ox, oy, oz, contributions, extra=(ovx,))
        # brute force from the global arrays
        xl = dom.local_x(G["x"])
        owner = dom.owner_of(G["x"])
        want_halo = (owner != rank) & ((xl < dom.halo) | ((xl >= dom.halo + dom.w) & (xl < 2 * dom.halo + dom.w)))
        got_halo_ids = loc["ids"][loc["n_own"]:]
        assert sorted(got_halo_ids.tolist()) == sorted(ids[want_halo].tolist()), (rank, it)
        assert (loc["ids"][:loc["n_own"]] == oid).all()
        # every local atom carries the global atom's data, x in the local frame, inside the local box
        gi = loc["ids"]
        assert torch.equal(loc["x"], dom.local_x(G["x"][gi])) and torch.equal(loc["y"], G["y"][gi])
        assert torch.equal(loc["extra"][0], G["vx"][gi])
        assert (loc["x"] >= 0).all() and (loc["x"] < dom.local_box[0] - 1.25 * r_list).all()
        # completeness: every atom within 2 r_list (minimum image) of an owned atom is local
        own_x = G["x"][oid]
        lo_face, hi_face = dom.lo, dom.lo + dom.w
        d_left = torch.remainder(lo_face - G["x"], box[0])
        d_right = torch.remainder(G["x"] - hi_face, box[0])
        near = (owner != rank) & ((d_left <= 2 * r_list - 1e-9) | (d_right < 2 * r_list - 1e-9))
        assert set(ids[near].tolist()) <= set(got_halo_ids.tolist())
    # ownership is a partition
    cnt = torch.tensor([oid.numel()])
    dist.all_reduce(cnt)
    assert int(cnt) == n
    dist.destroy_process_group()
    print(f"rank {rank} ok")


if __name__ == "__main__":
    main()
