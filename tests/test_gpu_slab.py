"""Slab decomposition on the GPU: the four slabs of a crystal are evaluated ONE AFTER
ANOTHER on the single GPU of the test box (no rank waits on another), each as the vacuum-padded local system
[owned | halo] that paper_1610_03343_b200.slab assembles; the owned atoms' energies, forces, virials and heat
currents must equal the single-domain evaluation.  The local frame re-bases x (x - lo + halo), so r_ij picks up
one more rounding of ~1e-15 A at |x| ~ 50 A; at a bond stiffness of ~30 eV/A^2 that is ~1e-13 eV/A per pair, hence
rel 1e-9 / floor 1e-11 here instead of the oracle tests' 1e-10 / 1e-12."""
import numpy as np
import pytest
import torch

import md_inputs as mi
import paper_1610_03343_b200 as md
from paper_1610_03343_b200 import slab
from gpu_util import DEV, GpuSystem, assert_close_fp64

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_four_slabs_reproduce_the_single_domain(pot):
    params = mi.TERSOFF_SI_C if pot == "tersoff" else mi.SW_SI
    K, rl = (16 if pot == "tersoff" else 32), mi.r_list(pot)
    world = 4
    s = mi.silicon_crystal(13 if pot == "sw" else 11, 0.08, 900.0, 5)          # 70.6 / 59.7 A: slabs >= 4 r_list
    n, box = s["n"], tuple(float(b) for b in s["box"])
    g = GpuSystem(s, K)
    g.build(rl)
    ref = g.force(pot, params)
    T = {k: torch.from_numpy(s[k]) for k in ("x", "y", "z", "vx", "vy", "vz")}
    ids = torch.arange(n)
    doms = [slab.SlabDomain(box, world, r, rl) for r in range(world)]
    owned = [slab.split_owned(d, ids, T["x"], T["y"], T["z"], T["vx"], T["vy"], T["vz"]) for d in doms]
    contributions = [slab.boundary_payload(d, o[0], o[1], o[2], o[3], extra=(o[4], o[5], o[6])) for d, o in zip(doms, owned)]
    seen = 0
    for d, o in zip(doms, owned):
        loc = slab.assemble_local(d, o[0], o[1], o[2], o[3], contributions, extra=(o[4], o[5], o[6]))
        m, no = loc["x"].numel(), loc["n_own"]
        assert no < m < n
        L = {"x": loc["x"].numpy(), "y": loc["y"].numpy(), "z": loc["z"].numpy(), "vx": loc["extra"][0].numpy(),
             "vy": loc["extra"][1].numpy(), "vz": loc["extra"][2].numpy(), "box": np.array(d.local_box)}
        gl = GpuSystem(L, K)
        gl.build(rl)
        out = gl.force(pot, params)
        gid = loc["ids"][:no].numpy()
        assert np.abs(out["pe"][:no] - ref["pe"][gid]).max() <= 1e-12 * np.abs(ref["pe"]).max()
        for k in ("f", "virial", "heat"):
            assert_close_fp64(k, out[k][:, :no], ref[k][:, gid], rel=1e-9, floor=1e-11)
        seen += no
    assert seen == n
