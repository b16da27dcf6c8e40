"""GPU parity of md_nve_heat_run (Green-Kubo workload) against the oracle's series."""
import numpy as np
import pytest
import torch

import md_inputs as mi
import oracle
import paper_1610_03343_b200 as md
from paper_1610_03343_b200 import green_kubo
from gpu_util import DEV, GpuSystem

pytestmark = pytest.mark.gpu
PARAMS = {"tersoff": mi.TERSOFF_SI_C, "sw": mi.SW_SI}


@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_heat_current_series_matches_oracle(pot):
    s = mi.silicon_crystal(3, 0.05, 600.0, 33)
    K, rl = (16 if pot == "tersoff" else 32), mi.r_list(pot)
    g = GpuSystem(s, K)
    f = torch.zeros((3, g.n), dtype=torch.float64, device=DEV)
    Jp, Jk = md.md_nve_heat_run(g.nl, pot, PARAMS[pot], g.n, g.x, g.y, g.z, g.vx, g.vy, g.vz, f, False, g.box,
                                g.mass, 1.0, 24, 10, rl, 3)
    md.md_neighbors_status(g.nl)
    ref = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in s.items()}
    r = oracle.nve_heat_run(pot, PARAMS[pot], ref, 24, 1.0, 10, rl, K if pot == "tersoff" else 40, 3)
    Jp, Jk = np.array(Jp), np.array(Jk)
    assert Jp.shape == (8, 3)
    assert np.abs(Jp - r["J_pot"]).max() <= 1e-8 * np.abs(r["J_pot"]).max()
    assert np.abs(Jk - r["J_kin"]).max() <= 1e-8 * np.abs(r["J_kin"]).max()
    st = g.state()
    for k in ("vx", "vy", "vz"):
        assert np.abs(st[k] - ref[k]).max() <= 1e-11, k
    kap = green_kubo.running_kappa(Jp + Jk, 3.0, 600.0, float(np.prod(s["box"])), 4)
    assert kap.shape == (4,) and kap[0] == 0.0 and np.isfinite(kap).all()


def test_heat_run_is_the_nve_trajectory_with_trailing_partial_segment():
    """25 steps sampled every 10th: two samples, and a trailing segment of 5 steps without one; the state must be
    bit for bit that of md_nve_run over the same 25 steps (the sampling only reads), also across the rebuilds."""
    s = mi.silicon_crystal(4, 0.05, 300.0, 5)
    p = mi.TERSOFF_SI_C
    a, b = GpuSystem(s, 16), GpuSystem(s, 16)
    fa = torch.zeros((3, a.n), dtype=torch.float64, device=DEV)
    fb = torch.zeros((3, b.n), dtype=torch.float64, device=DEV)
    Jp, Jk = md.md_nve_heat_run(a.nl, "tersoff", p, a.n, a.x, a.y, a.z, a.vx, a.vy, a.vz, fa, False, a.box, a.mass,
                                1.0, 25, 10, 3.5, 10)
    md.md_nve_run(b.nl, "tersoff", p, b.n, b.x, b.y, b.z, b.vx, b.vy, b.vz, fb, False, None, b.box, b.mass, 1.0, 25,
                  10, 3.5)
    md.md_neighbors_status(a.nl); md.md_neighbors_status(b.nl)
    assert len(Jp) == 2 and len(Jk) == 2
    for u, v in ((a.x, b.x), (a.y, b.y), (a.z, b.z), (a.vx, b.vx), (a.vy, b.vy), (a.vz, b.vz), (fa, fb)):
        assert torch.equal(u, v)
