"""GPU parity of the paper's literal Algorithm 3 + Algorithm 2 (md_tersoff_force_literal) against
the oracle, and agreement with the stored-P design."""
import math

import numpy as np
import pytest
import torch

import md_inputs as mi
import oracle
import paper_1610_03343_b200 as md
from gpu_util import DEV, GpuSystem, assert_close_energy, assert_close_fp32, assert_close_fp64

pytestmark = pytest.mark.gpu


def literal(g, precision=md.MD_FP64):
    n = g.n
    out = {k: torch.full(shape, float("nan"), dtype=torch.float64, device=DEV)
           for k, shape in (("pe", (n,)), ("f", (3, n)), ("virial", (9, n)), ("heat", (3, n)))}
    md.md_tersoff_force_literal(g.nl, n, g.x, g.y, g.z, g.vx, g.vy, g.vz, g.box, mi.TERSOFF_SI_C, precision,
                                pe=out["pe"], f=out["f"], virial=out["virial"], heat=out["heat"])
    md.md_neighbors_status(g.nl)
    return {k: v.cpu().numpy() for k, v in out.items()}


@pytest.mark.parametrize("ncell,sigma,T,seed", [(2, 0.05, 300.0, 1), (5, 0.15, 1500.0, 2), (7, 0.25, 1500.0, 3)])
def test_literal_all_outputs_fp64(ncell, sigma, T, seed):
    s = mi.silicon_crystal(ncell, sigma, T, seed)
    g = GpuSystem(s, 16)
    g.build(3.5)
    out = literal(g)
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], 3.5, 16)
    ref = oracle.evaluate("tersoff", mi.TERSOFF_SI_C, s["x"], s["y"], s["z"], s["box"], NN, NL,
                          v=(s["vx"], s["vy"], s["vz"]), precision="f80")
    assert_close_energy(out["pe"], ref["pe"])
    assert abs(math.fsum(out["pe"]) - math.fsum(ref["pe"])) <= 1e-12 * abs(math.fsum(ref["pe"]))
    for k in ("f", "virial", "heat"):
        assert_close_fp64(k, out[k], ref[k])
    stored = g.force("tersoff", mi.TERSOFF_SI_C)               # the two designs agree far inside the tolerance
    assert np.abs(stored["f"] - out["f"]).max() <= 1e-11 * max(1.0, np.abs(out["f"]).max())


def test_literal_fp32_and_dimer():
    s = mi.silicon_crystal(5, 0.15, 1500.0, 2)
    g = GpuSystem(s, 16)
    g.build(3.5)
    out = literal(g, md.MD_FP32)
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], 3.5, 16)
    ref = oracle.evaluate("tersoff", mi.TERSOFF_SI_C, s["x"], s["y"], s["z"], s["box"], NN, NL,
                          v=(s["vx"], s["vy"], s["vz"]))
    for k in ("f", "virial", "heat"):
        assert_close_fp32(k, out[k], ref[k])
    box = np.array([40.0, 40.0, 40.0])                         # zeta = 0 path and an isolated atom
    d = {"x": np.array([10.0, 12.85, 30.0]), "y": np.array([10.0, 10.0, 30.0]), "z": np.array([10.0, 10.0, 30.0]),
         "box": box}
    g = GpuSystem(d, 16)
    g.build(3.5)
    out = literal(g)
    NN, NL = oracle.neighbors(d["x"], d["y"], d["z"], box, 3.5, 16)
    ref = oracle.evaluate("tersoff", mi.TERSOFF_SI_C, d["x"], d["y"], d["z"], box, NN, NL, v=(np.zeros(3),) * 3,
                          precision="f80")
    assert_close_fp64("f", out["f"], ref["f"])
    assert (out["f"][:, 2] == 0).all() and out["pe"][2] == 0


def test_literal_512k_atoms():
    c = mi.make_config(1)
    g = GpuSystem(c, 16)
    g.build(c["r_list"])
    out = literal(g)
    NN, NL = g.export_list()
    ref = oracle.evaluate("tersoff", c["params"], c["x"], c["y"], c["z"], c["box"], NN, NL,
                          v=(c["vx"], c["vy"], c["vz"]))
    assert_close_energy(out["pe"], ref["pe"])
    for k in ("f", "virial", "heat"):
        assert_close_fp64(k, out[k], ref[k])
