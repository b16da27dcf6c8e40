"""GPU parity of md_tersoff_multi_force (multi-element Tersoff, reading A17) against the
oracle's multi-element functions, element by element."""
import math

import numpy as np
import pytest
import torch

import md_inputs as mi
import oracle
import paper_1610_03343_b200 as md
from gpu_util import (DEV, GpuSystem, assert_close_energy, assert_close_fp32, assert_close_fp64, dev)

pytestmark = pytest.mark.gpu
EL, CHI = mi.TERSOFF_SIC_ELEMENTS, mi.TERSOFF_SIC_CHI


def gpu_multi(s, types, precision=md.MD_FP64, K=32, elements=EL, chi=CHI):
    g = GpuSystem(s, K)
    g.build(3.5)
    n = g.n
    out = {k: torch.full(shape, float("nan"), dtype=torch.float64, device=DEV)
           for k, shape in (("pe", (n,)), ("f", (3, n)), ("virial", (9, n)), ("heat", (3, n)))}
    md.md_tersoff_multi_force(g.nl, n, g.x, g.y, g.z, g.vx, g.vy, g.vz, g.box, dev(types, torch.int32), elements,
                              chi, precision, pe=out["pe"], f=out["f"], virial=out["virial"], heat=out["heat"])
    md.md_neighbors_status(g.nl)
    return g, {k: v.cpu().numpy() for k, v in out.items()}


def reference(s, types, K=32):
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], 3.5, K)
    return oracle.evaluate_multi(EL, CHI, types, s["x"], s["y"], s["z"], s["box"], NN, NL,
                                 v=(s["vx"], s["vy"], s["vz"]), precision="f80"), NN, NL


@pytest.mark.parametrize("ncell,sigma,mixed", [(3, 0.05, False), (5, 0.10, False), (5, 0.08, True), (7, 0.12, True)])
def test_sic_all_outputs_fp64(ncell, sigma, mixed):
    s = mi.zincblende_crystal(ncell, mi.SIC_LATTICE_A, sigma, 900.0, 17 + ncell)
    types = s["types"].copy()
    if mixed:                                   # antisite disorder: every element pair occurs at every shell
        rng = np.random.default_rng(ncell)
        flip = rng.random(types.size) < 0.2
        types[flip] = 1 - types[flip]
    g, out = gpu_multi(s, types)
    ref, NN, NL = reference(s, types)
    gNN, gNL = g.export_list()
    assert (gNN == NN).all() and (gNL == NL).all()
    assert_close_energy(out["pe"], ref["pe"])
    assert abs(math.fsum(out["pe"]) - math.fsum(ref["pe"])) <= 1e-12 * abs(math.fsum(ref["pe"]))
    assert_close_fp64("f", out["f"], ref["f"])                 # conventional (Alg. 1) forces
    assert_close_fp64("virial", out["virial"], ref["virial"])
    assert_close_fp64("heat", out["heat"], ref["heat"])


def test_sic_fp32_mode():
    s = mi.zincblende_crystal(5, mi.SIC_LATTICE_A, 0.1, 900.0, 23)
    g, out = gpu_multi(s, s["types"], precision=md.MD_FP32)
    ref, _, _ = reference(s, s["types"])
    assert_close_fp32("f", out["f"], ref["f"])
    assert_close_fp32("virial", out["virial"], ref["virial"])
    assert_close_fp32("heat", out["heat"], ref["heat"])
    assert_close_energy(out["pe"], ref["pe"], rel=1e-4)


def test_one_element_through_the_multi_entry_is_the_single_element_potential():
    s = mi.silicon_crystal(5, 0.15, 1500.0, 2)
    g, out = gpu_multi(s, np.zeros(s["n"], np.int32), K=16, elements=[mi.TERSOFF_SI_C], chi=[[1.0]])
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], 3.5, 16)
    ref = oracle.evaluate("tersoff", mi.TERSOFF_SI_C, s["x"], s["y"], s["z"], s["box"], NN, NL,
                          v=(s["vx"], s["vy"], s["vz"]), precision="f80")
    assert_close_energy(out["pe"], ref["pe"])
    for k in ("f", "virial", "heat"):
        assert_close_fp64(k, out[k], ref[k])


def test_sic_512k_atoms_all_outputs():
    """Full size (40^3 cells = 512 000 atoms), the launch configuration bench.py times."""
    s = mi.zincblende_crystal(40, mi.SIC_LATTICE_A, 0.05, 300.0, mi.BASE_SEED + 7)
    g, out = gpu_multi(s, s["types"])
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], 3.5, 32)
    ref = oracle.evaluate_multi(EL, CHI, s["types"], s["x"], s["y"], s["z"], s["box"], NN, NL,
                                v=(s["vx"], s["vy"], s["vz"]))
    assert_close_energy(out["pe"], ref["pe"])
    for k in ("f", "virial", "heat"):
        assert_close_fp64(k, out[k], ref[k])
