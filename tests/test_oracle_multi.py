"""Pins of the oracle's multi-element Tersoff functions (reading A17) against things
other than themselves: published SiC / diamond values, the single-element oracle, finite differences,
Eqs. 15-16 (pairwise == conventional), momentum."""
import math

import numpy as np
import pytest

import md_inputs as mi
import oracle
from test_oracle_pins import golden, golden_min

EL, CHI = mi.TERSOFF_SIC_ELEMENTS, mi.TERSOFF_SIC_CHI


def lattice_energy_multi(a, kind):
    x, y, z, L = mi.diamond_lattice(2, a)
    n = x.size
    types = {"sic": ((np.arange(n) % 8) >= 4), "c": np.ones(n), "si": np.zeros(n)}[kind].astype(np.int32)
    box = np.array([L, L, L])
    NN, NL = oracle.neighbors(x, y, z, box, 3.05, 40, method="brute")
    o = oracle.evaluate_multi(EL, CHI, types, x, y, z, box, NN, NL, want=("pe",))
    return math.fsum(o["pe"]) / n


def test_textbook_sic_and_diamond():
    g = golden()
    a0, e0 = golden_min(lambda a: lattice_energy_multi(a, "sic"), 4.1, 4.6)
    assert abs(a0 - g["tersoff_sic_3c_a0_A"][0]) <= g["tersoff_sic_3c_a0_A"][1]
    assert abs(e0 - g["tersoff_sic_3c_ecoh_eV"][0]) <= g["tersoff_sic_3c_ecoh_eV"][1]
    a0, e0 = golden_min(lambda a: lattice_energy_multi(a, "c"), 3.3, 3.8)
    assert abs(a0 - g["tersoff_c_diamond_a0_A"][0]) <= g["tersoff_c_diamond_a0_A"][1]
    assert abs(e0 - g["tersoff_c_diamond_ecoh_eV"][0]) <= g["tersoff_c_diamond_ecoh_eV"][1]
    # the pins have teeth: chi off by 2 %, or geometric instead of arithmetic mixing of lambda, fails them
    bad_chi = [[1.0, 0.9776 * 1.02], [0.9776 * 1.02, 1.0]]
    x, y, z, L = mi.diamond_lattice(2, 4.321)
    types = ((np.arange(x.size) % 8) >= 4).astype(np.int32)
    box = np.array([L, L, L])
    NN, NL = oracle.neighbors(x, y, z, box, 3.05, 40, method="brute")
    e_bad = oracle.evaluate_multi(EL, bad_chi, types, x, y, z, box, NN, NL, want=("pe",))["pe"].mean()
    assert abs(e_bad - g["tersoff_sic_3c_ecoh_eV"][0]) > 20 * g["tersoff_sic_3c_ecoh_eV"][1]


def sic_sample(ncell=2, sigma=0.08, seed=3):
    s = mi.zincblende_crystal(ncell, mi.SIC_LATTICE_A, sigma, 600.0, seed)
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], 3.5, 40, method="brute")
    return s, NN, NL


def test_single_type_reduces_to_the_single_element_oracle():
    s = mi.silicon_crystal(2, 0.1, 300.0, 4)
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], 3.5, 16)
    v = (s["vx"], s["vy"], s["vz"])
    ref = oracle.evaluate("tersoff", mi.TERSOFF_SI_C, s["x"], s["y"], s["z"], s["box"], NN, NL, v=v)
    got = oracle.evaluate_multi(EL, CHI, np.zeros(s["n"], np.int32), s["x"], s["y"], s["z"], s["box"], NN, NL, v=v)
    for k in ("pe", "f", "f_pair", "virial", "heat"):
        assert np.abs(got[k] - ref[k]).max() <= 1e-12 * max(1.0, np.abs(ref[k]).max()), k


def test_forces_are_minus_the_gradient_and_sum_to_zero():
    s, NN, NL = sic_sample()
    assert NN.max() > 4                                         # second-shell Si-Si pairs inside the window
    o = oracle.evaluate_multi(EL, CHI, s["types"], s["x"], s["y"], s["z"], s["box"], NN, NL, want=("pe", "f", "f_pair"))
    assert np.abs(o["f"].sum(axis=1)).max() <= 1e-11
    assert np.abs(o["f"] - o["f_pair"]).max() <= 1e-12 * np.abs(o["f"]).max()     # Eqs. 15-16

    def U(x, y, z):
        return math.fsum(oracle.evaluate_multi(EL, CHI, s["types"], x, y, z, s["box"], NN, NL, want=("pe",))["pe"])
    h = 1e-5
    for i in (0, 5, 11, 30, 63):
        for a, k in enumerate("xyz"):
            p = {q: s[q].copy() for q in "xyz"}; m = {q: s[q].copy() for q in "xyz"}
            p[k][i] += h; m[k][i] -= h
            fd = -(U(p["x"], p["y"], p["z"]) - U(m["x"], m["y"], m["z"])) / (2 * h)
            assert abs(fd - o["f"][a, i]) <= 1e-6 * max(1.0, abs(o["f"][a, i])), (i, k)


def test_pair_partial_derivative_by_finite_differences():
    """P_ij = dU_i/dr_ij of an Si atom with C and Si neighbours: central differences of the plain U_i."""
    s, NN, NL = sic_sample(sigma=0.12)
    o = oracle.evaluate_multi(EL, CHI, s["types"], s["x"], s["y"], s["z"], s["box"], NN, NL, want=("P",))
    i = int(np.argmax(NN))
    rows = NL[i, :NN[i]]
    rv = np.stack([s[k][rows] - s[k][i] for k in "xyz"], axis=1)
    rv -= s["box"] * np.round(rv / s["box"])
    tj = s["types"][rows]
    h = 1e-6
    for a in range(NN[i]):
        for q in range(3):
            p, m = rv.copy(), rv.copy()
            p[a, q] += h; m[a, q] -= h
            fd = (oracle.atom_energy_multi(EL, CHI, int(s["types"][i]), tj, p) -
                  oracle.atom_energy_multi(EL, CHI, int(s["types"][i]), tj, m)) / (2 * h)
            assert abs(fd - o["P"][i, a, q]) <= 2e-8 * max(1.0, abs(o["P"][i, a, q])), (a, q)
