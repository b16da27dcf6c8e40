"""Pins of the CPU oracle against things other than itself (run with -m "not gpu").

Each test names the pin of DESIGN.md / SURVEY.md section 8(c) it implements.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

import md_inputs as mi
import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "textbook.txt")


def golden():
    out = {}
    for line in open(GOLDEN):
        line = line.split("#")[0].strip()
        if line:
            k, v, tol = line.split()
            out[k] = (float(v), float(tol))
    return out


def lattice_energy(pot, params, a, ncell=2):
    x, y, z, L = mi.diamond_lattice(ncell, a)
    box = np.array([L, L, L])
    rl = (params["S"] if pot == "tersoff" else params["a"] * params["sigma"]) + 0.05
    NN, NL = oracle.neighbors(x, y, z, box, rl, 40, method="brute")
    o = oracle.evaluate(pot, params, x, y, z, box, NN, NL, want=("pe",))
    return math.fsum(o["pe"]) / x.size


def golden_min(f, lo, hi, it=60):
    g = (math.sqrt(5) - 1) / 2
    c, d = hi - g * (hi - lo), lo + g * (hi - lo)
    fc, fd = f(c), f(d)
    for _ in range(it):
        if fc < fd:
            hi, d, fd = d, c, fc
            c = hi - g * (hi - lo); fc = f(c)
        else:
            lo, c, fc = c, d, fd
            d = lo + g * (hi - lo); fd = f(d)
    xm = 0.5 * (lo + hi)
    return xm, f(xm)


def displaced(pot, ncell=2, sigma=0.05, seed=7, T=300.0):
    s = mi.silicon_crystal(ncell, sigma, T, seed)
    K = 16 if pot == "tersoff" else 40
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list(pot), K, method="brute")
    return s, NN, NL


PARAMS = {"tersoff": mi.TERSOFF_SI_C, "sw": mi.SW_SI}


# ---------------------------------------------------------------- P1 / P2 textbook
def test_tersoff_textbook_cohesive_energy_and_lattice_constant():
    g = golden()
    a0, e0 = golden_min(lambda a: lattice_energy("tersoff", mi.TERSOFF_SI_C, a), 5.3, 5.6)
    assert abs(a0 - g["tersoff_sic_a0_A"][0]) <= g["tersoff_sic_a0_A"][1]
    assert abs(e0 - g["tersoff_sic_ecoh_eV"][0]) <= g["tersoff_sic_ecoh_eV"][1]


def test_sw_textbook_minimum():
    g = golden()
    p = mi.SW_SI
    a0, e0 = golden_min(lambda a: lattice_energy("sw", p, a), 5.3, 5.6)
    r0 = a0 * math.sqrt(3) / 4
    assert abs(r0 / p["sigma"] - g["sw_r0_over_sigma"][0]) <= g["sw_r0_over_sigma"][1]
    assert abs(e0 / p["epsilon"] - g["sw_ecoh_over_epsilon"][0]) <= g["sw_ecoh_over_epsilon"][1]


def test_tersoff_perfect_lattice_closed_form():
    """P1: on the perfect lattice the sums collapse analytically: 4 neighbours at r0 = a sqrt(3)/4,
    all angles cos = -1/3, zeta = 3 g(-1/3); evaluated with 40-digit mpmath."""
    mp.mp.dps = 40
    p = {k: mp.mpf(repr(v)) for k, v in mi.TERSOFF_SI_C.items()}
    a = mp.mpf("5.43")
    r0 = a * mp.sqrt(3) / 4
    x = p["h"] + mp.mpf(1) / 3
    g = 1 + p["c"] ** 2 / p["d"] ** 2 - p["c"] ** 2 / (p["d"] ** 2 + x ** 2)
    zeta = 3 * g
    b = (1 + (p["beta"] * zeta) ** p["n"]) ** (-1 / (2 * p["n"]))
    Ui = 2 * (p["A"] * mp.e ** (-p["lam"] * r0) - b * p["B"] * mp.e ** (-p["mu"] * r0))
    e = lattice_energy("tersoff", mi.TERSOFF_SI_C, 5.43)
    assert abs(e - float(Ui)) <= 1e-13 * abs(float(Ui))
    assert abs(float(Ui) - (-4.6295875)) < 1e-6


# ---------------------------------------------------------------- P5 dimer closed form
@pytest.mark.parametrize("r", [2.0, 2.35, 2.7, 2.85, 2.95, 3.2])
def test_tersoff_dimer_closed_form(r):
    """zeta = 0 => b = 1: U = fC(r)(A e^{-lam r} - B e^{-mu r}); F = -dU/dr along the bond.
    r = 2.85 is the middle of the R..S window where fC = 1/2 exactly."""
    mp.mp.dps = 40
    p = {k: mp.mpf(repr(v)) for k, v in mi.TERSOFF_SI_C.items()}

    def U(rr):
        if rr <= p["R"]:
            fc = mp.mpf(1)
        elif rr >= p["S"]:
            fc = mp.mpf(0)
        else:
            fc = (1 + mp.cos(mp.pi * (rr - p["R"]) / (p["S"] - p["R"]))) / 2
        return fc * (p["A"] * mp.e ** (-p["lam"] * rr) - p["B"] * mp.e ** (-p["mu"] * rr))
    rr = mp.mpf(repr(r))
    u = float(U(rr))
    du = float(mp.diff(U, rr)) if r not in (2.7,) else None
    box = np.array([40.0, 40.0, 40.0])
    x = np.array([10.0, 10.0 + r]); y = np.array([10.0, 10.0]); z = np.array([10.0, 10.0])
    NN, NL = oracle.neighbors(x, y, z, box, 3.5, 16)
    o = oracle.evaluate("tersoff", mi.TERSOFF_SI_C, x, y, z, box, NN, NL)
    if r == 2.85:
        assert abs(u - 0.5 * float(p["A"] * mp.e ** (-p["lam"] * rr) - p["B"] * mp.e ** (-p["mu"] * rr))) < 1e-15
    assert abs(o["pe"].sum() - u) <= 1e-13 * max(1.0, abs(u))
    assert abs(o["pe"][0] - o["pe"][1]) < 1e-15
    if du is not None:
        # force on atom 0 (at smaller x) is +dU/dr along +x
        assert abs(o["f"][0, 0] - du) <= 1e-12 * max(1.0, abs(du))
        assert abs(o["f"][0, 1] + du) <= 1e-12 * max(1.0, abs(du))
        assert np.abs(o["f"][1:]).max() == 0.0


# ---------------------------------------------------------------- P3 / P4 / P14 perfect lattice
@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_perfect_lattice_zero_force_and_virial(pot):
    p = PARAMS[pot]
    a = 5.43
    x, y, z, L = mi.diamond_lattice(3, a)
    box = np.array([L, L, L])
    NN, NL = oracle.neighbors(x, y, z, box, mi.r_list(pot), 40, method="brute")
    assert (NN == (4 if pot == "tersoff" else 16)).all()
    assert golden()["si_crystal_neighbours"][0] == 4
    o = oracle.evaluate(pot, p, x, y, z, box, NN, NL)
    assert np.abs(o["f"]).max() <= 1e-12          # P3
    assert np.abs(o["f_pair"]).max() <= 1e-12
    # P4: hydrostatic virial per atom = -(a/3) dE/da, off-diagonals 0; dE/da by central difference
    h = 1e-4
    dEda = (lattice_energy(pot, p, a + h, 3) - lattice_energy(pot, p, a - h, 3)) / (2 * h)
    W = o["virial"].sum(axis=1) / x.size
    for q in (0, 4, 8):
        assert abs(W[q] - (-(a / 3) * dEda)) <= 1e-7
    for q in (1, 2, 3, 5, 6, 7):
        assert abs(W[q]) <= 1e-13


# ---------------------------------------------------------------- P6, P7, P9 forces
@pytest.mark.parametrize("pot,sigma", [("tersoff", 0.05), ("tersoff", 0.15), ("tersoff", 0.25),
                                       ("sw", 0.05), ("sw", 0.15)])
def test_forces_finite_difference_momentum_and_pairwise_equivalence(pot, sigma):
    p = PARAMS[pot]
    s, NN, NL = displaced(pot, 2, sigma, seed=11)
    n = s["n"]
    o = oracle.evaluate(pot, p, s["x"], s["y"], s["z"], s["box"], NN, NL, precision="f80")
    fmax = np.abs(o["f"]).max()
    assert np.abs(o["f"].sum(axis=1)).max() <= 1e-12 * math.sqrt(n) * max(1.0, fmax)   # P6
    assert np.abs(o["f"] - o["f_pair"]).max() <= 1e-12 * fmax                          # P9, Eqs. 15-16
    # P7: central differences of the total energy, h = 1e-5 A (list has a 0.5 A skin: no rebuild needed)
    h = 1e-5
    rng = np.random.default_rng(3)
    for i in rng.choice(n, 6, replace=False):
        for a, key in enumerate("xyz"):
            e = []
            for sgn in (+1, -1):
                c = {k: s[k].copy() for k in "xyz"}
                c[key][i] += sgn * h
                oo = oracle.evaluate(pot, p, c["x"], c["y"], c["z"], s["box"], NN, NL,
                                     precision="f80", want=("pe",))
                e.append(math.fsum(oo["pe"]))
            fd = -(e[0] - e[1]) / (2 * h)
            assert abs(fd - o["f"][a, i]) <= 1e-6 * max(abs(o["f"][a, i]), 1e-2 * fmax), (i, a, fd, o["f"][a, i])


# ---------------------------------------------------------------- P8 dU_i/dr_ij
@pytest.mark.parametrize("pot,sigma", [("tersoff", 0.15), ("sw", 0.15)])
def test_partial_derivative_finite_difference(pot, sigma):
    p = PARAMS[pot]
    s, NN, NL = displaced(pot, 2, sigma, seed=5)
    o = oracle.evaluate(pot, p, s["x"], s["y"], s["z"], s["box"], NN, NL, precision="f80",
                        want=("pe", "P"))
    rf = mi.r_force(pot)
    L = s["box"][0]
    h = 1e-5
    for i in (0, 17, 42):
        rv, slots = [], []
        for m in range(NN[i]):
            j = NL[i, m]
            d = np.array([s[k][j] - s[k][i] for k in "xyz"])
            d -= L * np.round(d / L)
            if np.linalg.norm(d) < rf:
                rv.append(d); slots.append(m)
        rv = np.array(rv)
        assert abs(oracle.atom_energy(pot, p, rv) - o["pe"][i]) <= 1e-13 * abs(o["pe"][i])
        scale = np.abs(o["P"][i]).max()
        for a, m in enumerate(slots):
            for q in range(3):
                rp = rv.copy(); rp[a, q] += h
                rm = rv.copy(); rm[a, q] -= h
                fd = (oracle.atom_energy(pot, p, rp) - oracle.atom_energy(pot, p, rm)) / (2 * h)
                assert abs(fd - o["P"][i, m, q]) <= 2e-8 * scale, (i, m, q, fd, o["P"][i, m, q])


# ---------------------------------------------------------------- P10 virial = -dU/d(strain)
@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_total_virial_is_strain_derivative(pot):
    p = PARAMS[pot]
    # vacuum-padded cluster: no pair crosses the boundary, all 9 strain components can be applied
    s = mi.silicon_crystal(2, 0.1, 300.0, 21)
    big = 60.0
    box = np.array([big, big, big])
    r = np.stack([s["x"], s["y"], s["z"]]) + 20.0
    K = 16 if pot == "tersoff" else 40
    NN, NL = oracle.neighbors(r[0], r[1], r[2], box, mi.r_list(pot), K)
    o = oracle.evaluate(pot, p, r[0], r[1], r[2], box, NN, NL, precision="f80")
    W = o["virial"].sum(axis=1).reshape(3, 3)
    assert np.abs(W - W.T).max() <= 1e-12 * np.abs(W).max()
    # W = sum_i r_i (x) F_i (Eq. 17) holds literally in the cluster
    W17 = np.einsum("ai,bi->ab", r, o["f"])
    assert np.abs(W - W17).max() <= 1e-11 * np.abs(W).max()
    eps = 1e-6
    for a in range(3):
        for b in range(3):
            e = []
            for sgn in (+1, -1):
                rr = r.copy()
                rr[a] += sgn * eps * r[b]                       # r^a += eps_ab r^b
                oo = oracle.evaluate(pot, p, rr[0], rr[1], rr[2], box, NN, NL, precision="f80", want=("pe",))
                e.append(math.fsum(oo["pe"]))
            dU = (e[0] - e[1]) / (2 * eps)
            assert abs(W[b, a] + dU) <= 2e-7 * np.abs(W).max(), (a, b, W[b, a], -dU)
    # periodic box, diagonal components: strain the box with the positions
    s, NN, NL = displaced(pot, 2, 0.05, seed=9)
    o = oracle.evaluate(pot, p, s["x"], s["y"], s["z"], s["box"], NN, NL, precision="f80")
    W = o["virial"].sum(axis=1)
    for a, key in enumerate("xyz"):
        e = []
        for sgn in (+1, -1):
            c = {k: s[k].copy() for k in "xyz"}
            bx = s["box"].copy()
            c[key] *= (1 + sgn * eps); bx[a] *= (1 + sgn * eps)
            oo = oracle.evaluate(pot, p, c["x"], c["y"], c["z"], bx, NN, NL, precision="f80", want=("pe",))
            e.append(math.fsum(oo["pe"]))
        dU = (e[0] - e[1]) / (2 * eps)
        assert abs(W[4 * a] + dU) <= 2e-7 * max(1.0, np.abs(W).max())


# ---------------------------------------------------------------- P17 elastic constants (three-body magnitude)
EV_PER_A3_IN_GPA = 160.21766208


def strained_lattice_energy(pot, params, a, strain, ncell=2):
    """Total energy and reference volume of the perfect lattice under a homogeneous diagonal strain
    (box and positions scaled together; no internal relaxation, which C11 and C12 do not need)."""
    x, y, z, L = mi.diamond_lattice(ncell, a)
    s = np.asarray(strain, dtype=float)
    box = np.array([L, L, L]) * (1.0 + s)
    rl = (params["S"] if pot == "tersoff" else params["a"] * params["sigma"]) + 0.05
    NN, NL = oracle.neighbors(x * (1 + s[0]), y * (1 + s[1]), z * (1 + s[2]), box, rl, 40, method="brute")
    o = oracle.evaluate(pot, params, x * (1 + s[0]), y * (1 + s[1]), z * (1 + s[2]), box, NN, NL, want=("pe",))
    return math.fsum(o["pe"]), L ** 3


def cubic_elastic_constants(pot, params, a, h=1e-3):
    """C11, C12, B in GPa by central second differences of the energy:
    E/V = 1/2 C11 sum e_aa^2 + C12 sum_{a<b} e_aa e_bb, so d2E/de_xx^2 = V C11 and, with
    e_xx = e_yy = e, d2E/de^2 = 2 V (C11 + C12)."""
    e0, V = strained_lattice_energy(pot, params, a, (0, 0, 0))
    d2 = lambda s: (strained_lattice_energy(pot, params, a, s)[0] - 2 * e0 +
                    strained_lattice_energy(pot, params, a, tuple(-c for c in s))[0]) / h ** 2 / V * EV_PER_A3_IN_GPA
    c11 = d2((h, 0, 0))
    c12 = 0.5 * d2((h, h, 0)) - c11
    return c11, c12, (c11 + 2 * c12) / 3


def test_sw_elastic_constants_pin_three_body_magnitude():
    """every other SW pin is blind to the size of V3 (it vanishes on the diamond lattice at any
    lattice constant; finite-difference pins pass for any lambda, gamma).  C11 - C12 is carried by V3 alone."""
    g = golden()
    p = mi.SW_SI
    a0 = 4 * 2 ** (1 / 6) * p["sigma"] / math.sqrt(3)            # zero-pressure lattice constant (P2)
    c11, c12, bulk = cubic_elastic_constants("sw", p, a0)
    for got, key in ((c11, "sw_c11_GPa"), (c12, "sw_c12_GPa"), (bulk, "sw_bulk_GPa")):
        assert abs(got - g[key][0]) <= g[key][1], (key, got)
    # the pin has teeth: 5 % in lambda or in gamma fails it
    for k in ("lam", "gamma"):
        q = dict(p); q[k] = 0.95 * p[k]
        bad11, bad12, _ = cubic_elastic_constants("sw", q, a0)
        assert abs(bad11 - g["sw_c11_GPa"][0]) > 5 * g["sw_c11_GPa"][1], k
        assert abs(bad12 - g["sw_c12_GPa"][0]) > 3 * g["sw_c12_GPa"][1], k


def test_tersoff_elastic_constants_pin_angular_term():
    """The same pin for g(theta) and b(zeta): Tersoff (1988) fitted Si(C) to improve exactly these."""
    g = golden()
    t = mi.TERSOFF_SI_C
    c11, c12, bulk = cubic_elastic_constants("tersoff", t, g["tersoff_sic_a0_A"][0])
    for got, key in ((c11, "tersoff_sic_c11_GPa"), (c12, "tersoff_sic_c12_GPa"), (bulk, "tersoff_sic_bulk_GPa")):
        assert abs(got - g[key][0]) <= g[key][1], (key, got)
    for k, fac in (("h", 1.05), ("d", 1.05), ("c", 1.05)):
        q = dict(t); q[k] = fac * t[k]
        bad11, bad12, _ = cubic_elastic_constants("tersoff", q, g["tersoff_sic_a0_A"][0])
        assert max(abs(bad11 - g["tersoff_sic_c11_GPa"][0]), abs(bad12 - g["tersoff_sic_c12_GPa"][0])) > \
            3 * g["tersoff_sic_c11_GPa"][1], k
