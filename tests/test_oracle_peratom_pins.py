"""Per-atom pins of the CPU oracle: W_i (Eq. 29) and J_i (Eq. 30) atom by atom.

The sums of W_i and J_i are pinned elsewhere (strain derivative, energy-moment identity).  Here the
values of the single atoms are fixed on clusters whose site energies have a closed form: a dimer in a
skew direction and a bent, asymmetric trimer (central atom 0, ends 1 and 2 out of each other's range).
There U_0 is an explicit function of the two bond vectors (Eqs. 1-6, resp. the
Stillinger-Weber form with V_2 split half-half and V_3 given to the central atom, A6) and
U_1, U_2 are pair terms (zeta = 0, b = 1).  The closed forms are written in 40-digit mpmath and
differentiated numerically there, so neither the oracle's dual numbers nor its hand-derived
derivatives are involved; the bent trimer makes r_10 (x) F_10 non-symmetric, so a transposed virial
or an exchanged i/j in Eq. 30 fails.  Run with -m "not gpu".
"""
import mpmath as mp
import numpy as np
import pytest

import md_inputs as mi
import oracle

mp.mp.dps = 40


def M(v):
    return mp.mpf(repr(float(v)))


def vec(a):
    return [M(c) for c in a]


def norm(a):
    return mp.sqrt(sum(c * c for c in a))


def grad(fn, a):
    """Gradient of fn(vector) at a, component by component (mpmath numerical differentiation)."""
    out = []
    for k in range(3):
        def f1(t, k=k):
            b = list(a)
            b[k] = t
            return fn(b)
        out.append(mp.diff(f1, a[k]))
    return out


# ------------------------------------------------------------------ closed-form site energies
def tersoff_forms(p):
    P = {k: M(v) for k, v in p.items()}

    def fC(r):
        if r <= P["R"]:
            return mp.mpf(1)
        if r >= P["S"]:
            return mp.mpf(0)
        return (1 + mp.cos(mp.pi * (r - P["R"]) / (P["S"] - P["R"]))) / 2

    def pair(r):                       # f_C (f_R - f_A) with b = 1
        return fC(r) * (P["A"] * mp.e ** (-P["lam"] * r) - P["B"] * mp.e ** (-P["mu"] * r))

    def g(cs):
        return 1 + P["c"] ** 2 / P["d"] ** 2 - P["c"] ** 2 / (P["d"] ** 2 + (P["h"] - cs) ** 2)

    def bond(z):
        return (1 + (P["beta"] * z) ** P["n"]) ** (-1 / (2 * P["n"]))

    def U_centre(a, b):                # U_0 of the trimer, a = r_01, b = r_02
        ra, rb = norm(a), norm(b)
        cs = sum(x * y for x, y in zip(a, b)) / (ra * rb)
        za, zb = fC(rb) * g(cs), fC(ra) * g(cs)
        ua = fC(ra) * (P["A"] * mp.e ** (-P["lam"] * ra) - bond(za) * P["B"] * mp.e ** (-P["mu"] * ra))
        ub = fC(rb) * (P["A"] * mp.e ** (-P["lam"] * rb) - bond(zb) * P["B"] * mp.e ** (-P["mu"] * rb))
        return (ua + ub) / 2

    def U_end(a):                      # U_1 (or U_2): one neighbour, zeta = 0
        return pair(norm(a)) / 2
    return U_centre, U_end


def sw_forms(p):
    P = {k: M(v) for k, v in p.items()}
    rc = P["a"] * P["sigma"]

    def V2(r):
        if r >= rc:
            return mp.mpf(0)
        s = P["sigma"] / r
        return P["epsilon"] * P["A"] * (P["B"] * s ** P["p"] - s ** P["q"]) * mp.e ** (P["sigma"] / (r - rc))

    def U_centre(a, b):
        ra, rb = norm(a), norm(b)
        cs = sum(x * y for x, y in zip(a, b)) / (ra * rb)
        v3 = mp.mpf(0)
        if ra < rc and rb < rc:
            v3 = (P["epsilon"] * P["lam"] * mp.e ** (P["gamma"] * P["sigma"] / (ra - rc) + P["gamma"] * P["sigma"] / (rb - rc))
                  * (cs - P["cos0"]) ** 2)
        return (V2(ra) + V2(rb)) / 2 + v3

    def U_end(a):
        return V2(norm(a)) / 2
    return U_centre, U_end


FORMS = {"tersoff": (tersoff_forms, mi.TERSOFF_SI_C), "sw": (sw_forms, mi.SW_SI)}


def expected_trimer(pot, r01, r02, v):
    """Per-atom U, F (Eq. 28), W (Eq. 29), J (Eq. 30) of the trimer from the closed forms."""
    make, p = FORMS[pot]
    U_centre, U_end = make(p)
    a, b = vec(r01), vec(r02)
    na, nb = [-c for c in a], [-c for c in b]
    dU0 = {1: grad(lambda t: U_centre(t, b), a), 2: grad(lambda t: U_centre(a, t), b)}   # dU_0/dr_0j
    dUj = {1: grad(U_end, na), 2: grad(U_end, nb)}                                        # dU_j/dr_j0
    rij = {(0, 1): a, (0, 2): b, (1, 0): na, (2, 0): nb}
    Pij = {(0, 1): dU0[1], (0, 2): dU0[2], (1, 0): dUj[1], (2, 0): dUj[2]}
    U = [U_centre(a, b), U_end(na), U_end(nb)]
    F = np.zeros((3, 3)); W = np.zeros((3, 3, 3)); J = np.zeros((3, 3))
    for (i, j), r in rij.items():
        Fij = [x - y for x, y in zip(Pij[(i, j)], Pij[(j, i)])]
        dot = sum(x * M(c) for x, c in zip(Pij[(j, i)], v[i]))
        for s in range(3):
            F[i, s] += float(Fij[s])
            J[i, s] += float(r[s] * dot)
            for t in range(3):
                W[i, s, t] += float(-r[s] * Fij[t] / 2)
    return np.array([float(u) for u in U]), F, W, J


def run_oracle(pot, pos, v):
    box = np.array([60.0, 55.0, 50.0])
    x, y, z = (np.ascontiguousarray(pos[:, k]) for k in range(3))
    NN, NL = oracle.neighbors(x, y, z, box, mi.r_list(pot), 16, method="brute")
    return oracle.evaluate(pot, FORMS[pot][1], x, y, z, box, NN, NL,
                           v=tuple(np.ascontiguousarray(v[:, k]) for k in range(3)))


def unit(theta, phi):
    return np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])


def rot(vv, axis, ang):
    axis = axis / np.linalg.norm(axis)
    return vv * np.cos(ang) + np.cross(axis, vv) * np.sin(ang) + axis * np.dot(axis, vv) * (1 - np.cos(ang))


V = np.array([[0.31, -0.72, 0.23], [-0.44, 0.15, 0.61], [0.08, 0.52, -0.37]])

# (potential, |r_01|, |r_02|, bond angle in degrees); the ends must be out of each other's force range.
TRIMERS = [
    ("tersoff", 2.30, 2.45, 100.0),      # both bonds below R
    ("tersoff", 2.35, 2.85, 112.0),      # second bond in the middle of the cut-off window: f_C' terms
    ("tersoff", 2.78, 2.93, 95.0),       # both in the window
    ("sw", 2.30, 2.45, 140.0),
    ("sw", 2.20, 3.10, 150.0),           # second bond near the cut-off
]


@pytest.mark.parametrize("pot,r1,r2,ang", TRIMERS)
def test_trimer_per_atom_energy_force_virial_heat_closed_form(pot, r1, r2, ang):
    u1 = unit(0.7, 1.9)
    perp = np.cross(u1, np.array([0.2, -0.5, 0.84]))
    u2 = rot(u1, perp, np.deg2rad(ang))
    r01, r02 = r1 * u1, r2 * u2
    assert np.linalg.norm(r01 - r02) > mi.r_force(pot) + 1e-3
    c0 = np.array([20.3, 21.7, 19.1])
    pos = np.stack([c0, c0 + r01, c0 + r02])
    # the oracle sees rounded coordinates: take the bond vectors it will form
    r01, r02 = pos[1] - pos[0], pos[2] - pos[0]
    U, F, W, J = expected_trimer(pot, r01, r02, V)
    o = run_oracle(pot, pos, V)
    sc_f = np.abs(F).max()
    assert np.abs(o["pe"] - U).max() <= 1e-13 * np.abs(U).max()
    assert np.abs(o["f"].T - F).max() <= 2e-13 * sc_f            # conventional Algorithm 1 forces
    assert np.abs(o["f_pair"].T - F).max() <= 2e-13 * sc_f       # Eq. 28 from the pair derivatives
    Wo = o["virial"].T.reshape(3, 3, 3)                            # [atom][a from r][b from F]
    assert np.abs(Wo - W).max() <= 2e-13 * np.abs(W).max()
    assert np.abs(o["heat"].T - J).max() <= 2e-13 * np.abs(J).max()
    # the pin can tell a transposed virial and an exchanged pair of indices in Eq. 30 apart
    # (W_0 is symmetric by the rotational invariance of U_0; an end atom's W_1 = -r_10 (x) F_10 / 2 is not)
    assert np.abs(W[1] - W[1].T).max() > 1e-4 * np.abs(W[1]).max()
    assert np.abs(J[1] - W[1] @ V[1]).max() > 1e-4 * np.abs(J[1]).max()


@pytest.mark.parametrize("pot,r", [("tersoff", 2.35), ("tersoff", 2.85), ("sw", 2.35), ("sw", 3.2)])
def test_dimer_per_atom_virial_and_heat_closed_form(pot, r):
    """Dimer in a skew direction: U_1 = U_2 = phi(r)/2, W_1 = W_2 = -(r phi'/2) d(x)d,
    J_1 = -(r phi'/2)(d.v_1) d, J_2 = -(r phi'/2)(d.v_2) d."""
    make, p = FORMS[pot]
    _, U_end = make(p)
    d = unit(1.1, 0.4)
    c0 = np.array([30.0, 31.0, 29.0])
    pos = np.stack([c0, c0 + r * d])
    bond = pos[1] - pos[0]
    rr = float(np.linalg.norm(bond)); dd = bond / rr
    dphi = float(mp.diff(lambda t: 2 * U_end([t, mp.mpf(0), mp.mpf(0)]), M(rr)))
    o = run_oracle(pot, pos, V[:2])
    Wexp = -0.5 * rr * dphi * np.outer(dd, dd)
    Wo = o["virial"].T.reshape(2, 3, 3)
    tol = 1e-12 * max(1.0, abs(rr * dphi))
    assert np.abs(Wo[0] - Wexp).max() <= tol and np.abs(Wo[1] - Wexp).max() <= tol
    for i in range(2):
        Jexp = -0.5 * rr * dphi * np.dot(dd, V[i]) * dd
        assert np.abs(o["heat"][:, i] - Jexp).max() <= tol
