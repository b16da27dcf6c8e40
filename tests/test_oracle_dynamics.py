"""Heat-current, NVE and neighbour-list pins of the CPU oracle (-m "not gpu")."""
import math

import numpy as np
import pytest

import md_inputs as mi
import oracle

PARAMS = {"tersoff": mi.TERSOFF_SI_C, "sw": mi.SW_SI}


def cluster(pot, seed=31, sigma=0.1, T=1000.0):
    """Vacuum-padded 64-atom cluster: r_ij = r_j - r_i exactly (no image shifts)."""
    s = mi.silicon_crystal(2, sigma, T, seed)
    box = np.array([60.0, 60.0, 60.0])
    st = {"x": s["x"] + 20.0, "y": s["y"] + 20.0, "z": s["z"] + 20.0,
          "vx": s["vx"].copy(), "vy": s["vy"].copy(), "vz": s["vz"].copy(),
          "box": box, "mass": s["mass"], "n": s["n"]}
    return st


def evaluate_state(pot, st, K, want=("pe", "f", "virial", "heat")):
    NN, NL = oracle.neighbors(st["x"], st["y"], st["z"], st["box"], mi.r_list(pot), K)
    return oracle.evaluate(pot, PARAMS[pot], st["x"], st["y"], st["z"], st["box"], NN, NL,
                           v=(st["vx"], st["vy"], st["vz"]), want=want)


# ---------------------------------------------------------------- P11
@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_heat_current_uniform_velocity_and_linearity(pot):
    """All v_i = v0  =>  sum_i J_i = (sum_i W_i) . v0 (from Eqs. 29, 30); J is linear in v."""
    K = 16 if pot == "tersoff" else 40
    s = mi.silicon_crystal(2, 0.1, 300.0, 13)
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list(pot), K)
    n = s["n"]
    v0 = np.array([0.3, -0.7, 0.2])
    v = tuple(np.full(n, c) for c in v0)
    o = oracle.evaluate(pot, PARAMS[pot], s["x"], s["y"], s["z"], s["box"], NN, NL, v=v)
    W = o["virial"].sum(axis=1).reshape(3, 3)
    J = o["heat"].sum(axis=1)
    assert np.abs(J - W @ v0).max() <= 1e-12 * np.abs(W).max()
    va = (s["vx"], s["vy"], s["vz"])
    vb = tuple(np.roll(c, 5) for c in va)
    Ja = oracle.evaluate(pot, PARAMS[pot], s["x"], s["y"], s["z"], s["box"], NN, NL, v=va, want=("heat",))["heat"]
    Jb = oracle.evaluate(pot, PARAMS[pot], s["x"], s["y"], s["z"], s["box"], NN, NL, v=vb, want=("heat",))["heat"]
    vc = tuple(2.0 * a - 3.0 * b for a, b in zip(va, vb))
    Jc = oracle.evaluate(pot, PARAMS[pot], s["x"], s["y"], s["z"], s["box"], NN, NL, v=vc, want=("heat",))["heat"]
    assert np.abs(Jc - (2.0 * Ja - 3.0 * Jb)).max() <= 1e-12 * max(np.abs(Ja).max(), np.abs(Jb).max())


# ---------------------------------------------------------------- P12
@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_heat_current_energy_moment(pot):
    """d/dt sum_i r_i E_i = sum_i v_i E_i + sum_i J_i with E_i = m v_i^2/2 + U_i (definition of the
    heat current; J_i of Eq. (27) is its potential part).  Central difference over +-h of a
    velocity-Verlet step: the mismatch must be small and shrink as h^2.  Pins the total J and the
    per-atom partition U_i."""
    K = 16 if pot == "tersoff" else 40
    base = cluster(pot)
    m = base["mass"]

    def moment(st):
        o = evaluate_state(pot, st, K, want=("pe",))
        ke = 0.5 * m * (st["vx"] ** 2 + st["vy"] ** 2 + st["vz"] ** 2) / mi.KAPPA
        E = ke + o["pe"]
        return np.array([math.fsum(st[k] * E) for k in "xyz"]), E

    o0 = evaluate_state(pot, base, K)
    _, E0 = moment(base)
    rhs = np.array([math.fsum(base["v" + k] * E0) for k in "xyz"]) + o0["heat"].sum(axis=1)
    scale = np.abs(o0["heat"].sum(axis=1)).max()
    errs = []
    for h in (0.04, 0.02):
        R = []
        for sgn in (+1, -1):
            st = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in base.items()}
            oracle.nve_run(pot, PARAMS[pot], st, 1, sgn * h, 1, mi.r_list(pot), K)
            R.append(moment(st)[0])
        lhs = (R[0] - R[1]) / (2 * h)
        errs.append(np.abs(lhs - rhs).max() / scale)
    assert errs[1] <= 2e-4, errs
    assert 3.0 <= errs[0] / errs[1] <= 5.0, errs


# ---------------------------------------------------------------- P13
@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_nve_energy_conservation_second_order(pot):
    K = 16 if pot == "tersoff" else 40
    dev = []
    for dt, nsteps in ((1.0, 100), (0.5, 200)):
        s = mi.silicon_crystal(2, 0.05, 300.0, 17)
        n = s["n"]
        o = evaluate_state(pot, s, K, want=("pe",))
        ke0 = 0.5 * s["mass"] * math.fsum(s["vx"] ** 2 + s["vy"] ** 2 + s["vz"] ** 2) / mi.KAPPA
        e0 = ke0 + math.fsum(o["pe"])
        emax = 0.0
        f = None
        for _ in range(nsteps // 10):
            r = oracle.nve_run(pot, PARAMS[pot], s, 10, dt, 10, mi.r_list(pot), K, f=f)
            f = r["f"]
            ke = 0.5 * s["mass"] * math.fsum(s["vx"] ** 2 + s["vy"] ** 2 + s["vz"] ** 2) / mi.KAPPA
            emax = max(emax, abs(ke + math.fsum(r["pe"]) - e0) / n)
        dev.append(emax)
    assert dev[0] <= 1e-4, dev
    assert 3.0 <= dev[0] / dev[1] <= 5.0, dev


# ---------------------------------------------------------------- P14
@pytest.mark.parametrize("pot,ncell,sigma", [("tersoff", 5, 0.05), ("tersoff", 5, 0.15), ("sw", 6, 0.15)])
def test_cell_list_equals_brute_force_and_is_symmetric(pot, ncell, sigma):
    s = mi.silicon_crystal(ncell, sigma, 300.0, 23)
    K = 16 if pot == "tersoff" else 40
    a = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list(pot), K, method="brute")
    b = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list(pot), K, method="cell")
    assert (a[0] == b[0]).all() and (a[1] == b[1]).all()
    NN, NL = a
    for i in range(0, s["n"], 7):
        row = NL[i, :NN[i]]
        assert (np.diff(row) > 0).all()
        for j in row:
            assert i in NL[j, :NN[j]]
    # independent numpy check of a few rows with the plain definition |r_ij|_min-image < r_list
    L = s["box"][0]
    P = np.stack([s["x"], s["y"], s["z"]], axis=1)
    for i in (0, 101, s["n"] - 1):
        d = P - P[i]
        d -= L * np.round(d / L)
        idx = np.nonzero((d ** 2).sum(axis=1) < mi.r_list(pot) ** 2)[0]
        idx = idx[idx != i]
        assert list(idx) == list(NL[i, :NN[i]])


def test_brute_force_non_cubic_box_wraps_every_axis():
    rng = np.random.default_rng(0)
    box = np.array([9.0, 11.0, 14.0])
    n = 300
    P = rng.random((n, 3)) * box
    NN, NL = oracle.neighbors(P[:, 0].copy(), P[:, 1].copy(), P[:, 2].copy(), box, 3.0, 64, method="brute")
    NN2, NL2 = oracle.neighbors(P[:, 0].copy(), P[:, 1].copy(), P[:, 2].copy(), box, 3.0, 64, method="cell")
    assert (NN == NN2).all() and (NL == NL2).all()
    for i in range(0, n, 11):
        d = P - P[i]
        d -= box * np.round(d / box)
        idx = np.nonzero((d ** 2).sum(axis=1) < 9.0)[0]
        idx = idx[idx != i]
        assert list(idx) == list(NL[i, :NN[i]])


@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_double_and_long_double_oracle_agree(pot):
    K = 16 if pot == "tersoff" else 40
    s = mi.silicon_crystal(2, 0.15, 300.0, 3)
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list(pot), K)
    v = (s["vx"], s["vy"], s["vz"])
    a = oracle.evaluate(pot, PARAMS[pot], s["x"], s["y"], s["z"], s["box"], NN, NL, v=v, precision="f64")
    b = oracle.evaluate(pot, PARAMS[pot], s["x"], s["y"], s["z"], s["box"], NN, NL, v=v, precision="f80")
    for k in ("pe", "f", "virial", "heat"):
        assert np.abs(a[k] - b[k]).max() <= 1e-11 * np.abs(b[k]).max(), k


def test_generator_is_counter_based_and_has_the_stated_statistics():
    a = mi.normal_deviates(5, 1, 30000)
    b = mi.normal_deviates(5, 1, 60000)
    assert (a == b[:30000]).all()
    assert (mi.normal_deviates(6, 1, 100) != a[:100]).any()
    assert abs(b.mean()) < 0.02 and abs(b.std() - 1.0) < 0.02
    c = mi.make_config(0)
    assert c["n"] == 512 and abs(c["box"][0] - 21.72) < 1e-12
    for k in "xyz":
        assert (c[k] >= 0).all() and (c[k] < c["box"][0]).all()
    assert abs(c["vx"].mean()) < 1e-15
    sv = math.sqrt(mi.KB_EV_PER_K * 300.0 / mi.SI_MASS_AMU * mi.KAPPA)
    assert abs(sv - 2.980140e-3) < 1e-8
    v = np.concatenate([c["vx"], c["vy"], c["vz"]])
    assert abs(v.std() / sv - 1.0) < 0.06


def test_threaded_evaluation_equals_single_thread():
    """bench.py's all-core timing entry splits the atoms over threads; it must give what the oracle gives."""
    s = mi.silicon_crystal(3, 0.1, 800.0, 5)
    for pot, K in (("tersoff", 16), ("sw", 40)):
        par = mi.TERSOFF_SI_C if pot == "tersoff" else mi.SW_SI
        NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list(pot), K)
        ref = oracle.evaluate(pot, par, s["x"], s["y"], s["z"], s["box"], NN, NL, want=("pe", "f"))
        pe, f = oracle.evaluate_threads(pot, par, s["x"], s["y"], s["z"], s["box"], NN, NL, 3)
        assert (pe == ref["pe"]).all()
        assert np.abs(f - ref["f"]).max() <= 1e-13 * np.abs(ref["f"]).max()


# ---------------------------------------------------------------- Berendsen NPT (reading A18)
BER = dict(T0=300.0, tau_T=100.0, P0=0.0, tau_P=1000.0, beta=1.0 / 0.61)     # beta ~ 1/B of Si (98 GPa = 0.61 eV/A^3)


def dilute_gas(n=64, L=200.0, T=900.0, seed=3):
    """Atoms further apart than any cut-off for the whole run: no forces, P = N kB T / V exactly."""
    rng = np.random.default_rng(seed)
    g = np.stack(np.meshgrid(*[np.arange(4)] * 3, indexing="ij"), -1).reshape(-1, 3)[:n] * 40.0 + 20.0
    sv = math.sqrt(mi.KB_EV_PER_K * T / mi.SI_MASS_AMU * mi.KAPPA)
    v = rng.normal(size=(n, 3)) * sv
    return {"x": g[:, 0].copy(), "y": g[:, 1].copy(), "z": g[:, 2].copy(), "vx": v[:, 0].copy(),
            "vy": v[:, 1].copy(), "vz": v[:, 2].copy(), "box": np.array([L, L, L]), "mass": mi.SI_MASS_AMU, "n": n}


def test_berendsen_ideal_gas_closed_forms():
    """Without forces the weak-coupling recursions close: T_{k+1} = T_k + (dt/tau_T)(T0 - T_k), and with
    P = N kB T / V the volume obeys V_{k+1} = V_k (1 - beta dt/tau_P (P0 - P_k)).  Pins thermostat, barostat,
    the temperature and pressure definitions and their units."""
    s = dilute_gas()
    n, dt, steps = s["n"], 1.0, 40
    v2 = (s["vx"] ** 2 + s["vy"] ** 2 + s["vz"] ** 2).sum()
    T = s["mass"] * v2 / mi.KAPPA / (3 * n * mi.KB_EV_PER_K)
    V = float(np.prod(s["box"]))
    ber = dict(BER, P0=2e-7, tau_P=50.0, beta=1000.0)
    r = oracle.npt_run("tersoff", mi.TERSOFF_SI_C, s, steps, dt, 10, 3.5, 16, ber)
    for k in range(steps):
        P = n * mi.KB_EV_PER_K * T / V
        assert abs(r["T_trace"][k] - T) <= 1e-12 * T, k
        assert abs(r["P_trace"][k] - P) <= 1e-12 * P, k
        T, V = T + dt / ber["tau_T"] * (ber["T0"] - T), V * (1.0 - ber["beta"] * dt / ber["tau_P"] * (ber["P0"] - P))
        # positions and box are scaled AFTER the measurement, so the scaled velocities' T follows next step
    assert abs(float(np.prod(s["box"])) - V) <= 1e-12 * V


def test_berendsen_crystal_relaxes_to_zero_pressure_lattice_constant():
    """Physics pin: a cold Tersoff crystal started 1 % expanded contracts towards the zero-pressure lattice
    constant of the potential (5.432 A, tests/golden).  With beta = 1/B (B = 97.8 GPa = 0.6104 eV/A^3, the
    bulk modulus pinned in test_oracle_pins) weak coupling makes the pressure decay as exp(-t/tau_P)."""
    x, y, z, L = mi.diamond_lattice(2, 5.432 * 1.01)
    n = x.size
    s = {"x": x, "y": y, "z": z, "vx": np.zeros(n), "vy": np.zeros(n), "vz": np.zeros(n),
         "box": np.array([L, L, L]), "mass": mi.SI_MASS_AMU, "n": n}
    ber = dict(T0=1.0, tau_T=50.0, P0=0.0, tau_P=200.0, beta=1.0 / 0.6104)
    r = oracle.npt_run("tersoff", mi.TERSOFF_SI_C, s, 1000, 1.0, 10, 3.5, 16, ber)
    P = r["P_trace"]
    assert P[0] < 0                                              # expanded crystal: tensile
    assert 0.30 <= P[200] / P[0] <= 0.45                         # e^-1 = 0.37 (B softens a little under tension)
    assert abs(P[-1]) < 0.02 * abs(P[0])                         # e^-5
    assert abs(s["box"][0] / 2 - 5.432) < 0.001


# ---------------------------------------------------------------- Green-Kubo heat-current time series
def test_heat_current_series_is_the_energy_moment_rate():
    """Pins oracle_nve_heat_run against the identity P12 uses for a single evaluation, now along a trajectory:
    on a free (vacuum-padded) cluster d/dt sum_i r_i E_i = J_kin + J_pot, so the series' time integral over a
    window equals the change of the energy moment R = sum_i r_i E_i (trapezoid rule, error O(dt^2))."""
    x, y, z, L = mi.diamond_lattice(2)
    rng = np.random.default_rng(8)
    n = x.size
    box = np.array([60.0, 60.0, 60.0])
    s = {"x": x + 20 + rng.normal(size=n) * 0.05, "y": y + 20 + rng.normal(size=n) * 0.05,
         "z": z + 20 + rng.normal(size=n) * 0.05, "box": box, "mass": mi.SI_MASS_AMU, "n": n}
    v = rng.normal(size=(n, 3)) * 3e-3
    v -= v.mean(axis=0)
    s["vx"], s["vy"], s["vz"] = v[:, 0].copy(), v[:, 1].copy(), v[:, 2].copy()

    def moment(st):
        NN, NL = oracle.neighbors(st["x"], st["y"], st["z"], box, 3.5, 16)
        pe = oracle.evaluate("tersoff", mi.TERSOFF_SI_C, st["x"], st["y"], st["z"], box, NN, NL, want=("pe",))["pe"]
        e = 0.5 * st["mass"] / mi.KAPPA * (st["vx"] ** 2 + st["vy"] ** 2 + st["vz"] ** 2) + pe
        return np.array([(st[k] * e).sum() for k in "xyz"])
    errs = []
    for dt in (0.4, 0.2):
        st = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in s.items()}
        r0 = oracle.nve_heat_run("tersoff", mi.TERSOFF_SI_C, st, 1, dt, 10, 3.5, 16, 1)     # J at t = dt
        R0 = moment(st)
        nst = int(round(8.0 / dt))
        r = oracle.nve_heat_run("tersoff", mi.TERSOFF_SI_C, st, nst, dt, 10, 3.5, 16, 1, f=r0["f"])
        R1 = moment(st)
        Jt = np.vstack([r0["J_pot"] + r0["J_kin"], r["J_pot"] + r["J_kin"]])                 # t = dt .. dt (1 + nst)
        integral = dt * (Jt[0] / 2 + Jt[1:-1].sum(axis=0) + Jt[-1] / 2)
        errs.append(np.abs(integral - (R1 - R0)).max() / np.abs(R1 - R0).max())
    assert errs[0] < 2e-2 and 3.3 <= errs[0] / errs[1] <= 5.0, errs      # trapezoid + Verlet: O(dt^2)
