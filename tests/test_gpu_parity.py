"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element."""
import math

import numpy as np
import pytest
import torch

import md_inputs as mi
import oracle
import paper_1610_03343_b200 as md
from gpu_util import (DEV, GpuSystem, assert_close_energy, assert_close_fp32, assert_close_fp64, dev)

pytestmark = pytest.mark.gpu
PARAMS = {"tersoff": mi.TERSOFF_SI_C, "sw": mi.SW_SI}
KMAX = {"tersoff": 16, "sw": 32}

CASES = [  # potential, ncell, sigma, T, seed
    ("tersoff", 2, 0.05, 300.0, 1), ("tersoff", 4, 0.05, 300.0, mi.BASE_SEED), ("tersoff", 5, 0.15, 1500.0, 2),
    ("tersoff", 7, 0.25, 1500.0, 3), ("sw", 3, 0.05, 300.0, 4), ("sw", 5, 0.15, 1500.0, 5),
]


# ------------------------------------------------------------------ neighbour lists: bit exact
@pytest.mark.parametrize("pot,ncell,sigma,T,seed", CASES)
def test_neighbor_list_bit_exact(pot, ncell, sigma, T, seed):
    s = mi.silicon_crystal(ncell, sigma, T, seed)
    g = GpuSystem(s, KMAX[pot])
    mx = g.build(mi.r_list(pot))
    NN, NL = g.export_list()
    rNN, rNL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list(pot), KMAX[pot])
    assert mx == rNN.max()
    assert (NN == rNN).all()
    assert (NL == rNL).all()


def test_neighbor_list_random_gas_non_cubic_box():
    rng = np.random.default_rng(12)
    box = np.array([13.0, 17.5, 22.0])
    n = 1200
    P = rng.random((n, 3)) * box
    s = {"x": P[:, 0].copy(), "y": P[:, 1].copy(), "z": P[:, 2].copy(), "box": box}
    g = GpuSystem(s, 64)
    g.build(3.1)
    NN, NL = g.export_list()
    rNN, rNL = oracle.neighbors(s["x"], s["y"], s["z"], box, 3.1, 64, method="brute")
    assert (NN == rNN).all() and (NL == rNL).all()
    assert NN.min() < NN.max()


# ------------------------------------------------------------------ FP64 forces, all outputs
@pytest.mark.parametrize("pot,ncell,sigma,T,seed", CASES)
def test_force_virial_heat_energy_fp64(pot, ncell, sigma, T, seed):
    s = mi.silicon_crystal(ncell, sigma, T, seed)
    g = GpuSystem(s, KMAX[pot])
    g.build(mi.r_list(pot))
    out = g.force(pot, PARAMS[pot])
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list(pot), KMAX[pot])
    ref = oracle.evaluate(pot, PARAMS[pot], s["x"], s["y"], s["z"], s["box"], NN, NL,
                          v=(s["vx"], s["vy"], s["vz"]), precision="f80")
    assert_close_energy(out["pe"], ref["pe"])
    assert abs(math.fsum(out["pe"]) - math.fsum(ref["pe"])) <= 1e-12 * abs(math.fsum(ref["pe"]))
    assert_close_fp64("f", out["f"], ref["f"])                 # conventional (Alg. 1) forces
    assert_close_fp64("virial", out["virial"], ref["virial"])
    assert_close_fp64("heat", out["heat"], ref["heat"])


def test_force_with_imported_oracle_list_and_optional_outputs():
    s = mi.make_config(0)
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], s["r_list"], 16)
    g = GpuSystem(s, 16)
    g.import_list(NN, NL)
    ref = oracle.evaluate("tersoff", s["params"], s["x"], s["y"], s["z"], s["box"], NN, NL, precision="f80")
    full = g.force("tersoff", s["params"])
    only_f = g.force("tersoff", s["params"], want=("f",))
    only_pe = g.force("tersoff", s["params"], want=("pe",))
    assert_close_fp64("f", full["f"], ref["f"])
    assert (only_f["f"] == full["f"]).all()                    # bitwise: outputs do not depend on what is asked
    assert (only_pe["pe"] == full["pe"]).all()


def test_lean_register_kernel_next_to_general_path_atoms():
    """Force-only calls on a crystal use the 128-register lean kernel (no f_C terms); atoms with a list row longer
    than 4 or with a pair inside the cut-off window R < r < S take the general per-thread path inside the same
    launch, and their partners gather the records it pushes.  One atom is displaced so that both cases occur."""
    s = mi.silicon_crystal(8, 0.05, 300.0, 21)
    p = mi.TERSOFF_SI_C
    i = 1234
    NN0, NL0 = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list("tersoff"), 16)
    j = NL0[i][0]
    d = np.array([s[k][j] - s[k][i] for k in "xyz"])
    d -= s["box"] * np.round(d / s["box"])
    shift = -(0.5 / np.linalg.norm(d)) * d                    # stretch the bond i-j from ~2.35 A to ~2.85 A
    for a, k in enumerate("xyz"):
        s[k][i] = (s[k][i] + shift[a]) % s["box"][a]
    g = GpuSystem(s, 16)
    g.build(mi.r_list("tersoff"))
    max_row, long_rows = md.md_neighbors_row_stats(g.nl)
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list("tersoff"), 16)
    ref = oracle.evaluate("tersoff", p, s["x"], s["y"], s["z"], s["box"], NN, NL, precision="f80", want=("pe", "f"))
    dij = np.array([s[k][j] - s[k][i] for k in "xyz"])
    dij -= s["box"] * np.round(dij / s["box"])
    assert p["R"] < np.linalg.norm(dij) < p["S"]             # a window pair exists
    assert max_row > 4 and 0 < long_rows and long_rows * 256 <= g.n   # long rows exist, register kernel still chosen
    for _ in range(2):                                        # twice: a stale record of the first call must not help
        out = g.force("tersoff", p, want=("pe", "f"))
        assert_close_fp64("f", out["f"], ref["f"])
        assert_close_energy(out["pe"], ref["pe"])
    full = g.force("tersoff", p)                              # the instantiation with the virial own half
    assert_close_fp64("f", full["f"], ref["f"])


def test_general_path_interstitial_ten_neighbours():
    """An atom at the tetrahedral interstitial site has 10 neighbours inside the force range, 6 of them inside the
    cut-off window; it and its neighbours (rows of 5..10 entries) take the warp-per-atom general path of both
    register kernels while the other 4086 atoms take the register bodies; n = 4097 leaves a ragged last tile."""
    s = mi.silicon_crystal(8, 0.05, 300.0, 33)
    p = mi.TERSOFF_SI_C
    for k in "xyz":
        s[k] = np.append(s[k], 3.5 * mi.SI_LATTICE_A)
    for k in ("vx", "vy", "vz"):
        s[k] = np.append(s[k], 1e-3)
    g = GpuSystem(s, 16)
    g.build(mi.r_list("tersoff"))
    max_row, long_rows = md.md_neighbors_row_stats(g.nl)
    assert max_row >= 10 and long_rows * 256 <= g.n
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list("tersoff"), 16)
    ref = oracle.evaluate("tersoff", p, s["x"], s["y"], s["z"], s["box"], NN, NL, v=(s["vx"], s["vy"], s["vz"]),
                          precision="f80")
    lean = g.force("tersoff", p, want=("pe", "f"))            # k_tersoff_lean + general path
    full = g.force("tersoff", p)                              # k_tersoff_lean with the virial own half + general path
    for out in (lean, full):
        assert_close_fp64("f", out["f"], ref["f"])
        assert_close_energy(out["pe"], ref["pe"])
    assert_close_fp64("virial", full["virial"], ref["virial"])
    assert_close_fp64("heat", full["heat"], ref["heat"])
    f32 = g.force("tersoff", p, precision=md.MD_FP32, want=("pe", "f"))
    assert_close_fp32("f", f32["f"], ref["f"])


def test_run_to_run_bitwise_reproducible():
    s = mi.silicon_crystal(6, 0.15, 1500.0, 77)
    a = GpuSystem(s, 16); a.build(3.5); oa = a.force("tersoff", mi.TERSOFF_SI_C)
    b = GpuSystem(s, 16); b.build(3.5); ob = b.force("tersoff", mi.TERSOFF_SI_C)
    for k in oa:
        assert (oa[k] == ob[k]).all(), k


# ------------------------------------------------------------------ FP32 mode
@pytest.mark.parametrize("pot,ncell,sigma,T,seed", [("tersoff", 5, 0.15, 1500.0, 2), ("sw", 5, 0.05, 300.0, 8)])
def test_fp32_mode_within_1e4_of_fp64_oracle(pot, ncell, sigma, T, seed):
    s = mi.silicon_crystal(ncell, sigma, T, seed)
    g = GpuSystem(s, KMAX[pot])
    g.build(mi.r_list(pot))
    out = g.force(pot, PARAMS[pot], precision=md.MD_FP32)
    NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], s["box"], mi.r_list(pot), KMAX[pot])
    ref = oracle.evaluate(pot, PARAMS[pot], s["x"], s["y"], s["z"], s["box"], NN, NL,
                          v=(s["vx"], s["vy"], s["vz"]))
    assert np.abs(out["pe"] - ref["pe"]).max() <= 1e-4 * np.abs(ref["pe"]).min()
    assert abs(out["pe"].sum() - ref["pe"].sum()) <= 1e-4 * abs(ref["pe"].sum())
    assert_close_fp32("f", out["f"], ref["f"])
    assert_close_fp32("virial", out["virial"], ref["virial"])
    assert_close_fp32("heat", out["heat"], ref["heat"])


# ------------------------------------------------------------------ degenerate cases
def test_dimer_and_isolated_atoms_zeta_zero_path():
    box = np.array([40.0, 40.0, 40.0])
    for r in (2.0, 2.35, 2.85, 2.95, 3.2):
        s = {"x": np.array([10.0, 10.0 + r, 30.0]), "y": np.array([10.0, 10.0, 30.0]),
             "z": np.array([10.0, 10.0, 30.0]), "box": box}
        g = GpuSystem(s, 16)
        g.build(3.5)
        out = g.force("tersoff", mi.TERSOFF_SI_C)
        NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], box, 3.5, 16)
        ref = oracle.evaluate("tersoff", mi.TERSOFF_SI_C, s["x"], s["y"], s["z"], box, NN, NL,
                              v=(np.zeros(3),) * 3, precision="f80")
        assert np.isfinite(out["f"]).all()
        assert_close_fp64("pe", out["pe"], ref["pe"], rel=1e-12, floor=1e-15)
        assert_close_fp64("f", out["f"], ref["f"])
        assert (out["f"][:, 2] == 0).all() and out["pe"][2] == 0


def test_bent_trimers_and_skew_dimers_all_outputs():
    """The clusters of tests/test_oracle_peratom_pins.py (closed-form pins of the oracle's per-atom U, F, W, J)
    through the CUDA path: a central atom with two ends out of each other's range, bonds below R, inside the
    cut-off window, near the SW cut-off; vacuum-padded non-cubic box; n = 3 (one ragged CTA)."""
    def unit(theta, phi):
        return np.array([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])
    v = np.array([[0.31, -0.72, 0.23], [-0.44, 0.15, 0.61], [0.08, 0.52, -0.37]])
    box = np.array([60.0, 55.0, 50.0])
    cases = [("tersoff", 2.30, 2.45, 100.0), ("tersoff", 2.35, 2.85, 112.0), ("tersoff", 2.78, 2.93, 95.0),
             ("sw", 2.30, 2.45, 140.0), ("sw", 2.20, 3.10, 150.0), ("tersoff", 2.35, None, 0.0), ("sw", 3.2, None, 0.0)]
    for pot, r1, r2, ang in cases:
        u1 = unit(0.7, 1.9)
        c0 = np.array([20.3, 21.7, 19.1])
        pos = [c0, c0 + r1 * u1]
        if r2 is not None:
            ax = np.cross(u1, np.array([0.2, -0.5, 0.84])); ax /= np.linalg.norm(ax)
            a = np.deg2rad(ang)
            u2 = u1 * np.cos(a) + np.cross(ax, u1) * np.sin(a) + ax * np.dot(ax, u1) * (1 - np.cos(a))
            pos.append(c0 + r2 * u2)
        pos = np.stack(pos)
        n = pos.shape[0]
        s = {"x": pos[:, 0].copy(), "y": pos[:, 1].copy(), "z": pos[:, 2].copy(), "box": box,
             "vx": v[:n, 0].copy(), "vy": v[:n, 1].copy(), "vz": v[:n, 2].copy()}
        g = GpuSystem(s, KMAX[pot])
        g.build(mi.r_list(pot))
        out = g.force(pot, PARAMS[pot])
        NN, NL = oracle.neighbors(s["x"], s["y"], s["z"], box, mi.r_list(pot), KMAX[pot])
        ref = oracle.evaluate(pot, PARAMS[pot], s["x"], s["y"], s["z"], box, NN, NL,
                              v=(s["vx"], s["vy"], s["vz"]), precision="f80")
        assert_close_energy(out["pe"], ref["pe"])
        for k in ("f", "virial", "heat"):
            assert_close_fp64(f"{pot} {r1} {r2} {k}", out[k], ref[k])


def test_perfect_lattice_zero_force():
    x, y, z, L = mi.diamond_lattice(4)
    s = {"x": x, "y": y, "z": z, "box": np.array([L, L, L])}
    for pot in ("tersoff", "sw"):
        g = GpuSystem(s, KMAX[pot])
        mx = g.build(mi.r_list(pot))
        assert mx == (4 if pot == "tersoff" else 16)
        out = g.force(pot, PARAMS[pot])
        assert np.abs(out["f"]).max() <= 1e-12


def test_errors_and_empty_input():
    s = mi.silicon_crystal(2, 0.05, 300.0, 1)
    g = GpuSystem(s, 16)
    with pytest.raises(md.MDError) as e:                      # force before any list
        g.force("tersoff", mi.TERSOFF_SI_C)
    assert e.value.code == md.MD_ERR_NO_LIST
    with pytest.raises(md.MDError) as e:                      # 10.86 / 4.0 -> 2 cells
        md.md_build_neighbors(g.nl, g.n, g.x, g.y, g.z, g.box, 4.0)
    assert e.value.code == md.MD_ERR_BOX_TOO_SMALL
    small = GpuSystem(s, 3)                                    # rows of 4 do not fit in K = 3
    md.md_build_neighbors(small.nl, small.n, small.x, small.y, small.z, small.box, 3.5)
    assert md.md_neighbors_status(small.nl, check=False) == md.MD_ERR_NEIGHBOR_OVERFLOW
    with pytest.raises(md.MDError):
        md.md_neighbors_create(10, 65)
    # n = 0 is legal everywhere
    e0 = md.md_neighbors_create(0, 16)
    z0 = torch.zeros(0, dtype=torch.float64, device=DEV)
    md.md_build_neighbors(e0, 0, z0, z0, z0, [10.0, 10.0, 10.0], 3.0)
    md.md_tersoff_force(e0, 0, z0, z0, z0, z0, z0, z0, [10.0, 10.0, 10.0], mi.TERSOFF_SI_C, f=z0)
    md.md_velocity_verlet_step(0, 0, z0, z0, z0, z0, z0, z0, z0, 28.0, 1.0, [10.0, 10.0, 10.0])
    assert md.md_neighbors_status(e0) == 0


# ------------------------------------------------------------------ integrator and NVE loop
def test_velocity_verlet_half_steps_match_oracle():
    s = mi.silicon_crystal(3, 0.05, 300.0, 9)
    rng = np.random.default_rng(1)
    f = rng.normal(size=(3, s["n"]))
    s["x"][:5] = [0.0, 1e-9, s["box"][0] - 1e-12, s["box"][0] * (1 - 2e-16), 5.0]   # wrap edges
    s["vx"][:5] = [-1e-3, -1.0, 1.0, 1e-3, 0.0]
    g = GpuSystem(s, 16)
    fd = dev(f)
    md.md_velocity_verlet_step(0, g.n, g.x, g.y, g.z, g.vx, g.vy, g.vz, fd, g.mass, 1.0, g.box)
    ref = {k: s[k].copy() for k in ("x", "y", "z", "vx", "vy", "vz")}
    oracle.vv_kick_drift(ref["x"], ref["y"], ref["z"], ref["vx"], ref["vy"], ref["vz"], f, s["mass"], 1.0, s["box"])
    st = g.state()
    for k in ref:
        assert np.abs(st[k] - ref[k]).max() <= 1e-13 * max(1.0, np.abs(ref[k]).max()), k
    for k in "xyz":
        assert (st[k] >= 0).all() and (st[k] < s["box"][0]).all()
    md.md_velocity_verlet_step(1, g.n, g.x, g.y, g.z, g.vx, g.vy, g.vz, fd, g.mass, 1.0, g.box)
    oracle.vv_kick(ref["vx"], ref["vy"], ref["vz"], f, s["mass"], 1.0)
    st = g.state()
    for k in ("vx", "vy", "vz"):
        assert np.abs(st[k] - ref[k]).max() <= 1e-15


@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_nve_run_short_trajectory_and_snapshot_parity(pot):
    """25 steps stay within rounding-amplified distance of the oracle trajectory; then snapshot parity:
    the GPU state is handed to the oracle and one evaluation is compared at full tolerance."""
    s = mi.silicon_crystal(3, 0.05, 300.0, 15)
    K = KMAX[pot]
    g = GpuSystem(s, K)
    n = g.n
    f = torch.zeros((3, n), dtype=torch.float64, device=DEV)
    pe = torch.zeros(n, dtype=torch.float64, device=DEV)
    md.md_nve_run(g.nl, pot, PARAMS[pot], n, g.x, g.y, g.z, g.vx, g.vy, g.vz, f, False, pe, g.box, g.mass,
                  1.0, 25, 10, mi.r_list(pot))
    md.md_neighbors_status(g.nl)
    ref = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in s.items()}
    r = oracle.nve_run(pot, PARAMS[pot], ref, 25, 1.0, 10, mi.r_list(pot), K)
    st = g.state()
    for k in ("x", "y", "z"):
        d = np.abs(st[k] - ref[k]); d = np.minimum(d, s["box"][0] - d)
        assert d.max() <= 1e-9, k
    for k in ("vx", "vy", "vz"):
        assert np.abs(st[k] - ref[k]).max() <= 1e-11, k
    # snapshot parity on the GPU's own final state (list of step 20, as the GPU used it)
    NN, NL = g.export_list()
    snap = oracle.evaluate(pot, PARAMS[pot], st["x"], st["y"], st["z"], st["box"], NN, NL, precision="f80")
    assert_close_fp64("f", f.cpu().numpy(), snap["f"])
    assert_close_energy(pe.cpu().numpy(), snap["pe"])
    assert abs(math.fsum(r["pe"]) - math.fsum(snap["pe"])) <= 1e-9 * abs(math.fsum(snap["pe"]))


@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_nve_energy_conservation_on_gpu(pot):
    s = mi.silicon_crystal(4, 0.05, 300.0, 19)
    K = KMAX[pot]
    dev_e = []
    for dt, nsteps in ((1.0, 100), (0.5, 200)):
        g = GpuSystem(s, K)
        n = g.n
        f = torch.zeros((3, n), dtype=torch.float64, device=DEV)
        pe = torch.zeros(n, dtype=torch.float64, device=DEV)

        def total():
            ke = 0.5 * g.mass * float((g.vx ** 2 + g.vy ** 2 + g.vz ** 2).sum()) / mi.KAPPA
            return ke + float(pe.sum())
        md.md_nve_run(g.nl, pot, PARAMS[pot], n, g.x, g.y, g.z, g.vx, g.vy, g.vz, f, False, pe, g.box, g.mass,
                      dt, 0, 10, mi.r_list(pot))
        e0 = total()
        worst = 0.0
        for _ in range(nsteps // 10):
            md.md_nve_run(g.nl, pot, PARAMS[pot], n, g.x, g.y, g.z, g.vx, g.vy, g.vz, f, True, pe, g.box, g.mass,
                          dt, 10, 10, mi.r_list(pot))
            worst = max(worst, abs(total() - e0) / n)
        md.md_neighbors_status(g.nl)
        dev_e.append(worst)
    assert dev_e[0] <= 1e-4, dev_e
    assert 3.0 <= dev_e[0] / dev_e[1] <= 5.0, dev_e


@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_nve_run_is_bitwise_the_composition_of_the_four_calls(pot):
    """md_nve_run fuses the half-kicks into its gather kernel; the result must be bit for bit what the
    public calls give when composed by hand: kick+drift, [build], force, kick."""
    s = mi.silicon_crystal(3, 0.05, 300.0, 21)
    K, P, rl = KMAX[pot], PARAMS[pot], mi.r_list(pot)
    force = md.md_tersoff_force if pot == "tersoff" else md.md_sw_force
    a, b = GpuSystem(s, K), GpuSystem(s, K)
    n = a.n
    fa = torch.zeros((3, n), dtype=torch.float64, device=DEV)
    fb = torch.zeros((3, n), dtype=torch.float64, device=DEV)
    pea = torch.zeros(n, dtype=torch.float64, device=DEV)
    peb = torch.zeros(n, dtype=torch.float64, device=DEV)
    nsteps, every, dt = 13, 5, 1.0
    md.md_nve_run(a.nl, pot, P, n, a.x, a.y, a.z, a.vx, a.vy, a.vz, fa, False, pea, a.box, a.mass, dt, nsteps,
                  every, rl)
    md.md_build_neighbors(b.nl, n, b.x, b.y, b.z, b.box, rl)
    force(b.nl, n, b.x, b.y, b.z, b.vx, b.vy, b.vz, b.box, P, f=fb)
    for step in range(nsteps):
        md.md_velocity_verlet_step(0, n, b.x, b.y, b.z, b.vx, b.vy, b.vz, fb, b.mass, dt, b.box)
        if step % every == 0:
            md.md_build_neighbors(b.nl, n, b.x, b.y, b.z, b.box, rl)
        force(b.nl, n, b.x, b.y, b.z, b.vx, b.vy, b.vz, b.box, P, pe=peb, f=fb)
        md.md_velocity_verlet_step(1, n, b.x, b.y, b.z, b.vx, b.vy, b.vz, fb, b.mass, dt, b.box)
    md.md_neighbors_status(a.nl); md.md_neighbors_status(b.nl)
    sa, sb = a.state(), b.state()
    for k in ("x", "y", "z", "vx", "vy", "vz"):
        assert (sa[k] == sb[k]).all(), k
    assert (fa.cpu().numpy() == fb.cpu().numpy()).all()
    assert (pea.cpu().numpy() == peb.cpu().numpy()).all()
    # and continuing a run (f_valid = 1, first_step > 0) is the same as one long run
    c = GpuSystem(s, K)
    fc = torch.zeros((3, n), dtype=torch.float64, device=DEV)
    md.md_nve_run(c.nl, pot, P, n, c.x, c.y, c.z, c.vx, c.vy, c.vz, fc, False, None, c.box, c.mass, dt, 6, every, rl)
    md.md_nve_run(c.nl, pot, P, n, c.x, c.y, c.z, c.vx, c.vy, c.vz, fc, True, None, c.box, c.mass, dt, nsteps - 6,
                  every, rl, first_step=6)
    sc = c.state()
    for k in ("x", "y", "z", "vx", "vy", "vz"):
        assert (sa[k] == sc[k]).all(), k


def test_nve_run_host_matches_device_run():
    s = mi.silicon_crystal(3, 0.05, 300.0, 15)
    g = GpuSystem(s, 16)
    n = g.n
    f = torch.zeros((3, n), dtype=torch.float64, device=DEV)
    pe = torch.zeros(n, dtype=torch.float64, device=DEV)
    md.md_nve_run(g.nl, "tersoff", mi.TERSOFF_SI_C, n, g.x, g.y, g.z, g.vx, g.vy, g.vz, f, False, pe, g.box,
                  g.mass, 1.0, 12, 10, 3.5)
    h = {k: torch.from_numpy(s[k].copy()).pin_memory() for k in ("x", "y", "z", "vx", "vy", "vz")}
    hf = torch.zeros((3, n), dtype=torch.float64).pin_memory()
    hpe = torch.zeros(n, dtype=torch.float64).pin_memory()
    nl2 = md.md_neighbors_create(n, 16)
    md.md_nve_run_host(nl2, "tersoff", mi.TERSOFF_SI_C, n, h["x"], h["y"], h["z"], h["vx"], h["vy"], h["vz"],
                       hf, hpe, g.box, g.mass, 1.0, 12, 10, 3.5)
    st = g.state()
    for k in h:
        assert (h[k].numpy() == st[k]).all(), k
    assert (hf.numpy() == f.cpu().numpy()).all() and (hpe.numpy() == pe.cpu().numpy()).all()
