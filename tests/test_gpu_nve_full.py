"""GPU parity of the kernels bench.py actually times (md_nve_run: pair kernel + k_gather_vv) at BASELINE.json's
full sizes, the FP32 NVE path, energy drift over the configs' own run lengths, and guard bands around the
caller's arrays (compute-sanitizer is closed on this GPU pool, so out-of-range writes are caught this way).

Trajectories are chaotic, so parity after many steps is snapshot parity: the GPU's final state
and the list it used are handed to the oracle and ONE evaluation is compared at the full tolerance.
"""
import math

import numpy as np
import pytest
import torch

import md_inputs as mi
import oracle
import paper_1610_03343_b200 as md
from gpu_util import (DEV, GpuSystem, assert_close_energy, assert_close_fp32, assert_close_fp64)

pytestmark = pytest.mark.gpu
PARAMS = {"tersoff": mi.TERSOFF_SI_C, "sw": mi.SW_SI}


def nve(g, c, f, pe, nsteps, f_valid, precision=md.MD_FP64, first_step=0):
    md.md_nve_run(g.nl, c["potential"], c["params"], g.n, g.x, g.y, g.z, g.vx, g.vy, g.vz, f, f_valid, pe, g.box,
                  g.mass, c["dt"], nsteps, c["rebuild_every"], c["r_list"], precision=precision,
                  first_step=first_step)


def total_energy(g, pe):
    ke = 0.5 * g.mass * float((g.vx ** 2 + g.vy ** 2 + g.vz ** 2).sum()) / mi.KAPPA
    return ke + float(pe.sum())


@pytest.mark.parametrize("index,precision", [(1, md.MD_FP64), (2, md.MD_FP64), (4, md.MD_FP64), (4, md.MD_FP32)])
def test_512k_nve_run_two_cycles_then_snapshot_parity(index, precision):
    """Two rebuild cycles (20 steps) of md_nve_run on the 512 000-atom configs 2, 3, 5 (5 also in FP32 mode:
    k_gather_vv<float>), then the forces and energies md_nve_run left behind against the oracle's evaluation
    of the same state with the same list."""
    c = mi.make_config(index)
    K = c["max_neighbors"]
    g = GpuSystem(c, K)
    f = torch.full((3, g.n), float("nan"), dtype=torch.float64, device=DEV)
    pe = torch.full((g.n,), float("nan"), dtype=torch.float64, device=DEV)
    nve(g, c, f, pe, 20, False, precision)
    md.md_neighbors_status(g.nl)
    st = g.state()
    NN, NL = g.export_list()
    ref = oracle.evaluate(c["potential"], c["params"], st["x"], st["y"], st["z"], st["box"], NN, NL, want=("pe", "f"))
    got_f, got_pe = f.cpu().numpy(), pe.cpu().numpy()
    if precision == md.MD_FP64:
        assert_close_fp64("f", got_f, ref["f"])
        assert_close_energy(got_pe, ref["pe"])
        assert abs(math.fsum(got_pe) - math.fsum(ref["pe"])) <= 1e-12 * abs(math.fsum(ref["pe"]))
    else:
        assert_close_fp32("f", got_f, ref["f"])
        assert_close_energy(got_pe, ref["pe"], rel=1e-4)
        assert abs(got_pe.sum() - ref["pe"].sum()) <= 1e-4 * abs(ref["pe"].sum())
    # the state moved (this is not the initial configuration) and stayed inside the box
    assert np.abs(st["x"] - c["x"]).max() > 1e-3
    for k in "xyz":
        assert (st[k] >= 0).all() and (st[k] < st["box"][0]).all()


@pytest.mark.parametrize("pot,precision", [("tersoff", md.MD_FP32), ("sw", md.MD_FP32)])
def test_fp32_nve_run_small_snapshot_parity(pot, precision):
    """25 FP32-mode steps on 1000 atoms (ragged tile tail), both potentials, then snapshot parity against the
    FP64 oracle at the FP32 tolerance (reading A10)."""
    s = mi.silicon_crystal(5, 0.15 if pot == "tersoff" else 0.05, 1500.0 if pot == "tersoff" else 300.0, 31)
    K = 16 if pot == "tersoff" else 32
    c = dict(s, potential=pot, params=PARAMS[pot], dt=0.5, rebuild_every=10, r_list=mi.r_list(pot))
    g = GpuSystem(s, K)
    f = torch.zeros((3, g.n), dtype=torch.float64, device=DEV)
    pe = torch.zeros(g.n, dtype=torch.float64, device=DEV)
    nve(g, c, f, pe, 25, False, precision)
    md.md_neighbors_status(g.nl)
    st = g.state()
    NN, NL = g.export_list()
    ref = oracle.evaluate(pot, PARAMS[pot], st["x"], st["y"], st["z"], st["box"], NN, NL, want=("pe", "f"))
    assert_close_fp32("f", f.cpu().numpy(), ref["f"])
    assert_close_energy(pe.cpu().numpy(), ref["pe"], rel=1e-4)


def max_energy_deviation(c, dt, nsteps):
    g = GpuSystem(c, c["max_neighbors"])
    cc = dict(c, dt=dt)
    f = torch.zeros((3, g.n), dtype=torch.float64, device=DEV)
    pe = torch.zeros(g.n, dtype=torch.float64, device=DEV)
    nve(g, cc, f, pe, 0, False)
    e0 = total_energy(g, pe)
    worst, done = 0.0, 0
    while done < nsteps:
        k = min(100, nsteps - done)
        nve(g, cc, f, pe, k, True, first_step=done)
        done += k
        worst = max(worst, abs(total_energy(g, pe) - e0) / g.n)
    md.md_neighbors_status(g.nl)
    return worst


@pytest.mark.parametrize("index", [1, 2])
def test_nve_energy_drift_over_config_length(index):
    """no drift above 1e-4 eV/atom over the configs' own lengths (1000 steps at 1 fs, configs 2 and
    3, 300 K), list rebuilt every 10 steps, 512 000 atoms."""
    c = mi.make_config(index)
    assert max_energy_deviation(c, c["dt"], c["steps"]) <= 1e-4


def test_nve_energy_config5_bounded_and_second_order():
    """Config 5 (sigma = 0.15 A, 1500 K start) equilibrates near 3000 K; SURVEY P13's 1e-4 eV/atom was probed
    at 300 K and does not transfer.  The oracle's own velocity-Verlet on this recipe (512 and 1728 atoms, 200
    steps of 0.5 fs) deviates by 2.8e-4 .. 3.0e-4 eV/atom, and by 6.8e-5 .. 7.2e-5 at 0.25 fs (ratio 4.1,
    _work probe recorded in DESIGN.md section 5).  So: the same bound with a little room, and the error must
    fall by ~4 when dt is halved over the same 100 fs (a bounded second-order fluctuation, not a drift)."""
    c = mi.make_config(4)
    e1 = max_energy_deviation(c, 0.5, 200)
    e2 = max_energy_deviation(c, 0.25, 400)
    assert e1 <= 4e-4, e1
    assert 3.0 <= e1 / e2 <= 5.0, (e1, e2)


def test_fp32_per_atom_error_distribution_config5():
    """Reading A10's per-atom bound is |dF_i| <= 1e-4 RMS_k|F_k|.  Measured on config 5 (512 000 atoms): the
    assertion is that bound itself, not ten times it."""
    c = mi.make_config(4)
    g = GpuSystem(c, c["max_neighbors"])
    g.build(c["r_list"])
    out = g.force("tersoff", c["params"], precision=md.MD_FP32)
    NN, NL = g.export_list()
    ref = oracle.evaluate("tersoff", c["params"], c["x"], c["y"], c["z"], c["box"], NN, NL,
                          v=(c["vx"], c["vy"], c["vz"]))
    for name in ("f", "virial", "heat"):
        d = out[name] - ref[name]
        per_atom = np.sqrt((d ** 2).sum(axis=0))
        rms = np.sqrt((ref[name] ** 2).sum(axis=0).mean())
        assert per_atom.max() <= 1e-4 * rms, (name, per_atom.max() / rms)
    assert_close_energy(out["pe"], ref["pe"], rel=1e-4)


@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_guard_bands_around_caller_arrays(pot):
    """Every caller-owned array sits between two 4 KiB bands of a sentinel pattern; after a build, a full-output
    force call and an NVE run (n = 1000: tiles with a ragged tail) the bands must be untouched and every
    output element written (no NaN sentinel left)."""
    s = mi.silicon_crystal(5, 0.15, 1500.0, 44)
    n, K, G = s["x"].size, (16 if pot == "tersoff" else 32), 512
    SENT = -7.25e300

    def guarded(rows, init=None):
        buf = torch.full((rows * n + 2 * G,), SENT, dtype=torch.float64, device=DEV)
        view = buf[G:G + rows * n].view(rows, n) if rows > 1 else buf[G:G + n]
        view.fill_(float("nan")) if init is None else view.copy_(torch.as_tensor(init, device=DEV))
        return buf, view
    bufs = {}
    arr = {}
    for k in ("x", "y", "z", "vx", "vy", "vz"):
        bufs[k], arr[k] = guarded(1, s[k])
    for k, rows in (("pe", 1), ("f", 3), ("virial", 9), ("heat", 3)):
        bufs[k], arr[k] = guarded(rows)
    nl = md.md_neighbors_create(n, K)
    box = [float(b) for b in s["box"]]
    md.md_build_neighbors(nl, n, arr["x"], arr["y"], arr["z"], box, mi.r_list(pot))
    fn = md.md_tersoff_force if pot == "tersoff" else md.md_sw_force
    fn(nl, n, arr["x"], arr["y"], arr["z"], arr["vx"], arr["vy"], arr["vz"], box, PARAMS[pot], md.MD_FP64,
       pe=arr["pe"], f=arr["f"], virial=arr["virial"], heat=arr["heat"])
    md.md_neighbors_status(nl)
    for k in ("pe", "f", "virial", "heat"):
        assert not torch.isnan(arr[k]).any(), k
    md.md_nve_run(nl, pot, PARAMS[pot], n, arr["x"], arr["y"], arr["z"], arr["vx"], arr["vy"], arr["vz"], arr["f"],
                  True, arr["pe"], box, float(s["mass"]), 0.5, 23, 10, mi.r_list(pot))
    md.md_neighbors_status(nl)
    for k, b in bufs.items():
        assert (b[:G] == SENT).all() and (b[-G:] == SENT).all(), k
        assert torch.isfinite(arr[k]).all(), k


@pytest.mark.parametrize("pot,ncell,sigma", [("sw", 6, 0.05), ("sw", 5, 0.15), ("tersoff", 6, 0.15)])
def test_sorted_kernels_run_to_run_bitwise_reproducible(pot, ncell, sigma):
    """The sorted loop kernels stage data through shared memory behind barriers (pair_sort.cuh); a missing
    barrier shows up as run-to-run differences.  Five evaluations on fresh handles must agree bit for bit."""
    s = mi.silicon_crystal(ncell, sigma, 1500.0, 91)
    K = 16 if pot == "tersoff" else 32
    first = None
    for _ in range(5):
        g = GpuSystem(s, K)
        g.build(mi.r_list(pot))
        out = g.force(pot, PARAMS[pot])
        if first is None:
            first = out
        else:
            for k in out:
                assert (out[k] == first[k]).all(), k
