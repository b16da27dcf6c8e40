"""GPU parity of md_npt_run (Berendsen NPT) against the oracle's NPT loop."""
import numpy as np
import pytest
import torch

import md_inputs as mi
import oracle
import paper_1610_03343_b200 as md
from gpu_util import DEV, GpuSystem, assert_close_fp64

pytestmark = pytest.mark.gpu
PARAMS = {"tersoff": mi.TERSOFF_SI_C, "sw": mi.SW_SI}
BER = dict(T0=300.0, tau_T=100.0, P0=0.0, tau_P=1000.0, beta=1.0 / 0.6104)


@pytest.mark.parametrize("pot", ["tersoff", "sw"])
def test_npt_traces_box_and_snapshot(pot):
    s = mi.silicon_crystal(3, 0.05, 600.0, 27)
    K, rl = (16 if pot == "tersoff" else 32), mi.r_list(pot)
    g = GpuSystem(s, K)
    f = torch.zeros((3, g.n), dtype=torch.float64, device=DEV)
    box = list(g.box)
    Tt, Pt = md.md_npt_run(g.nl, pot, PARAMS[pot], g.n, g.x, g.y, g.z, g.vx, g.vy, g.vz, f, False, box, g.mass,
                           1.0, 25, 10, rl, BER)
    md.md_neighbors_status(g.nl)
    ref = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in s.items()}
    r = oracle.npt_run(pot, PARAMS[pot], ref, 25, 1.0, 10, rl, K if pot == "tersoff" else 40, BER)
    assert np.abs(np.array(Tt) - r["T_trace"]).max() <= 1e-9 * r["T_trace"].max()
    assert np.abs(np.array(Pt) - r["P_trace"]).max() <= 1e-9 * np.abs(r["P_trace"]).max()
    assert np.abs(np.array(box) - ref["box"]).max() <= 1e-12 * ref["box"][0]
    assert box[0] != s["box"][0]                               # the barostat acted
    g.box = box
    st = g.state()
    for k in ("x", "y", "z"):
        d = np.abs(st[k] - ref[k]); d = np.minimum(d, box[0] - d)
        assert d.max() <= 1e-9, k
    for k in ("vx", "vy", "vz"):
        assert np.abs(st[k] - ref[k]).max() <= 1e-11, k


def test_npt_ideal_gas_closed_form_on_gpu():
    """No forces: T_{k+1} = T_k + (dt/tau_T)(T0 - T_k) and P = n kB T / V, exactly as for the oracle."""
    n, L = 64, 200.0
    rng = np.random.default_rng(3)
    gpos = np.stack(np.meshgrid(*[np.arange(4)] * 3, indexing="ij"), -1).reshape(-1, 3) * 40.0 + 20.0
    v = rng.normal(size=(n, 3)) * 5e-3
    s = {"x": gpos[:, 0].copy(), "y": gpos[:, 1].copy(), "z": gpos[:, 2].copy(), "vx": v[:, 0].copy(),
         "vy": v[:, 1].copy(), "vz": v[:, 2].copy(), "box": np.array([L, L, L]), "mass": mi.SI_MASS_AMU}
    g = GpuSystem(s, 16)
    f = torch.zeros((3, n), dtype=torch.float64, device=DEV)
    box = list(g.box)
    ber = dict(BER, P0=2e-7, tau_P=50.0, beta=1000.0)
    Tt, Pt = md.md_npt_run(g.nl, "tersoff", mi.TERSOFF_SI_C, n, g.x, g.y, g.z, g.vx, g.vy, g.vz, f, False, box,
                           g.mass, 1.0, 30, 10, 3.5, ber)
    T = s["mass"] * (v ** 2).sum() / mi.KAPPA / (3 * n * mi.KB_EV_PER_K)
    V = L ** 3
    for k in range(30):
        P = n * mi.KB_EV_PER_K * T / V
        assert abs(Tt[k] - T) <= 1e-12 * T and abs(Pt[k] - P) <= 1e-12 * P, k
        T, V = T + 1.0 / ber["tau_T"] * (ber["T0"] - T), V * (1.0 - ber["beta"] / ber["tau_P"] * (ber["P0"] - P))
    assert abs(box[0] * box[1] * box[2] - V) <= 1e-12 * V
