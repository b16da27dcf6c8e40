"""GPU parity at BASELINE.json's full sizes, through the calls and launch configuration bench.py times.

512 000-atom configs (2, 3, 5): the oracle evaluates every atom (a few seconds each) and everything is
compared.  The 8 000 000-atom config (4): sampled outputs.  A sample is a spatial block of the big system
handed to the oracle as a free cluster; an atom further than 2 r_list from the block's faces has, inside
the block, every atom its force depends on (its neighbours and their neighbours), so the oracle's value
for it is the full system's value.  Two blocks: one in the interior of the box (coordinates untouched, so
the full FP64 tolerance applies) and one across the periodic corner (atoms beyond the faces are brought
next to the others by an exact shift of one box length).  For the corner block the GPU forms
r_ij = (x_j - x_i) -+ L with two roundings at |x| ~ 543 A (ulp 1.1e-13 A) where the cluster has one; with
bond stiffness ~ 30 eV/A^2 that is ~ 5e-12 eV/A of legitimate difference, so its absolute floor is 2e-11.
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


def full_eval(c, K, precision=md.MD_FP64):
    g = GpuSystem(c, K)
    mx = g.build(c["r_list"])
    out = g.force(c["potential"], c["params"], precision=precision)
    return g, mx, out


@pytest.mark.parametrize("index", [1, 2, 4])
def test_512k_configs_all_atoms_fp64(index):
    c = mi.make_config(index)
    K = c["max_neighbors"]
    g, mx, out = full_eval(c, K)
    NN, NL = g.export_list()
    rNN, rNL = oracle.neighbors(c["x"], c["y"], c["z"], c["box"], c["r_list"], K)
    assert mx == rNN.max()
    assert (NN == rNN).all() and (NL == rNL).all()                  # bit exact, all 512 000 rows
    ref = oracle.evaluate(c["potential"], c["params"], c["x"], c["y"], c["z"], c["box"], rNN, rNL,
                          v=(c["vx"], c["vy"], c["vz"]))
    assert_close_energy(out["pe"], ref["pe"])
    assert abs(math.fsum(out["pe"]) - math.fsum(ref["pe"])) <= 1e-12 * abs(math.fsum(ref["pe"]))
    assert_close_fp64("f", out["f"], ref["f"])
    assert_close_fp64("virial", out["virial"], ref["virial"])
    assert_close_fp64("heat", out["heat"], ref["heat"])
    assert np.abs(out["f"].sum(axis=1)).max() <= 1e-9               # momentum, 512 000 atoms


def test_config5_fp32_mode_against_fp64_oracle():
    c = mi.make_config(4)
    K = c["max_neighbors"]
    g, mx, out = full_eval(c, K, precision=md.MD_FP32)
    assert mx > 4                                                    # variable rows: the long-row path ran
    rNN, rNL = oracle.neighbors(c["x"], c["y"], c["z"], c["box"], c["r_list"], K)
    ref = oracle.evaluate("tersoff", c["params"], c["x"], c["y"], c["z"], c["box"], rNN, rNL,
                          v=(c["vx"], c["vy"], c["vz"]))
    assert abs(out["pe"].sum() - ref["pe"].sum()) <= 1e-4 * abs(ref["pe"].sum())
    assert_close_energy(out["pe"], ref["pe"], rel=1e-4)              # per atom (reading A10)
    assert_close_fp32("f", out["f"], ref["f"])
    assert_close_fp32("virial", out["virial"], ref["virial"])
    assert_close_fp32("heat", out["heat"], ref["heat"])


def block_cluster(c, lo, size, margin):
    """Atoms whose coordinates, taken relative to the periodic corner when lo < 0 (x -> x - L for
    x >= L + lo: exact, Sterbenz), lie in [lo, lo + size) on every axis.  Returns (global indices,
    coordinates [3][m] in that frame, mask of the atoms further than `margin` from the block's faces)."""
    L = c["box"]
    rel = []
    sel = np.ones(c["n"], dtype=bool)
    for a, k in enumerate("xyz"):
        v = c[k]
        r = np.where(v >= L[a] + lo, v - L[a], v) if lo < 0 else v
        rel.append(r)
        sel &= (r >= lo) & (r < lo + size)
    idx = np.nonzero(sel)[0]
    P = np.stack([r[idx] for r in rel])
    inner = np.ones(idx.size, dtype=bool)
    for a in range(3):
        inner &= (P[a] >= lo + margin) & (P[a] < lo + size - margin)
    return idx, P, inner


def test_8m_config_sampled_blocks():
    c = mi.make_config(3)
    K, rl = c["max_neighbors"], c["r_list"]
    g, mx, out = full_eval(c, K)
    assert mx in (4, 5)
    NN = torch.zeros(g.n, dtype=torch.int32, device=DEV)
    NLd = torch.full((K, g.n), -1, dtype=torch.int32, device=DEV)
    md.md_neighbors_export(g.nl, NN, NLd)
    torch.cuda.synchronize()
    NN = NN.cpu().numpy()
    size, margin = 70.0, 2 * rl + 0.25
    for lo, floor in ((200.0, 1e-12), (-35.0, 2e-11)):
        idx, P, inner = block_cluster(c, lo, size, margin)
        assert inner.sum() > 5000
        if lo > 0:
            X, big = P, np.array(c["box"])          # untouched coordinates in the original box: nothing wraps
        else:
            X, big = P + 55.0, np.array([110.0] * 3)   # free cluster; images are >= 40 A away
        cNN, cNL = oracle.neighbors(X[0], X[1], X[2], big, rl, K)
        v = tuple(c[k][idx] for k in ("vx", "vy", "vz"))
        ref = oracle.evaluate("tersoff", c["params"], X[0], X[1], X[2], big, cNN, cNL, v=v)
        # neighbour rows of interior atoms as sets of global indices: bit exact
        pick = np.nonzero(inner)[0][::7][:4000]
        rows_gpu = NLd[:, torch.from_numpy(idx[pick]).to(DEV)].cpu().numpy().T
        for q, a in enumerate(pick):
            want = np.sort(idx[cNL[a, :cNN[a]]])
            assert NN[idx[a]] == cNN[a] and (rows_gpu[q, :cNN[a]] == want).all()
        sub = idx[inner]
        assert_close_energy(out["pe"][sub], ref["pe"][inner])
        for name in ("f", "virial", "heat"):
            assert_close_fp64(name, out[name][:, sub], ref[name][:, inner], floor=floor)
