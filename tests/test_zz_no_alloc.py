"""md_tersoff_force_static -- the entry point that allocates nothing (pair records in a fixed device array of the
library) -- against the handle-based md_tersoff_force and the oracle, on calls in a row that share the array.

Collected last on purpose (file name): the suite runs with pytest -x.  Needs nothing from the tests before it and
passes alone in a fresh process as well as after them."""
import pytest
import torch

import md_inputs as mi
import oracle
import paper_1610_03343_b200 as md
from gpu_util import DEV, GpuSystem, assert_close_energy, assert_close_fp64

pytestmark = pytest.mark.gpu

K = 16
R_LIST = 3.5


class Case:
    """A seeded silicon configuration, its list on the device, and the existing path's U_i and F_i."""

    def __init__(self, ncell, sigma, T, seed):
        self.s = mi.silicon_crystal(ncell, sigma, T, seed)
        self.g = GpuSystem(self.s, K)
        self.g.build(R_LIST)
        self.n = self.g.n
        self.NN = torch.zeros(self.n, dtype=torch.int32, device=DEV)
        self.NL = torch.zeros((K, self.n), dtype=torch.int32, device=DEV)
        md.md_neighbors_export(self.g.nl, self.NN, self.NL)
        self.ref = self.g.force("tersoff", mi.TERSOFF_SI_C, want=("pe", "f"))

    def static_call(self, want_pe=True, want_f=True):
        n = self.n
        pe = torch.full((n,), float("nan"), dtype=torch.float64, device=DEV) if want_pe else None
        f = torch.full((3, n), float("nan"), dtype=torch.float64, device=DEV) if want_f else None
        st = torch.full((1,), -1, dtype=torch.int32, device=DEV)
        g = self.g
        md.md_tersoff_force_static(n, K, self.NN, self.NL, g.x, g.y, g.z, g.box, mi.TERSOFF_SI_C, pe=pe, f=f, status=st)
        return pe, f, st

    def check(self, pe, f, st):
        torch.cuda.synchronize()
        assert int(st.item()) == 0
        assert_close_energy(pe.cpu().numpy(), self.ref["pe"])
        assert_close_fp64("f", f.cpu().numpy(), self.ref["f"])


def test_static_scratch_force_matches_handle_path_on_calls_in_a_row():
    a = Case(5, 0.15, 1500.0, 11)          # 1000 atoms, hot: rows of 4 and more in range, window pairs
    b = Case(4, 0.05, 300.0, 12)           # 512 atoms: another n, so every record lands somewhere else in the array
    # two calls in a row on one stream, checked only afterwards: the second reuses the array the first filled
    ra = a.static_call()
    rb = b.static_call()
    a.check(*ra)
    b.check(*rb)
    # and again the first system on top of the second's leftovers; the call must not allocate device memory
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    md.md_tersoff_force_static(a.n, K, a.NN, a.NL, a.g.x, a.g.y, a.g.z, a.g.box, mi.TERSOFF_SI_C,
                               pe=ra[0], f=ra[1], status=ra[2])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0
    a.check(*ra)
    # the oracle on the same list and positions, at the tolerances of the parity tests
    NN, NL = a.g.export_list()
    ref = oracle.evaluate("tersoff", mi.TERSOFF_SI_C, a.s["x"], a.s["y"], a.s["z"], a.s["box"], NN, NL,
                          v=(a.s["vx"], a.s["vy"], a.s["vz"]), precision="f80")
    assert_close_energy(ra[0].cpu().numpy(), ref["pe"])
    assert_close_fp64("f", ra[1].cpu().numpy(), ref["f"])
    # outputs are optional one by one
    pe, _, st = a.static_call(want_f=False)
    _, f, st2 = a.static_call(want_pe=False)
    torch.cuda.synchronize()
    assert int(st.item()) == 0 and int(st2.item()) == 0
    assert (pe == ra[0]).all() and (f == ra[1]).all()       # same inputs, same array: bitwise the same


def test_static_scratch_status_word_is_cleared_between_calls():
    a = Case(3, 0.05, 300.0, 13)
    NL_bad = a.NL.clone()
    j = int(NL_bad[0, 0].item())                      # drop atom 0 from the row of its first neighbour
    row = NL_bad[:, j].clone()
    nn_j = int(a.NN[j].item())
    pos = int((row[:nn_j] == 0).nonzero()[0].item())
    NN_bad = a.NN.clone()
    row[pos:nn_j - 1] = row[pos + 1:nn_j].clone()
    NL_bad[:, j] = row
    NN_bad[j] = nn_j - 1
    n = a.n
    f = torch.zeros((3, n), dtype=torch.float64, device=DEV)
    st = torch.zeros(1, dtype=torch.int32, device=DEV)
    md.md_tersoff_force_static(n, K, NN_bad, NL_bad, a.g.x, a.g.y, a.g.z, a.g.box, mi.TERSOFF_SI_C, f=f, status=st)
    torch.cuda.synchronize()
    assert int(st.item()) == 2 and bool(torch.isnan(f[:, 0]).all())
    assert int(torch.isnan(f).any(dim=0).sum().item()) == 1          # only the atom whose partner lost it
    a.check(*a.static_call())                         # the next call starts from a clean status word
    # a row count beyond max_neighbors is clamped and reported
    NN_long, NL_long = a.NN.clone(), a.NL.clone()
    NL_long[int(a.NN[5].item()):, 5] = NL_long[0, 5]  # valid indices in the slots the clamped row will read
    NN_long[5] = K + 3
    md.md_tersoff_force_static(n, K, NN_long, NL_long, a.g.x, a.g.y, a.g.z, a.g.box, mi.TERSOFF_SI_C, status=st)
    torch.cuda.synchronize()
    assert int(st.item()) & 1
    # an index outside [0, n) ends its row there and is reported; nothing is read out of bounds
    NL_oob = a.NL.clone()
    NL_oob[1, 7] = n + 100
    pe = torch.zeros(n, dtype=torch.float64, device=DEV)
    md.md_tersoff_force_static(n, K, a.NN, NL_oob, a.g.x, a.g.y, a.g.z, a.g.box, mi.TERSOFF_SI_C, pe=pe, status=st)
    torch.cuda.synchronize()
    assert int(st.item()) & 2 and bool(torch.isfinite(pe).all())


def test_static_scratch_limits_and_argument_errors():
    a = Case(2, 0.05, 300.0, 14)
    g = a.g
    with pytest.raises(md.MDError) as e:              # one pair more than the array holds: refused, nothing enqueued
        md.md_tersoff_force_static(md.MD_STATIC_MAX_PAIRS // K + 1, K, a.NN, a.NL, g.x, g.y, g.z, g.box,
                                   mi.TERSOFF_SI_C)
    assert e.value.code == md.MD_ERR_STATIC_CAPACITY
    for bad in (dict(n=-1), dict(k=0), dict(k=md.MD_MAX_NEIGHBORS + 1)):
        with pytest.raises(md.MDError) as e:
            md.md_tersoff_force_static(bad.get("n", a.n), bad.get("k", K), a.NN, a.NL, g.x, g.y, g.z, g.box,
                                       mi.TERSOFF_SI_C)
        assert e.value.code == md.MD_ERR_ARG
    with pytest.raises(md.MDError):
        md.md_tersoff_force_static(a.n, K, None, a.NL, g.x, g.y, g.z, g.box, mi.TERSOFF_SI_C)
    st = torch.full((1,), -1, dtype=torch.int32, device=DEV)
    md.md_tersoff_force_static(0, K, None, None, None, None, None, g.box, mi.TERSOFF_SI_C, status=st)   # empty input
    torch.cuda.synchronize()
    assert int(st.item()) == 0
    a.check(*a.static_call())
    big = Case(16, 0.05, 300.0, 15)                   # 32768 atoms x 16 slots: exactly the size of the array
    assert big.n * K == md.MD_STATIC_MAX_PAIRS
    big.check(*big.static_call())
    a.check(*a.static_call())
