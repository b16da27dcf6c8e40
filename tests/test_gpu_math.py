"""Accuracy of the pair kernels' FP64 device functions (csrc/fastmath.cuh) against 80-bit references,
on the argument ranges the potentials produce.  The force tolerance is 1e-10 and the energy tolerance
1e-12 (A11); these functions must sit far below both."""
import numpy as np
import pytest
import torch

import paper_1610_03343_b200 as md

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
LD = np.longdouble


def run(fn, a):
    inp = torch.from_numpy(np.ascontiguousarray(a)).to(DEV)
    out = torch.empty_like(inp)
    md.md_math_probe(fn, inp.numel(), inp, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def test_long_double_is_wider_than_double():
    assert np.finfo(LD).eps < 1e-18


def test_exp_relative_error():
    rng = np.random.default_rng(1)
    a = np.concatenate([rng.uniform(-80.0, 8.0, 400000), rng.uniform(-700.0, 700.0, 100000),
                        np.linspace(-9.0, -2.0, 100001), [0.0, -0.0, 1e-300, -1e-300, 1.0, -1.0]])
    got = run("exp", a)
    ref = np.exp(a.astype(LD))
    rel = np.abs((got.astype(LD) - ref) / ref).astype(np.float64)
    assert rel.max() < 4e-16, rel.max()
    assert run("exp", np.array([0.0]))[0] == 1.0
    sat = run("exp", np.array([-1e4, 1e4]))                  # saturates, no inf / nan / zero
    assert np.isfinite(sat).all() and sat[0] < 1e-290 and sat[1] > 1e290


def test_log_absolute_error():
    rng = np.random.default_rng(2)
    a = np.concatenate([np.exp(rng.uniform(-100.0, 20.0, 400000)), rng.uniform(1.0, 3.0, 200000),
                        1.0 + np.exp(rng.uniform(-40.0, 0.0, 100000)), rng.uniform(0.4, 1.0, 100000),
                        [1.0, 2.0, 0.5, 1.0 + 2.0 ** -52, 1e-300, 1e300]])
    got = run("log", a)
    ref = np.log(a.astype(LD))
    err = (np.abs(got.astype(LD) - ref) / np.maximum(1.0, np.abs(ref))).astype(np.float64)
    assert err.max() < 4e-16, err.max()


def test_rcp_rsqrt_relative_error():
    rng = np.random.default_rng(3)
    a = np.concatenate([np.exp(rng.uniform(-60.0, 60.0, 300000)), rng.uniform(1.0, 16.0, 300000)])
    for fn, ref in (("rcp", 1 / a.astype(LD)), ("rsqrt", 1 / np.sqrt(a.astype(LD)))):
        got = run(fn, a)
        rel = np.abs((got.astype(LD) - ref) / ref).astype(np.float64)
        assert rel.max() < 4e-16, (fn, rel.max())
    got = run("rcp", -a)
    assert (got < 0).all()


def test_sincos_on_zero_to_pi():
    rng = np.random.default_rng(4)
    a = np.concatenate([rng.uniform(0.0, np.pi, 400000), [0.0, np.pi, np.pi / 2, np.pi / 4, 3 * np.pi / 4]])
    s, c = run("sin", a), run("cos", a)
    assert np.abs(s.astype(LD) - np.sin(a.astype(LD))).max() < 3e-16
    assert np.abs(c.astype(LD) - np.cos(a.astype(LD))).max() < 3e-16
