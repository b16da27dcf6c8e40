"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

This module holds NONE of the method's arithmetic (no potential, no neighbour
search, no integrator): only the silicon-crystal workload recipe of
PAPER.md:355 ("silicon crystal ... cubic domain ... 300 K") as restated in
SURVEY.md section 8(d) and DESIGN.md "Input recipe".  It imports neither
`oracle/` nor the CUDA package; both consume the host arrays it returns.

Recipe
------
* diamond lattice, conventional cell a = 5.43 A, 8-atom basis, cells ordered
  (ix, iy, iz) with iz fastest and the basis index fastest of all;
* Gaussian displacements (sigma_disp) and Maxwell-Boltzmann velocities
  (sigma_v = sqrt(kB T / m)) from a counter-based generator: for atom i,
  component a, stream s: two SplitMix64 outputs of the key
  (seed, s, 3 i + a) -> Box-Muller -> one normal deviate.  Order independent.
* positions wrapped into [0, L); mean velocity removed.
"""
from __future__ import annotations

import numpy as np

# --- unit constants (units: Angstrom, fs, amu, eV) -------------------------
KB_EV_PER_K = 8.617333262e-5          # Boltzmann constant, eV/K (CODATA 2018)
# acceleration [A/fs^2] = KAPPA * force [eV/A] / mass [amu]
# KAPPA = e / (u * 1e10 * 1e... ) = 1.602176634e-19 / 1.66053906660e-27 * 1e-10 (m->A: 1e20, s->fs: 1e-30)
KAPPA = 9.648533215665e-3
SI_MASS_AMU = 28.0855
C_MASS_AMU = 12.011
SI_LATTICE_A = 5.43

_BASIS = np.array(
    [[0.0, 0.0, 0.0], [0.0, 0.5, 0.5], [0.5, 0.0, 0.5], [0.5, 0.5, 0.0],
     [0.25, 0.25, 0.25], [0.25, 0.75, 0.75], [0.75, 0.25, 0.75], [0.75, 0.75, 0.25]],
    dtype=np.float64)

STREAM_DISP = 1
STREAM_VEL = 2
BASE_SEED = 1610033430

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(z: np.ndarray) -> np.ndarray:
    """One SplitMix64 output step applied elementwise to uint64 states."""
    with np.errstate(over="ignore"):
        z = (z + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


def normal_deviates(seed: int, stream: int, count: int) -> np.ndarray:
    """`count` independent N(0,1) deviates; deviate c depends only on (seed, stream, c)."""
    c = np.arange(count, dtype=np.uint64)
    with np.errstate(over="ignore"):
        key = _splitmix64(np.uint64(seed) + np.zeros(count, dtype=np.uint64))
        key = _splitmix64(key ^ (np.uint64(stream) * np.uint64(0xD1B54A32D192ED03)))
        s0 = _splitmix64(key ^ (c * np.uint64(2)))
        s1 = _splitmix64(key ^ (c * np.uint64(2) + np.uint64(1)))
    # 53-bit uniforms; u1 in (0,1], u2 in [0,1)
    u1 = ((s0 >> np.uint64(11)).astype(np.float64) + 1.0) * (1.0 / 9007199254740992.0)
    u2 = (s1 >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def diamond_lattice(ncell: int, a: float = SI_LATTICE_A):
    """Perfect diamond lattice, N = 8 ncell^3 atoms, SoA float64 (x, y, z), box edge L."""
    ix, iy, iz, ib = np.meshgrid(np.arange(ncell), np.arange(ncell), np.arange(ncell),
                                 np.arange(8), indexing="ij")
    ix = ix.reshape(-1); iy = iy.reshape(-1); iz = iz.reshape(-1); ib = ib.reshape(-1)
    x = (ix + _BASIS[ib, 0]) * a
    y = (iy + _BASIS[ib, 1]) * a
    z = (iz + _BASIS[ib, 2]) * a
    return x, y, z, ncell * a


def wrap(x: np.ndarray, L: float) -> np.ndarray:
    x = x - L * np.floor(x / L)
    x[x >= L] = 0.0
    x[x < 0.0] = 0.0
    return x


def silicon_crystal(ncell: int, sigma_disp: float, temperature: float, seed: int,
                    a: float = SI_LATTICE_A, mass: float = SI_MASS_AMU) -> dict:
    """Displaced diamond crystal with thermal velocities (dict of host float64 arrays)."""
    x, y, z, L = diamond_lattice(ncell, a)
    n = x.size
    if sigma_disp > 0.0:
        d = normal_deviates(seed, STREAM_DISP, 3 * n).reshape(n, 3)
        x = x + sigma_disp * d[:, 0]
        y = y + sigma_disp * d[:, 1]
        z = z + sigma_disp * d[:, 2]
    x = wrap(x, L); y = wrap(y, L); z = wrap(z, L)
    sv = np.sqrt(KB_EV_PER_K * temperature / mass * KAPPA) if temperature > 0 else 0.0
    g = normal_deviates(seed, STREAM_VEL, 3 * n).reshape(n, 3) * sv
    g = g - g.mean(axis=0, keepdims=True)
    return {
        "n": n, "box": np.array([L, L, L], dtype=np.float64), "mass": mass,
        "x": np.ascontiguousarray(x), "y": np.ascontiguousarray(y), "z": np.ascontiguousarray(z),
        "vx": np.ascontiguousarray(g[:, 0]), "vy": np.ascontiguousarray(g[:, 1]),
        "vz": np.ascontiguousarray(g[:, 2]),
    }


def zincblende_crystal(ncell: int, a: float, sigma_disp: float, temperature: float, seed: int,
                       masses=(SI_MASS_AMU, C_MASS_AMU)) -> dict:
    """Zinc-blende AB crystal (the diamond sites of `diamond_lattice`: basis 0-3 = element 0, basis 4-7 =
    element 1), seeded displacements and per-element Maxwell-Boltzmann velocities; `types` int32 [n]."""
    x, y, z, L = diamond_lattice(ncell, a)
    n = x.size
    types = ((np.arange(n) % 8) >= 4).astype(np.int32)
    if sigma_disp > 0.0:
        d = normal_deviates(seed, STREAM_DISP, 3 * n).reshape(n, 3)
        x = x + sigma_disp * d[:, 0]; y = y + sigma_disp * d[:, 1]; z = z + sigma_disp * d[:, 2]
    x = wrap(x, L); y = wrap(y, L); z = wrap(z, L)
    m = np.asarray(masses, dtype=np.float64)[types]
    sv = np.sqrt(KB_EV_PER_K * temperature / m * KAPPA) if temperature > 0 else np.zeros(n)
    g = normal_deviates(seed, STREAM_VEL, 3 * n).reshape(n, 3) * sv[:, None]
    g = g - (g * m[:, None]).sum(axis=0, keepdims=True) / m.sum()       # zero total momentum
    return {"n": n, "box": np.array([L, L, L], dtype=np.float64), "types": types, "mass": m,
            "x": np.ascontiguousarray(x), "y": np.ascontiguousarray(y), "z": np.ascontiguousarray(z),
            "vx": np.ascontiguousarray(g[:, 0]), "vy": np.ascontiguousarray(g[:, 1]),
            "vz": np.ascontiguousarray(g[:, 2])}


# --- potential parameter sets (BASELINE.json configs) -----------------------
TERSOFF_SI_C = dict(A=1830.8, B=471.18, lam=2.4799, mu=1.7322, beta=1.1e-6, n=0.78734,
                    c=100390.0, d=16.217, h=-0.59825, R=2.7, S=3.0)
SW_SI = dict(epsilon=2.1683, sigma=2.0951, a=1.80, lam=21.0, gamma=1.20,
             A=7.049556277, B=0.6022245584, p=4.0, q=0.0, cos0=-1.0 / 3.0)

# Tersoff's multicomponent parameter sets (J. Tersoff, Phys. Rev. B 39, 5566 (1989), Table I): carbon and
# silicon (the silicon column is the Si(C) set above), chi_Si-C = 0.9776; element order: 0 = Si, 1 = C.
TERSOFF_C = dict(A=1393.6, B=346.74, lam=3.4879, mu=2.2119, beta=1.5724e-7, n=0.72751,
                 c=38049.0, d=4.3484, h=-0.57058, R=1.8, S=2.1)
TERSOFF_SIC_ELEMENTS = [TERSOFF_SI_C, TERSOFF_C]
TERSOFF_SIC_CHI = [[1.0, 0.9776], [0.9776, 1.0]]
SIC_LATTICE_A = 4.32

SKIN = 0.5
# BASELINE.json configs 1..5 (index 0..4).  r_list = r_force + SKIN.
CONFIGS = [
    dict(name="cfg1_tersoff_512", potential="tersoff", ncell=4, sigma=0.05, T=300.0,
         steps=0, dt=1.0, rebuild_every=10, max_neighbors=16),
    dict(name="cfg2_tersoff_512k", potential="tersoff", ncell=40, sigma=0.05, T=300.0,
         steps=1000, dt=1.0, rebuild_every=10, max_neighbors=16),
    dict(name="cfg3_sw_512k", potential="sw", ncell=40, sigma=0.05, T=300.0,
         steps=1000, dt=1.0, rebuild_every=10, max_neighbors=32),
    dict(name="cfg4_tersoff_8M", potential="tersoff", ncell=100, sigma=0.05, T=300.0,
         steps=100, dt=1.0, rebuild_every=10, max_neighbors=16),
    dict(name="cfg5_tersoff_512k_hot", potential="tersoff", ncell=40, sigma=0.15, T=1500.0,
         steps=200, dt=0.5, rebuild_every=10, max_neighbors=16),
]


def r_force(potential: str) -> float:
    if potential == "tersoff":
        return TERSOFF_SI_C["S"]
    return SW_SI["a"] * SW_SI["sigma"]


def r_list(potential: str) -> float:
    return r_force(potential) + SKIN


def make_config(index: int, ncell: int | None = None) -> dict:
    """Inputs of BASELINE.json config `index` (0-based); `ncell` overrides the size
    (same recipe, same seed) for reduced parity cases."""
    c = dict(CONFIGS[index])
    if ncell is not None:
        c["ncell"] = ncell
    s = silicon_crystal(c["ncell"], c["sigma"], c["T"], BASE_SEED + index)
    c.update(s)
    c["r_list"] = r_list(c["potential"])
    c["params"] = dict(TERSOFF_SI_C if c["potential"] == "tersoff" else SW_SI)
    return c
