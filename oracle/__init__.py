"""ctypes front end of the CPU oracle (oracle/md_oracle.cpp).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports the CUDA package.
All arrays are host numpy float64 / int32; vectors are SoA [3][n], virial [9][n].
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "md_oracle.cpp")
_LIB = os.path.join(_DIR, "libmd_oracle.so")
_lib = None

TERSOFF, SW = 0, 1
_TERSOFF_ORDER = ("A", "B", "lam", "mu", "beta", "n", "c", "d", "h", "R", "S")
_SW_ORDER = ("epsilon", "sigma", "a", "lam", "gamma", "A", "B", "p", "q", "cos0")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no fused multiply-add contraction: reading A7)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC",
                               "-o", _LIB, _SRC])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_atom_energy.restype = C.c_double
    return _lib


def _p(a, t=C.c_double):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def pack_params(potential, params) -> np.ndarray:
    order = _TERSOFF_ORDER if potential in (TERSOFF, "tersoff") else _SW_ORDER
    return np.array([float(params[k]) for k in order], dtype=np.float64)


def pot_id(potential) -> int:
    return {"tersoff": TERSOFF, "sw": SW, TERSOFF: TERSOFF, SW: SW}[potential]


def neighbors(x, y, z, box, r_list, K, method="auto"):
    """(NN[n], NL[n][K]) int32, rows sorted by j.  method: 'brute' | 'cell' | 'auto'."""
    x, y, z, box = _f64(x), _f64(y), _f64(z), _f64(box)
    n = x.size
    NN = np.zeros(n, dtype=np.int32)
    NL = np.full((n, K), -1, dtype=np.int32)
    if method == "auto":
        method = "brute" if n <= 4096 else "cell"
    fn = lib().oracle_neighbors_brute if method == "brute" else lib().oracle_neighbors_cell
    rc = fn(C.c_int64(n), _p(x), _p(y), _p(z), _p(box), C.c_double(r_list), C.c_int(K),
            _p(NN, C.c_int32), _p(NL, C.c_int32))
    if rc < 0:
        raise RuntimeError(f"oracle neighbour list overflow (K={K})")
    return NN, NL


def evaluate(potential, params, x, y, z, box, NN, NL, v=None, precision="f64",
             want=("pe", "f", "f_pair", "virial", "heat")):
    """One evaluation.  Returns dict with pe[n], f[3][n] (conventional, Alg. 1),
    f_pair[3][n] (sum_j P_ij - P_ji), virial[9][n], heat[3][n], P[n][K][3]."""
    x, y, z, box = _f64(x), _f64(y), _f64(z), _f64(box)
    n = x.size
    K = NL.shape[1]
    par = pack_params(potential, params)
    out = {}
    def alloc(name, shape):
        if name in want:
            out[name] = np.zeros(shape, dtype=np.float64)
            return out[name]
        return None
    pe = alloc("pe", n); f = alloc("f", (3, n)); fp = alloc("f_pair", (3, n))
    W = alloc("virial", (9, n)); J = alloc("heat", (3, n)) if v is not None else None
    P = alloc("P", (n, K, 3))
    vx = vy = vz = None
    if v is not None:
        vx, vy, vz = (_f64(c) for c in v)
    rc = lib().oracle_evaluate(C.c_int(pot_id(potential)), _p(par), C.c_int(1 if precision == "f80" else 0),
                               C.c_int64(n), _p(x), _p(y), _p(z), _p(vx), _p(vy), _p(vz), _p(box),
                               _p(np.ascontiguousarray(NN, dtype=np.int32), C.c_int32),
                               _p(np.ascontiguousarray(NL, dtype=np.int32), C.c_int32), C.c_int(K),
                               _p(pe), _p(f), _p(fp), _p(W), _p(J), _p(P))
    if rc != 0:
        raise RuntimeError(f"oracle_evaluate failed rc={rc}")
    return out


def evaluate_threads(potential, params, x, y, z, box, NN, NL, nthreads):
    """pe[n] and the conventional forces f[3][n] with the atoms split into `nthreads` contiguous ranges, one
    thread each (ctypes releases the GIL), each scattering into its own force buffer (Algorithm 1 writes to j
    and k: PAPER.md:157-161); the buffers are added afterwards.  Timing entry for bench.py's all-core
    cpu_baseline: the per-atom functions are the single-thread oracle's, unchanged."""
    from concurrent.futures import ThreadPoolExecutor
    x, y, z, box = _f64(x), _f64(y), _f64(z), _f64(box)
    n, K = x.size, NL.shape[1]
    par = pack_params(potential, params)
    NN = np.ascontiguousarray(NN, dtype=np.int32)
    NL = np.ascontiguousarray(NL, dtype=np.int32)
    pe = np.zeros(n)
    bounds = np.linspace(0, n, nthreads + 1).astype(np.int64)
    bufs = [np.zeros((3, n)) for _ in range(nthreads)]
    fn = lib().oracle_evaluate_range

    def work(t):
        rc = fn(C.c_int(pot_id(potential)), _p(par), C.c_int64(n), _p(x), _p(y), _p(z), _p(box),
                _p(NN, C.c_int32), _p(NL, C.c_int32), C.c_int(K), C.c_int64(int(bounds[t])),
                C.c_int64(int(bounds[t + 1])), _p(pe), _p(bufs[t]))
        if rc != 0:
            raise RuntimeError(f"oracle_evaluate_range failed rc={rc}")
    with ThreadPoolExecutor(nthreads) as ex:
        list(ex.map(work, range(nthreads)))
    f = bufs[0]
    for b in bufs[1:]:
        f += b
    return pe, f


def nve_run_threads(potential, params, state, nsteps, dt, rebuild_every, r_list, K, nthreads, f):
    """The NVE loop of nve_run with the force evaluation on `nthreads` threads (list build and integrator stay
    single-threaded).  `f` must hold the forces of the incoming state.  Returns the final forces."""
    NN = NL = None
    for s in range(nsteps):
        vv_kick_drift(state["x"], state["y"], state["z"], state["vx"], state["vy"], state["vz"], f,
                      state["mass"], dt, state["box"])
        if s % rebuild_every == 0 or NN is None:
            NN, NL = neighbors(state["x"], state["y"], state["z"], state["box"], r_list, K, method="cell")
        _, f = evaluate_threads(potential, params, state["x"], state["y"], state["z"], state["box"], NN, NL, nthreads)
        vv_kick(state["vx"], state["vy"], state["vz"], f, state["mass"], dt)
    return f


def pack_multi(elements, chi) -> np.ndarray:
    """Parameter blob of the multi-element Tersoff form: elements = list of per-element dicts (keys as
    TERSOFF_SI_C), chi = nt x nt matrix (chi_ii = 1)."""
    nt = len(elements)
    blob = [float(nt)]
    for e in elements:
        blob += [float(e[k]) for k in _TERSOFF_ORDER]
    blob += [float(v) for v in np.asarray(chi, dtype=np.float64).reshape(-1)]
    return np.array(blob, dtype=np.float64)


def evaluate_multi(elements, chi, types, x, y, z, box, NN, NL, v=None, precision="f64",
                   want=("pe", "f", "f_pair", "virial", "heat")):
    """evaluate() for the multi-element Tersoff form; types[n] int32 in 0..nt-1."""
    x, y, z, box = _f64(x), _f64(y), _f64(z), _f64(box)
    n, K = x.size, NL.shape[1]
    par = pack_multi(elements, chi)
    types = np.ascontiguousarray(types, dtype=np.int32)
    out = {}

    def alloc(name, shape):
        if name in want:
            out[name] = np.zeros(shape, dtype=np.float64)
            return out[name]
        return None
    pe = alloc("pe", n); f = alloc("f", (3, n)); fp = alloc("f_pair", (3, n))
    W = alloc("virial", (9, n)); J = alloc("heat", (3, n)) if v is not None else None
    P = alloc("P", (n, K, 3))
    vx = vy = vz = None
    if v is not None:
        vx, vy, vz = (_f64(c) for c in v)
    rc = lib().oracle_evaluate_multi(_p(par), C.c_int(1 if precision == "f80" else 0), C.c_int64(n),
                                     _p(x), _p(y), _p(z), _p(vx), _p(vy), _p(vz), _p(box), _p(types, C.c_int32),
                                     _p(np.ascontiguousarray(NN, dtype=np.int32), C.c_int32),
                                     _p(np.ascontiguousarray(NL, dtype=np.int32), C.c_int32), C.c_int(K),
                                     _p(pe), _p(f), _p(fp), _p(W), _p(J), _p(P))
    if rc != 0:
        raise RuntimeError(f"oracle_evaluate_multi failed rc={rc}")
    return out


def nve_heat_run(potential, params, state, nsteps, dt, rebuild_every, r_list, K, sample_every, f=None):
    """NVE with the total heat current sampled every `sample_every` steps (Green-Kubo workload).
    Returns dict(f, J_pot[ns][3], J_kin[ns][3])."""
    n = state["x"].size
    par = pack_params(potential, params)
    f_valid = 0 if f is None else 1
    f = np.zeros((3, n)) if f is None else np.ascontiguousarray(f, dtype=np.float64)
    ns = nsteps // sample_every
    Jp, Jk = np.zeros((max(ns, 1), 3)), np.zeros((max(ns, 1), 3))
    rc = lib().oracle_nve_heat_run(C.c_int(pot_id(potential)), _p(par), C.c_int64(n), _p(state["x"]), _p(state["y"]),
                                   _p(state["z"]), _p(state["vx"]), _p(state["vy"]), _p(state["vz"]),
                                   _p(_f64(state["box"])), C.c_double(state["mass"]), C.c_double(dt), C.c_int(nsteps),
                                   C.c_int(rebuild_every), C.c_double(r_list), C.c_int(K), _p(f), C.c_int(f_valid),
                                   C.c_int(sample_every), _p(Jp), _p(Jk))
    if rc != 0:
        raise RuntimeError(f"oracle_nve_heat_run failed rc={rc}")
    return {"f": f, "J_pot": Jp[:ns], "J_kin": Jk[:ns]}


def npt_run(potential, params, state, nsteps, dt, rebuild_every, r_list, K, berendsen, f=None):
    """Berendsen NPT (reading A18); `state` as in nve_run, its box is updated in place.
    berendsen = dict(T0, tau_T, P0, tau_P, beta) in K, fs, eV/A^3, fs, A^3/eV.
    Returns dict(f, T_trace, P_trace) with the values measured before each step's scaling."""
    n = state["x"].size
    par = pack_params(potential, params)
    f_valid = 0 if f is None else 1
    f = np.zeros((3, n)) if f is None else np.ascontiguousarray(f, dtype=np.float64)
    Tt, Pt = np.zeros(max(nsteps, 1)), np.zeros(max(nsteps, 1))
    b = berendsen
    rc = lib().oracle_npt_run(C.c_int(pot_id(potential)), _p(par), C.c_int64(n), _p(state["x"]), _p(state["y"]),
                              _p(state["z"]), _p(state["vx"]), _p(state["vy"]), _p(state["vz"]), _p(state["box"]),
                              C.c_double(state["mass"]), C.c_double(dt), C.c_int(nsteps), C.c_int(rebuild_every),
                              C.c_double(r_list), C.c_int(K), _p(f), C.c_int(f_valid), C.c_double(b["T0"]),
                              C.c_double(b["tau_T"]), C.c_double(b["P0"]), C.c_double(b["tau_P"]),
                              C.c_double(b["beta"]), _p(Tt), _p(Pt))
    if rc != 0:
        raise RuntimeError(f"oracle_npt_run failed rc={rc}")
    return {"f": f, "T_trace": Tt[:nsteps], "P_trace": Pt[:nsteps]}


def atom_energy_multi(elements, chi, ti, tj, rvecs) -> float:
    r = np.ascontiguousarray(rvecs, dtype=np.float64)
    rx, ry, rz = (np.ascontiguousarray(r[:, a]) for a in range(3))
    tj = np.ascontiguousarray(tj, dtype=np.int32)
    lib().oracle_atom_energy_multi.restype = C.c_double
    return lib().oracle_atom_energy_multi(_p(pack_multi(elements, chi)), C.c_int(ti), C.c_int(r.shape[0]),
                                          _p(tj, C.c_int32), _p(rx), _p(ry), _p(rz))


def atom_energy(potential, params, rvecs) -> float:
    """U_i from explicit relative vectors r_ij (shape [M][3]), long double inside."""
    r = np.ascontiguousarray(rvecs, dtype=np.float64)
    rx, ry, rz = (np.ascontiguousarray(r[:, a]) for a in range(3))
    par = pack_params(potential, params)
    return lib().oracle_atom_energy(C.c_int(pot_id(potential)), _p(par), C.c_int(r.shape[0]),
                                    _p(rx), _p(ry), _p(rz))


def vv_kick_drift(x, y, z, vx, vy, vz, f, mass, dt, box):
    lib().oracle_vv_kick_drift(C.c_int64(x.size), _p(x), _p(y), _p(z), _p(vx), _p(vy), _p(vz),
                               _p(np.ascontiguousarray(f)), C.c_double(mass), C.c_double(dt), _p(_f64(box)))


def vv_kick(vx, vy, vz, f, mass, dt):
    lib().oracle_vv_kick(C.c_int64(vx.size), _p(vx), _p(vy), _p(vz), _p(np.ascontiguousarray(f)),
                         C.c_double(mass), C.c_double(dt))


def nve_run(potential, params, state, nsteps, dt, rebuild_every, r_list, K, f=None):
    """Advance `state` (dict with x,y,z,vx,vy,vz,box,mass; arrays modified in place) by nsteps.
    Returns dict(f=[3][n], pe=[n], pe_trace=[nsteps])."""
    n = state["x"].size
    par = pack_params(potential, params)
    f_valid = 0 if f is None else 1
    f = np.zeros((3, n)) if f is None else np.ascontiguousarray(f, dtype=np.float64)
    pe = np.zeros(n); trace = np.zeros(max(nsteps, 1))
    rc = lib().oracle_nve_run(C.c_int(pot_id(potential)), _p(par), C.c_int64(n),
                              _p(state["x"]), _p(state["y"]), _p(state["z"]),
                              _p(state["vx"]), _p(state["vy"]), _p(state["vz"]), _p(_f64(state["box"])),
                              C.c_double(state["mass"]), C.c_double(dt), C.c_int(nsteps), C.c_int(rebuild_every),
                              C.c_double(r_list), C.c_int(K), _p(f), C.c_int(f_valid), _p(pe), _p(trace))
    if rc != 0:
        raise RuntimeError(f"oracle_nve_run failed rc={rc}")
    return {"f": f, "pe": pe, "pe_trace": trace[:nsteps]}
