"""Thin ctypes binding of include/md.h: argument marshalling only.

Every step of the path runs in the CUDA kernels of libmd_b200.so; there is no CPU fallback and
nothing here imports `oracle/`.  Device arrays are anything with a `.data_ptr()` (torch tensors)
or plain integer addresses; PyTorch is only used by callers for device memory and streams.
"""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

MD_OK = 0
MD_ERR_ARG, MD_ERR_ALLOC, MD_ERR_BOX_TOO_SMALL, MD_ERR_NEIGHBOR_OVERFLOW = -1, -2, -3, -4
MD_ERR_CUDA, MD_ERR_NO_LIST, MD_ERR_LIST_ASYMMETRIC = -5, -6, -7
MD_ERR_STATIC_CAPACITY = -8
MD_FP64, MD_FP32 = 0, 1
MD_TERSOFF, MD_SW = 0, 1
MD_MAX_NEIGHBORS = 64
MD_STATIC_MAX_PAIRS = 524288

_ERR = {-1: "MD_ERR_ARG", -2: "MD_ERR_ALLOC", -3: "MD_ERR_BOX_TOO_SMALL", -4: "MD_ERR_NEIGHBOR_OVERFLOW",
        -5: "MD_ERR_CUDA", -6: "MD_ERR_NO_LIST", -7: "MD_ERR_LIST_ASYMMETRIC", -8: "MD_ERR_STATIC_CAPACITY"}


class MDError(RuntimeError):
    def __init__(self, code, where):
        super().__init__(f"{where}: {_ERR.get(code, code)}")
        self.code = code


class md_tersoff_params(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("A", "B", "lambda_", "mu", "beta", "n", "c", "d", "h", "R", "S")]


class md_tersoff_multi_params(C.Structure):
    _fields_ = [("ntypes", C.c_int), ("elem", md_tersoff_params * 4), ("chi", (C.c_double * 4) * 4)]


class md_sw_params(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("epsilon", "sigma", "a", "lambda_", "gamma", "A", "B", "p", "q", "cos0")]


EXPORTS = ("md_version", "md_neighbors_create", "md_neighbors_destroy", "md_neighbors_status",
           "md_neighbors_export", "md_neighbors_import", "md_build_neighbors", "md_tersoff_force",
           "md_sw_force", "md_velocity_verlet_step", "md_nve_run", "md_nve_run_host", "md_probe_fp64_peak",
           "md_profile_enable", "md_profile_read", "md_math_probe", "md_neighbors_row_stats", "md_pair_counts",
           "md_tersoff_multi_force", "md_tersoff_force_literal", "md_npt_run", "md_nve_heat_run",
           "md_tersoff_force_static")

_lib = None


def lib_path() -> str:
    return _build.LIB


def load():
    """Load libmd_b200.so (building it with nvcc if the sources are newer).  Fails loudly."""
    global _lib
    if _lib is None:
        path = _build.build()
        if not os.path.exists(path):
            raise ImportError("libmd_b200.so is missing and could not be built: the CUDA extension is required")
        _lib = C.CDLL(path)
        _lib.md_version.restype = C.c_char_p
        for name in EXPORTS:
            getattr(_lib, name)          # AttributeError if a declared symbol is not exported
    return _lib


def _ptr(a):
    if a is None:
        return C.c_void_p(0)
    if hasattr(a, "data_ptr"):
        return C.c_void_p(a.data_ptr())
    if hasattr(a, "ctypes"):                       # numpy host array (HOST arguments only)
        return C.c_void_p(a.ctypes.data)
    return C.c_void_p(int(a))


def _box(box):
    return (C.c_double * 3)(*[float(b) for b in box])


def _stream(stream):
    if stream is None:
        return C.c_void_p(0)
    return C.c_void_p(getattr(stream, "cuda_stream", stream))


def _check(rc, where):
    if rc != MD_OK:
        raise MDError(rc, where)


def tersoff_params(p) -> md_tersoff_params:
    if isinstance(p, md_tersoff_params):
        return p
    return md_tersoff_params(p["A"], p["B"], p["lam"], p["mu"], p["beta"], p["n"], p["c"], p["d"], p["h"],
                             p["R"], p["S"])


def sw_params(p) -> md_sw_params:
    if isinstance(p, md_sw_params):
        return p
    return md_sw_params(p["epsilon"], p["sigma"], p["a"], p["lam"], p["gamma"], p["A"], p["B"], p["p"], p["q"],
                        p["cos0"])


def md_version() -> str:
    return load().md_version().decode()


class Neighbors:
    """Owner of an `md_neighbors*` handle."""

    def __init__(self, n_atoms: int, max_neighbors: int):
        self._h = C.c_void_p(0)
        self.n_atoms, self.max_neighbors = int(n_atoms), int(max_neighbors)
        _check(load().md_neighbors_create(C.byref(self._h), C.c_int64(n_atoms), C.c_int(max_neighbors)),
               "md_neighbors_create")

    def close(self):
        if self._h:
            load().md_neighbors_destroy(self._h)
            self._h = C.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def md_neighbors_create(n_atoms, max_neighbors) -> Neighbors:
    return Neighbors(n_atoms, max_neighbors)


def md_neighbors_destroy(nl: Neighbors):
    nl.close()


def md_neighbors_status(nl: Neighbors, stream=None, check=True) -> int:
    """Synchronises; returns the longest row of the last build.  Raises on a latched device error."""
    mx = C.c_int(0)
    rc = load().md_neighbors_status(nl._h, C.byref(mx), _stream(stream))
    if check:
        _check(rc, "md_neighbors_status")
        return mx.value
    return rc


def md_neighbors_export(nl, NN, NL, stream=None):
    _check(load().md_neighbors_export(nl._h, _ptr(NN), _ptr(NL), _stream(stream)), "md_neighbors_export")


def md_neighbors_import(nl, n, NN, NL, stream=None):
    _check(load().md_neighbors_import(nl._h, C.c_int64(n), _ptr(NN), _ptr(NL), _stream(stream)),
           "md_neighbors_import")


def md_build_neighbors(nl, n, x, y, z, box, r_list, stream=None):
    _check(load().md_build_neighbors(nl._h, C.c_int64(n), _ptr(x), _ptr(y), _ptr(z), _box(box),
                                     C.c_double(r_list), _stream(stream)), "md_build_neighbors")


def md_tersoff_force(nl, n, x, y, z, vx, vy, vz, box, params, precision=MD_FP64,
                     pe=None, f=None, virial=None, heat=None, stream=None):
    p = tersoff_params(params)
    _check(load().md_tersoff_force(nl._h, C.c_int64(n), _ptr(x), _ptr(y), _ptr(z), _ptr(vx), _ptr(vy), _ptr(vz),
                                   _box(box), C.byref(p), C.c_int(precision), _ptr(pe), _ptr(f), _ptr(virial),
                                   _ptr(heat), _stream(stream)), "md_tersoff_force")


def md_tersoff_force_literal(nl, n, x, y, z, vx, vy, vz, box, params, precision=MD_FP64,
                             pe=None, f=None, virial=None, heat=None, stream=None):
    """The paper's literal Algorithm 3 + Algorithm 2 (A/B against the stored-P design)."""
    p = tersoff_params(params)
    _check(load().md_tersoff_force_literal(nl._h, C.c_int64(n), _ptr(x), _ptr(y), _ptr(z), _ptr(vx), _ptr(vy),
                                           _ptr(vz), _box(box), C.byref(p), C.c_int(precision), _ptr(pe), _ptr(f),
                                           _ptr(virial), _ptr(heat), _stream(stream)), "md_tersoff_force_literal")


def md_tersoff_force_static(n, max_neighbors, NN, NL, x, y, z, box, params, pe=None, f=None, status=None, stream=None):
    """Tersoff U_i and F_i with the pair records in the library's fixed device array: no handle, no allocation.
    n * max_neighbors <= MD_STATIC_MAX_PAIRS; calls that overlap on one GPU race on the array (md.h)."""
    p = tersoff_params(params)
    _check(load().md_tersoff_force_static(C.c_int64(n), C.c_int(max_neighbors), _ptr(NN), _ptr(NL), _ptr(x), _ptr(y),
                                          _ptr(z), _box(box), C.byref(p), _ptr(pe), _ptr(f), _ptr(status),
                                          _stream(stream)), "md_tersoff_force_static")


def tersoff_multi_params(elements, chi) -> md_tersoff_multi_params:
    p = md_tersoff_multi_params()
    p.ntypes = len(elements)
    for t, e in enumerate(elements):
        p.elem[t] = tersoff_params(e)
        for u in range(len(elements)):
            p.chi[t][u] = float(chi[t][u])
    return p


def md_tersoff_multi_force(nl, n, x, y, z, vx, vy, vz, box, types, elements, chi, precision=MD_FP64,
                           pe=None, f=None, virial=None, heat=None, stream=None):
    p = tersoff_multi_params(elements, chi)
    _check(load().md_tersoff_multi_force(nl._h, C.c_int64(n), _ptr(x), _ptr(y), _ptr(z), _ptr(vx), _ptr(vy),
                                         _ptr(vz), _box(box), _ptr(types), C.byref(p), C.c_int(precision),
                                         _ptr(pe), _ptr(f), _ptr(virial), _ptr(heat), _stream(stream)),
           "md_tersoff_multi_force")


def md_sw_force(nl, n, x, y, z, vx, vy, vz, box, params, precision=MD_FP64,
                pe=None, f=None, virial=None, heat=None, stream=None):
    p = sw_params(params)
    _check(load().md_sw_force(nl._h, C.c_int64(n), _ptr(x), _ptr(y), _ptr(z), _ptr(vx), _ptr(vy), _ptr(vz),
                              _box(box), C.byref(p), C.c_int(precision), _ptr(pe), _ptr(f), _ptr(virial),
                              _ptr(heat), _stream(stream)), "md_sw_force")


def md_velocity_verlet_step(phase, n, x, y, z, vx, vy, vz, f, mass_amu, dt_fs, box, stream=None):
    _check(load().md_velocity_verlet_step(C.c_int(phase), C.c_int64(n), _ptr(x), _ptr(y), _ptr(z), _ptr(vx),
                                          _ptr(vy), _ptr(vz), _ptr(f), C.c_double(mass_amu), C.c_double(dt_fs),
                                          _box(box), _stream(stream)), "md_velocity_verlet_step")


def _pot(potential, params):
    if potential in (MD_TERSOFF, "tersoff"):
        return MD_TERSOFF, tersoff_params(params)
    if potential in (MD_SW, "sw"):
        return MD_SW, sw_params(params)
    raise MDError(MD_ERR_ARG, "potential")


def md_neighbors_row_stats(nl):
    """(longest row, rows longer than 4) of the current list."""
    a, b = C.c_int(0), C.c_int(0)
    _check(load().md_neighbors_row_stats(nl._h, C.byref(a), C.byref(b)), "md_neighbors_row_stats")
    return a.value, b.value


def md_nve_run(nl, potential, params, n, x, y, z, vx, vy, vz, f, f_valid, pe, box, mass_amu, dt_fs,
               nsteps, rebuild_every, r_list, precision=MD_FP64, stream=None, first_step=0):
    pid, p = _pot(potential, params)
    _check(load().md_nve_run(nl._h, C.c_int(pid), C.byref(p), C.c_int(precision), C.c_int64(n),
                             _ptr(x), _ptr(y), _ptr(z), _ptr(vx), _ptr(vy), _ptr(vz), _ptr(f),
                             C.c_int(1 if f_valid else 0), _ptr(pe), _box(box), C.c_double(mass_amu),
                             C.c_double(dt_fs), C.c_int(first_step), C.c_int(nsteps), C.c_int(rebuild_every),
                             C.c_double(r_list), _stream(stream)), "md_nve_run")


class md_berendsen_params(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("T0", "tau_T", "P0", "tau_P", "beta")]


def md_npt_run(nl, potential, params, n, x, y, z, vx, vy, vz, f, f_valid, box, mass_amu, dt_fs, nsteps,
               rebuild_every, r_list, berendsen, precision=MD_FP64, stream=None, first_step=0):
    """Berendsen NPT.  `box` is a list of 3 floats and is UPDATED in place; returns (T_trace, P_trace) lists."""
    import ctypes
    pid, p = _pot(potential, params)
    b = md_berendsen_params(berendsen["T0"], berendsen["tau_T"], berendsen["P0"], berendsen["tau_P"], berendsen["beta"])
    cbox = _box(box)
    Tt = (ctypes.c_double * max(1, nsteps))()
    Pt = (ctypes.c_double * max(1, nsteps))()
    _check(load().md_npt_run(nl._h, C.c_int(pid), C.byref(p), C.c_int(precision), C.c_int64(n), _ptr(x), _ptr(y),
                             _ptr(z), _ptr(vx), _ptr(vy), _ptr(vz), _ptr(f), C.c_int(1 if f_valid else 0), cbox,
                             C.c_double(mass_amu), C.c_double(dt_fs), C.c_int(first_step), C.c_int(nsteps),
                             C.c_int(rebuild_every), C.c_double(r_list), C.byref(b), Tt, Pt, _stream(stream)),
           "md_npt_run")
    for a in range(3):
        box[a] = cbox[a]
    return list(Tt)[:nsteps], list(Pt)[:nsteps]


def md_nve_heat_run(nl, potential, params, n, x, y, z, vx, vy, vz, f, f_valid, box, mass_amu, dt_fs, nsteps,
                    rebuild_every, r_list, sample_every, precision=MD_FP64, stream=None, first_step=0):
    """NVE with the total heat current sampled every `sample_every` steps.  Returns (J_pot, J_kin) as lists of
    [Jx, Jy, Jz] per sample (eV A/fs)."""
    pid, p = _pot(potential, params)
    ns = nsteps // sample_every
    Jp = (C.c_double * max(1, 3 * ns))()
    Jk = (C.c_double * max(1, 3 * ns))()
    _check(load().md_nve_heat_run(nl._h, C.c_int(pid), C.byref(p), C.c_int(precision), C.c_int64(n), _ptr(x), _ptr(y),
                                  _ptr(z), _ptr(vx), _ptr(vy), _ptr(vz), _ptr(f), C.c_int(1 if f_valid else 0),
                                  _box(box), C.c_double(mass_amu), C.c_double(dt_fs), C.c_int(first_step),
                                  C.c_int(nsteps), C.c_int(rebuild_every), C.c_double(r_list), C.c_int(sample_every),
                                  Jp, Jk, _stream(stream)), "md_nve_heat_run")
    return ([[Jp[3 * k + a] for a in range(3)] for k in range(ns)],
            [[Jk[3 * k + a] for a in range(3)] for k in range(ns)])


def md_nve_run_host(nl, potential, params, n, x, y, z, vx, vy, vz, f, pe, box, mass_amu, dt_fs,
                    nsteps, rebuild_every, r_list, precision=MD_FP64, stream=None):
    """HOST buffers (numpy arrays or pinned torch CPU tensors), updated in place."""
    pid, p = _pot(potential, params)
    _check(load().md_nve_run_host(nl._h, C.c_int(pid), C.byref(p), C.c_int(precision), C.c_int64(n),
                                  _ptr(x), _ptr(y), _ptr(z), _ptr(vx), _ptr(vy), _ptr(vz), _ptr(f), _ptr(pe),
                                  _box(box), C.c_double(mass_amu), C.c_double(dt_fs), C.c_int(nsteps),
                                  C.c_int(rebuild_every), C.c_double(r_list), _stream(stream)), "md_nve_run_host")


def md_probe_fp64_peak(iters=20000, stream=None) -> float:
    t = C.c_double(0.0)
    _check(load().md_probe_fp64_peak(C.c_int(iters), C.byref(t), _stream(stream)), "md_probe_fp64_peak")
    return t.value


def md_pair_counts(nl, stream=None):
    """(listed directed pairs, in-range directed pairs, ordered in-range triplets) of the current list and the
    masks the last force call left.  Synchronises."""
    out = (C.c_int64 * 3)()
    _check(load().md_pair_counts(nl._h, out, _stream(stream)), "md_pair_counts")
    return int(out[0]), int(out[1]), int(out[2])


MATH_FN = {"exp": 0, "log": 1, "rcp": 2, "rsqrt": 3, "sin": 4, "cos": 5}


def md_math_probe(fn, n, inp, out, stream=None):
    """out[k] = fn(inp[k]) with the pair kernels' FP64 device functions (DEVICE buffers)."""
    _check(load().md_math_probe(C.c_int(MATH_FN[fn] if isinstance(fn, str) else fn), C.c_int64(n), _ptr(inp),
                                _ptr(out), _stream(stream)), "md_math_probe")


KINDS = ("build", "pair", "gather", "integrate")


def md_profile_enable(nl, enable=True):
    _check(load().md_profile_enable(nl._h, C.c_int(1 if enable else 0)), "md_profile_enable")


def md_profile_read(nl):
    """Synchronises; returns ({kind: ms}, {kind: kernel launches}) since the last read."""
    ms = (C.c_double * 4)()
    ln = (C.c_int64 * 4)()
    _check(load().md_profile_read(nl._h, ms, ln), "md_profile_read")
    return {k: ms[i] for i, k in enumerate(KINDS)}, {k: int(ln[i]) for i, k in enumerate(KINDS)}
