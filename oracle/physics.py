"""ctypes front-end of ORACLE B (oracle/sph_physics.c).  TEST INFRASTRUCTURE ONLY - see the
header of sph_physics.c.  Builds ``oracle/_build/liborc.so`` with gcc on first use
(``-O2 -fopenmp -ffp-contract=off``: no FMA contraction, so the fp64 arithmetic is the
plain one written in the source).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sph_physics.c")
_OUT = os.path.join(_HERE, "_build", "liborc.so")
_lib = None


class OrcParams(C.Structure):
    _fields_ = [
        ("h", C.c_double), ("rho0", C.c_double), ("c0", C.c_double), ("alpha", C.c_double),
        ("gamma", C.c_double), ("g", C.c_double * 3),
        ("mass_fluid", C.c_double), ("mass_bound", C.c_double),
        ("kernel", C.c_int), ("periodic", C.c_int * 3),
        ("box_min", C.c_double * 3), ("box_len", C.c_double * 3),
    ]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_OUT) or os.path.getmtime(_OUT) < os.path.getmtime(_SRC):
        os.makedirs(os.path.dirname(_OUT), exist_ok=True)
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", _OUT, _SRC, "-lm"])
    return _OUT


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.orc_W.restype = C.c_double
        L.orc_W.argtypes = [C.POINTER(OrcParams), C.c_double]
        L.orc_F.restype = C.c_double
        L.orc_F.argtypes = [C.POINTER(OrcParams), C.c_double]
        L.orc_pressure.restype = C.c_double
        L.orc_pressure.argtypes = [C.POINTER(OrcParams), C.c_double]
        L.orc_sound_speed.restype = C.c_double
        L.orc_sound_speed.argtypes = [C.POINTER(OrcParams), C.c_double]
        L.orc_threads.restype = C.c_int
        L.orc_rates.restype = C.c_int
        L.orc_rates.argtypes = [C.POINTER(OrcParams), C.c_long, dp, dp, dp, C.c_void_p, C.c_void_p,
                                C.c_int, dp, dp]
        L.orc_verlet.restype = None
        L.orc_verlet.argtypes = [C.c_long, dp, dp, dp, dp, dp, C.c_void_p, dp, dp, C.c_double, C.c_int]
        L.orc_step.restype = C.c_int
        L.orc_step.argtypes = [C.POINTER(OrcParams), C.c_long, dp, dp, dp, dp, dp, C.c_void_p,
                               C.c_double, C.c_long, C.c_int, C.c_int, dp, dp]
        L.orc_time_step.restype = C.c_int
        L.orc_time_step.argtypes = [C.POINTER(OrcParams), C.c_long, dp, dp, dp, C.c_void_p, dp, C.c_double,
                                    C.c_double, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, dp]
        L.orc_neighbour_pairs.restype = C.c_int
        L.orc_neighbour_pairs.argtypes = [C.POINTER(OrcParams), C.c_long, dp, C.c_long,
                                          C.POINTER(C.c_long), C.POINTER(C.c_long)]
        _lib = L
    return _lib


def make_params(h, rho0=1000.0, c0=10.0, alpha=0.01, gamma=7.0, g=(0.0, 0.0, -9.81),
                mass_fluid=1.0, mass_bound=None, kernel=0, periodic=(0, 0, 0),
                box_min=(0.0, 0.0, 0.0), box_len=(1.0, 1.0, 1.0)) -> OrcParams:
    p = OrcParams()
    p.h, p.rho0, p.c0, p.alpha, p.gamma = float(h), float(rho0), float(c0), float(alpha), float(gamma)
    p.g[:] = [float(x) for x in g]
    p.mass_fluid = float(mass_fluid)
    p.mass_bound = float(mass_fluid if mass_bound is None else mass_bound)
    p.kernel = int(kernel)
    p.periodic[:] = [int(x) for x in periodic]
    p.box_min[:] = [float(x) for x in box_min]
    p.box_len[:] = [float(x) for x in box_len]
    return p


def params_from_workload(P: dict) -> OrcParams:
    """fp64 copies of the (fp32-representable) workload parameters."""
    return make_params(h=P["h"], rho0=P["rho0"], c0=P["c0"], alpha=P["alpha"], gamma=P["gamma"],
                       g=P["g"], mass_fluid=P["mass_fluid"], mass_bound=P["mass_bound"],
                       kernel=P.get("kernel", 0))


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def W(p: OrcParams, r: float) -> float:
    return lib().orc_W(C.byref(p), float(r))


def F(p: OrcParams, r: float) -> float:
    return lib().orc_F(C.byref(p), float(r))


def pressure(p: OrcParams, rho: float) -> float:
    return lib().orc_pressure(C.byref(p), float(rho))


def sound_speed(p: OrcParams, rho: float) -> float:
    return lib().orc_sound_speed(C.byref(p), float(rho))


def threads() -> int:
    return int(lib().orc_threads())


def rates(p: OrcParams, r, v, rho, typ, p_override=None, mode=1):
    """(acc (n,3), drho (n,)) - right-hand sides of Eqs. (9) and (7)."""
    r, rp = _d(r)
    v, vp = _d(v)
    rho, rhop = _d(rho)
    typ = np.ascontiguousarray(typ, dtype=np.uint8)
    n = rho.shape[0]
    acc = np.zeros((n, 3), dtype=np.float64)
    drho = np.zeros(n, dtype=np.float64)
    po = None
    if p_override is not None:
        pov = np.ascontiguousarray(p_override, dtype=np.float64)
        po = pov.ctypes.data
    rc = lib().orc_rates(C.byref(p), n, rp, vp, rhop, typ.ctypes.data, po, int(mode),
                         acc.ctypes.data_as(C.POINTER(C.c_double)),
                         drho.ctypes.data_as(C.POINTER(C.c_double)))
    assert rc == 0
    return acc, drho


def time_step(p: OrcParams, r, v, rho, typ, acc, cfl=0.2, cut=1.0, slab_of=None, n_slabs=0):
    """Variable time step of reading A8b: dict(dt, dt_f, dt_cv, mu (n,), amax_slab, smax_slab)."""
    r, rp = _d(r)
    v, vp = _d(v)
    rho, rhop = _d(rho)
    acc, ap = _d(acc)
    typ = np.ascontiguousarray(typ, dtype=np.uint8)
    n = rho.shape[0]
    mu = np.zeros(n, dtype=np.float64)
    out = np.zeros(3, dtype=np.float64)
    am = np.zeros(max(n_slabs, 1), dtype=np.float64)
    sm = np.zeros(max(n_slabs, 1), dtype=np.float64)
    so = None
    if slab_of is not None:
        sov = np.ascontiguousarray(slab_of, dtype=np.int64)
        so = sov.ctypes.data
    rc = lib().orc_time_step(C.byref(p), n, rp, vp, rhop, typ.ctypes.data, ap, float(cfl), float(cut), so,
                             int(n_slabs), am.ctypes.data, sm.ctypes.data, mu.ctypes.data,
                             out.ctypes.data_as(C.POINTER(C.c_double)))
    assert rc == 0
    return dict(dt=out[0], dt_f=out[1], dt_cv=out[2], mu=mu, amax_slab=am[:n_slabs], smax_slab=sm[:n_slabs])


class State:
    """fp64 particle state in id order."""

    def __init__(self, pos, vel, rho, typ):
        self.r = np.array(pos, dtype=np.float64, order="C")
        self.v = np.array(vel, dtype=np.float64, order="C")
        self.rho = np.array(rho, dtype=np.float64, order="C")
        self.v_m1 = self.v.copy()
        self.rho_m1 = self.rho.copy()
        self.type = np.ascontiguousarray(typ, dtype=np.uint8)
        self.n = self.rho.shape[0]
        self.acc = np.zeros((self.n, 3), dtype=np.float64)
        self.drho = np.zeros(self.n, dtype=np.float64)
        self.step_index = 0


def step(p: OrcParams, s: State, dt: float, verlet_ns: int = 40, mode: int = 1) -> None:
    dp = C.POINTER(C.c_double)
    rc = lib().orc_step(C.byref(p), s.n, s.r.ctypes.data_as(dp), s.v.ctypes.data_as(dp),
                        s.rho.ctypes.data_as(dp), s.v_m1.ctypes.data_as(dp),
                        s.rho_m1.ctypes.data_as(dp), s.type.ctypes.data, float(dt),
                        int(s.step_index), int(verlet_ns), int(mode),
                        s.acc.ctypes.data_as(dp), s.drho.ctypes.data_as(dp))
    assert rc == 0
    s.step_index += 1


def neighbour_pairs(p: OrcParams, r, max_pairs=None):
    """All ordered pairs (i, j), j != i, 0 < |r_ij| < 2h, by brute force."""
    r, rp = _d(r)
    n = r.shape[0]
    if max_pairs is None:
        max_pairs = max(1, 400 * n)
    out = np.zeros((max_pairs, 2), dtype=np.int64)
    cnt = C.c_long(0)
    rc = lib().orc_neighbour_pairs(C.byref(p), n, rp, max_pairs,
                                   out.ctypes.data_as(C.POINTER(C.c_long)), C.byref(cnt))
    assert rc == 0, "max_pairs too small"
    return out[:cnt.value]
