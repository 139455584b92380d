"""ctypes loader for the CPU oracle (oracle/orc.cpp).  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, bench.py's cpu_baseline / --impl reference legs and __graft_entry__.smoke() may
import this module.  It does not import the CUDA package and the CUDA package does not import it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "orc.cpp")
_LIB = os.path.join(_HERE, "liborc.so")
BUILD_CMD = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c++17", "-shared", "-fPIC", "-o", _LIB, _SRC]


class Params(C.Structure):
    _fields_ = [
        ("metric", C.c_int), ("bh_mass", C.c_double), ("bh_spin", C.c_double), ("r_excise", C.c_double),
        ("nbx", C.c_int), ("nby", C.c_int), ("nbz", C.c_int),
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ng", C.c_int),
        ("xmin", C.c_double * 3), ("xmax", C.c_double * 3), ("bc", (C.c_int * 2) * 3),
        ("gamma_ad", C.c_double), ("recon", C.c_int), ("riemann", C.c_int), ("use_ct", C.c_int),
        ("rho_floor", C.c_double), ("eps_floor", C.c_double), ("w_max", C.c_double),
        ("c2p_tol", C.c_double), ("c2p_maxit", C.c_int), ("shift", C.c_double * 3),
        ("nscalar", C.c_int), ("scalar_min", C.c_double), ("scalar_max", C.c_double),
        ("floor_form", C.c_int), ("floor_alpha_rho", C.c_double), ("floor_alpha_eps", C.c_double),
    ]

# parameters added after the first version of the ABI: optional in the dictionaries, with the values that switch them off
_OPTIONAL = dict(shift=(0.0, 0.0, 0.0), nscalar=0, scalar_min=0.0, scalar_max=1.0, floor_form=0,
                 floor_alpha_rho=2.0, floor_alpha_eps=1.0)


def make_params(p: dict) -> Params:
    q = Params()
    for name, _ in Params._fields_:
        v = p.get(name, _OPTIONAL[name]) if name in _OPTIONAL else p[name]
        if name in ("xmin", "xmax", "shift"):
            setattr(q, name, (C.c_double * 3)(*v))
        elif name == "bc":
            arr = ((C.c_int * 2) * 3)()
            for d in range(3):
                arr[d][0], arr[d][1] = int(v[d][0]), int(v[d][1])
            q.bc = arr
        else:
            setattr(q, name, v)
    return q


def build(force=False):
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.run(BUILD_CMD, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        dp, ucp, pp = C.POINTER(C.c_double), C.POINTER(C.c_ubyte), C.POINTER(Params)
        L.orc_field_elems.restype = C.c_size_t
        L.orc_field_elems.argtypes = [pp]
        L.orc_last_c2p_margin.restype = C.c_double
        L.orc_prim_to_cons.argtypes = [pp, dp, dp]
        L.orc_cons_to_prim.argtypes = [pp, dp, dp, ucp]
        L.orc_fill_ghosts.argtypes = [pp, dp]
        L.orc_rk_stage.argtypes = [pp, C.c_double, C.c_double, C.c_double, dp, dp, dp, ucp]
        L.orc_cfl_dt.argtypes = [pp, dp, C.c_double, dp]
        L.orc_stage_fluxes.argtypes = [pp, dp, dp, dp, dp]
        L.orc_metric.argtypes = [pp, dp, dp]
        L.orc_metric_derivs.argtypes = [pp, dp, dp]
        L.orc_split31.argtypes = [dp, dp]
        L.orc_point_cons.argtypes = [dp, C.c_double, dp, dp]
        L.orc_point_flux.argtypes = [dp, C.c_double, dp, C.c_int, dp]
        L.orc_point_speeds.argtypes = [dp, C.c_double, dp, C.c_int, dp, dp]
        L.orc_point_source.argtypes = [dp, dp, C.c_double, dp, dp]
        L.orc_point_stress_energy.argtypes = [dp, C.c_double, dp, dp]
        L.orc_point_c2p.argtypes = [pp, dp, dp, dp]
        L.orc_point_c2p.restype = C.c_int
        L.orc_point_riemann.argtypes = [pp, dp, C.c_int, dp, dp, dp]
        L.orc_recon_line.argtypes = [C.c_int, C.c_int, dp, dp, dp]
        L.orc_point_floors.argtypes = [pp, dp, dp, dp]
        L.orc_point_riemann_scalar.argtypes = [pp, dp, C.c_int, dp, dp, dp]
        _lib = L
    return _lib


def _d(a):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _u8(a):
    assert a.dtype == np.uint8 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_ubyte))


def set_threads(n):
    os.environ["OMP_NUM_THREADS"] = str(n)


# ----------------------------------------------------------------------------- field calls
def prim_to_cons(p, prim):
    cons = np.empty_like(prim)
    lib().orc_prim_to_cons(C.byref(make_params(p)), _d(prim), _d(cons))
    return cons


def cons_to_prim(p, cons, prim=None):
    """cons is rewritten where floored.  Returns (prim, mask)."""
    if prim is None:
        prim = np.zeros_like(cons)
    mask = np.zeros((cons.shape[0],) + cons.shape[2:], dtype=np.uint8)
    lib().orc_cons_to_prim(C.byref(make_params(p)), _d(cons), _d(prim), _u8(mask))
    return prim, mask


def fill_ghosts(p, prim):
    lib().orc_fill_ghosts(C.byref(make_params(p)), _d(prim))
    return prim


def rk_stage(p, g0, g1, beta_dt, cons0, cons, prim, mask):
    lib().orc_rk_stage(C.byref(make_params(p)), g0, g1, beta_dt, _d(cons0), _d(cons), _d(prim), _u8(mask))


def cfl_dt(p, prim, cfl):
    out = C.c_double(0.0)
    lib().orc_cfl_dt(C.byref(make_params(p)), _d(prim), cfl, C.byref(out))
    return out.value


def stage_fluxes(p, prim):
    F = [np.zeros_like(prim) for _ in range(3)]
    lib().orc_stage_fluxes(C.byref(make_params(p)), _d(prim), _d(F[0]), _d(F[1]), _d(F[2]))
    return F


def last_c2p_margin():
    return lib().orc_last_c2p_margin()


def reset_c2p_margin():
    lib().orc_reset_c2p_margin()


class Run:
    """RK2 (Heun / SSPRK2) driver over the oracle: stage (1,0,dt) then (1/2,1/2,dt/2)."""

    def __init__(self, p, prim):
        self.p = dict(p)
        self.prim = np.ascontiguousarray(prim, dtype=np.float64).copy()
        self.cons = prim_to_cons(self.p, self.prim)
        self.mask = np.zeros((prim.shape[0],) + prim.shape[2:], dtype=np.uint8)
        self.mask1 = np.zeros_like(self.mask)
        self.t = 0.0
        self.dts = []

    def step(self, dt):
        cons0 = self.cons.copy()
        rk_stage(self.p, 1.0, 0.0, dt, cons0, self.cons, self.prim, self.mask1)
        rk_stage(self.p, 0.5, 0.5, 0.5 * dt, cons0, self.cons, self.prim, self.mask)
        self.t += dt
        self.dts.append(dt)

    def dt(self, cfl):
        return cfl_dt(self.p, self.prim, cfl)


# ----------------------------------------------------------------------------- point hooks
def metric(p, x):
    g = np.zeros((4, 4)); x = np.asarray(x, dtype=np.float64)
    lib().orc_metric(C.byref(make_params(p)), _d(x), _d(g))
    return g


def metric_derivs(p, x):
    dg = np.zeros((3, 4, 4)); x = np.asarray(x, dtype=np.float64)
    lib().orc_metric_derivs(C.byref(make_params(p)), _d(x), _d(dg))
    return dg


def split31(g4):
    out = np.zeros(26); g4 = np.ascontiguousarray(g4, dtype=np.float64)
    lib().orc_split31(_d(g4), _d(out))
    return dict(alpha=out[0], beta_u=out[1:4].copy(), beta_l=out[4:7].copy(), gamma_l=out[7:16].reshape(3, 3).copy(),
                gamma_u=out[16:25].reshape(3, 3).copy(), sqrtg=out[25])


def point_cons(g4, gam, q):
    U = np.zeros(8); g4 = np.ascontiguousarray(g4); q = np.ascontiguousarray(q, dtype=np.float64)
    lib().orc_point_cons(_d(g4), gam, _d(q), _d(U))
    return U


def point_flux(g4, gam, q, d):
    F = np.zeros(8); g4 = np.ascontiguousarray(g4); q = np.ascontiguousarray(q, dtype=np.float64)
    lib().orc_point_flux(_d(g4), gam, _d(q), d, _d(F))
    return F


def point_speeds(g4, gam, q, d):
    lm, lp = C.c_double(), C.c_double()
    g4 = np.ascontiguousarray(g4); q = np.ascontiguousarray(q, dtype=np.float64)
    lib().orc_point_speeds(_d(g4), gam, _d(q), d, C.byref(lm), C.byref(lp))
    return lm.value, lp.value


def point_source(g4, dg, gam, q):
    S = np.zeros(8)
    g4 = np.ascontiguousarray(g4); dg = np.ascontiguousarray(dg); q = np.ascontiguousarray(q, dtype=np.float64)
    lib().orc_point_source(_d(g4), _d(dg), gam, _d(q), _d(S))
    return S


def point_stress_energy(g4, gam, q):
    T = np.zeros((4, 4)); g4 = np.ascontiguousarray(g4); q = np.ascontiguousarray(q, dtype=np.float64)
    lib().orc_point_stress_energy(_d(g4), gam, _d(q), _d(T))
    return T


def point_c2p(p, g4, U):
    """U densitised conserved (copied); returns (prim, mask, U_after)."""
    U = np.array(U, dtype=np.float64); q = np.zeros(8); g4 = np.ascontiguousarray(g4)
    m = lib().orc_point_c2p(C.byref(make_params(p)), _d(g4), _d(U), _d(q))
    return q, m, U


def point_riemann(p, g4, d, qL, qR):
    F = np.zeros(8); g4 = np.ascontiguousarray(g4)
    qL = np.ascontiguousarray(qL, dtype=np.float64); qR = np.ascontiguousarray(qR, dtype=np.float64)
    lib().orc_point_riemann(C.byref(make_params(p)), _d(g4), d, _d(qL), _d(qR), _d(F))
    return F


def point_floors(p, x):
    """(rho_flr, eps_flr) at the point x (PAPER.md:288 forms)."""
    x = np.asarray(x, dtype=np.float64); r, e = C.c_double(), C.c_double()
    lib().orc_point_floors(C.byref(make_params(p)), _d(x), C.byref(r), C.byref(e))
    return r.value, e.value


def point_riemann_scalar(p, g4, d, qL, qR):
    """Riemann flux of the 8 variables and the passive scalar (9 entries in, 9 out)."""
    F = np.zeros(9); g4 = np.ascontiguousarray(g4)
    qL = np.ascontiguousarray(qL, dtype=np.float64); qR = np.ascontiguousarray(qR, dtype=np.float64)
    lib().orc_point_riemann_scalar(C.byref(make_params(p)), _d(g4), d, _d(qL), _d(qR), _d(F))
    return F


def recon_line(recon, f):
    f = np.ascontiguousarray(f, dtype=np.float64)
    qm = np.full_like(f, np.nan); qp = np.full_like(f, np.nan)
    lib().orc_recon_line(recon, len(f), _d(f), _d(qm), _d(qp))
    return qm, qp
