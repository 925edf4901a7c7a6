"""ORACLE — TEST INFRASTRUCTURE ONLY.  ctypes front end of oracle/libmfc_oracle.so.

Importers allowed: tests/, __graft_entry__.smoke(), bench.py's cpu_baseline and
--impl reference legs.  Nothing under paper_2503_07953_b200/ imports this module and
this module imports nothing from there.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

BC_PERIODIC, BC_EXTRAP = 0, 1
RECON_PC, RECON_WENO5 = 1, 5
RECON_WENO5_M, RECON_WENO5_Z = 6, 7   # mapped (Henrick) and WENO-Z weights
MODEL_BY_NAME = {"allaire": 0, "kapila": 1}   # PAPER.md:86 / 59, 78-86
RECON_BY_NAME = {"js": RECON_WENO5, "m": RECON_WENO5_M, "z": RECON_WENO5_Z}
_MAXF = 4


class OracleParams(C.Structure):
    _fields_ = [("ndim", C.c_int), ("n", C.c_int * 3), ("dx", C.c_double * 3), ("nfluids", C.c_int),
                ("gamma", C.c_double * _MAXF), ("pi_inf", C.c_double * _MAXF),
                ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3),
                ("weno_eps", C.c_double), ("alpha_floor", C.c_double), ("clamp", C.c_int), ("recon", C.c_int), ("model", C.c_int), ("eta", C.c_double),
                ("form", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        pp = C.POINTER(OracleParams)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_num_eqns.argtypes = [pp]
        L.oracle_ghost_index.argtypes = [C.c_int] * 4
        L.oracle_prim_from_cons.argtypes = [pp, dp, dp]; L.oracle_prim_from_cons.restype = C.c_long
        L.oracle_rhs.argtypes = [pp, dp, dp, C.c_int]; L.oracle_rhs.restype = C.c_long
        L.oracle_rk3_step.argtypes = [pp, dp, C.c_double]; L.oracle_rk3_step.restype = C.c_long
        L.oracle_cfl_dt.argtypes = [pp, dp, C.c_double]; L.oracle_cfl_dt.restype = C.c_double
        L.oracle_weno5_js.argtypes = [dp, C.c_double, dp, dp]; L.oracle_weno5_js.restype = None
        L.oracle_weno5_js_ld.argtypes = [dp, C.c_double, dp, dp]; L.oracle_weno5_js_ld.restype = None
        L.oracle_weno5_js_textbook.argtypes = [dp, C.c_double, dp, dp]; L.oracle_weno5_js_textbook.restype = None
        L.oracle_weno5_js_textbook_ld.argtypes = [dp, C.c_double, dp, dp]; L.oracle_weno5_js_textbook_ld.restype = None
        L.oracle_weno5.argtypes = [C.c_int, dp, C.c_double, dp, dp]; L.oracle_weno5.restype = None
        L.oracle_weno5_ld.argtypes = [C.c_int, dp, C.c_double, dp, dp]; L.oracle_weno5_ld.restype = None
        L.oracle_kapila_K.argtypes = [C.POINTER(OracleParams), C.c_double, C.c_double, C.c_double]
        L.oracle_kapila_K.restype = C.c_double
        L.oracle_weno5_weights.argtypes = [C.c_int, dp, dp, C.c_double, dp]; L.oracle_weno5_weights.restype = None
        L.oracle_hllc_face.argtypes = [pp, C.c_int, dp, dp, dp, dp]
        L.oracle_clamp_cell.argtypes = [pp, dp]; L.oracle_clamp_cell.restype = None
        L.oracle_rhs_ld.argtypes = [pp, dp, dp, C.c_int]; L.oracle_rhs_ld.restype = C.c_long
        L.oracle_rk3_steps_ld.argtypes = [pp, dp, C.c_double, C.c_int]; L.oracle_rk3_steps_ld.restype = C.c_long
        L.oracle_count_rhs.argtypes = [pp, dp, C.POINTER(C.c_longlong)]; L.oracle_count_rhs.restype = None
        _lib = L
    return _lib


def _dp(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def make_params(case, recon=None):
    """case: a workloads.Case (n, dx, gamma, pi_inf, bc_lo, bc_hi, weno_eps, alpha_floor, clamp[, weno])."""
    if recon is None:
        recon = RECON_BY_NAME[getattr(case, "weno", "js")]
    p = OracleParams()
    p.ndim = case.ndim
    for d in range(3):
        p.n[d] = case.n[d]
        p.dx[d] = case.dx[d]
        p.bc_lo[d] = case.bc_lo[d]
        p.bc_hi[d] = case.bc_hi[d]
    p.nfluids = case.nfluids
    for i in range(case.nfluids):
        p.gamma[i] = case.gamma[i]
        p.pi_inf[i] = case.pi_inf[i]
    p.weno_eps = case.weno_eps
    p.alpha_floor = case.alpha_floor
    p.clamp = int(case.clamp)
    p.recon = recon
    p.model = MODEL_BY_NAME[getattr(case, "model", "allaire")]
    p.eta = float(getattr(case, "eta", 0.0))
    return p


class Oracle:
    """The five operations of include/mfc_b200.h on host numpy arrays (SoA, x fastest)."""

    def __init__(self, case, recon=None, form="difference"):
        """form: "difference" (readings N2/N3, what the parity bars are measured against) or "textbook" (O3 and O4 typed
        as PAPER.md:163 / 197 print them) — mfc_oracle.hpp FORM_*"""
        self.case = case
        self.p = make_params(case, recon)
        self.p.form = {"difference": 0, "textbook": 1}[form]
        self.neq = 2 * case.nfluids + case.ndim + 1
        self.shape = (self.neq, case.n[2], case.n[1], case.n[0])

    def prim_from_cons(self, q):
        w = np.empty_like(q)
        self.bad = lib().oracle_prim_from_cons(C.byref(self.p), _dp(q), _dp(w))
        return w

    def rhs(self, q, dir_mask=7):
        r = np.empty_like(q)
        self.bad = lib().oracle_rhs(C.byref(self.p), _dp(q), _dp(r), dir_mask)
        return r

    def rhs_ld(self, q, dir_mask=7):
        r = np.empty_like(q)
        self.bad = lib().oracle_rhs_ld(C.byref(self.p), _dp(q), _dp(r), dir_mask)
        return r

    def rk3_step(self, q, dt):
        """in place"""
        self.bad = lib().oracle_rk3_step(C.byref(self.p), _dp(q), float(dt))
        return q

    def rk3_steps_ld(self, q, dt, nsteps):
        self.bad = lib().oracle_rk3_steps_ld(C.byref(self.p), _dp(q), float(dt), int(nsteps))
        return q

    def cfl_dt(self, q, cfl):
        return lib().oracle_cfl_dt(C.byref(self.p), _dp(q), float(cfl))

    def count_rhs(self, q):
        c = (C.c_longlong * 5)()
        lib().oracle_count_rhs(C.byref(self.p), _dp(q), c)
        return dict(add=c[0], mul=c[1], div=c[2], sqrt=c[3], cmp=c[4])

    def hllc_face(self, d, wL, wR):
        wL = np.ascontiguousarray(wL, dtype=np.float64)
        wR = np.ascontiguousarray(wR, dtype=np.float64)
        F = np.empty(self.neq)
        uf = C.c_double()
        bad = lib().oracle_hllc_face(C.byref(self.p), d, _dp(wL), _dp(wR), _dp(F), C.byref(uf))
        return F, uf.value, bad

    def kapila_K(self, p, alpha1, alpha2):
        return lib().oracle_kapila_K(C.byref(self.p), float(p), float(alpha1), float(alpha2))

    def clamp_cell(self, q):
        q = np.ascontiguousarray(q, dtype=np.float64).copy()
        lib().oracle_clamp_cell(C.byref(self.p), _dp(q))
        return q


def weno5_js(s, eps, form="difference"):
    """form: "difference" (weno5_js, reading N2) or "textbook" (weno5_js_textbook, PAPER.md:163 as printed)"""
    s = np.ascontiguousarray(s, dtype=np.float64)
    l, r = C.c_double(), C.c_double()
    fn = {"difference": lib().oracle_weno5_js, "textbook": lib().oracle_weno5_js_textbook}[form]
    fn(_dp(s), float(eps), C.byref(l), C.byref(r))
    return l.value, r.value


def weno5(recon, s, eps, ld=False):
    """general routine with the weights variant `recon`; ld: the same text in 80-bit arithmetic"""
    s = np.ascontiguousarray(s, dtype=np.float64)
    l, r = C.c_double(), C.c_double()
    (lib().oracle_weno5_ld if ld else lib().oracle_weno5)(int(recon), _dp(s), float(eps), C.byref(l), C.byref(r))
    return l.value, r.value


def weno5_weights(recon, dr, beta, eps):
    dr = np.ascontiguousarray(dr, dtype=np.float64)
    beta = np.ascontiguousarray(beta, dtype=np.float64)
    om = np.empty(3)
    lib().oracle_weno5_weights(int(recon), _dp(dr), _dp(beta), float(eps), _dp(om))
    return om


def weno5_js_ld(s, eps, form="difference"):
    s = np.ascontiguousarray(s, dtype=np.float64)
    l, r = C.c_double(), C.c_double()
    fn = {"difference": lib().oracle_weno5_js_ld, "textbook": lib().oracle_weno5_js_textbook_ld}[form]
    fn(_dp(s), float(eps), C.byref(l), C.byref(r))
    return l.value, r.value


def ghost_index(g, n, lo, hi):
    return lib().oracle_ghost_index(g, n, lo, hi)


def num_threads():
    return lib().oracle_num_threads()
