"""ORACLE — TEST INFRASTRUCTURE ONLY.

ctypes binding of oracle/liboracle.so (built from cavity_oracle.cpp by oracle/build.py).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package; the product (paper_0809_3098_b200) never does.
"""
import ctypes as C

import numpy as np

from .build import build

MODE_PLAIN = 0
MODE_FMA = 1
SWEEP_REDBLACK, SWEEP_JACOBI, SWEEP_COMPACT9 = 0, 1, 2

_lib = None


class OrcDiag(C.Structure):
    _fields_ = [("t", C.c_double), ("step", C.c_longlong), ("res_inf", C.c_double), ("res_l2", C.c_double),
                ("kinetic_energy", C.c_double), ("enstrophy", C.c_double)]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.orc_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_double, C.c_double, C.c_double, C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_destroy.restype = None
        L.orc_set_mode.argtypes = [C.c_void_p, C.c_int]
        L.orc_set_lid.argtypes = [C.c_void_p, C.c_double]
        L.orc_set_fields.argtypes = [C.c_void_p, dp, dp]
        L.orc_get_fields.argtypes = [C.c_void_p, dp, dp]
        L.orc_step.argtypes = [C.c_void_p, C.c_int]
        L.orc_poisson.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_get_diag.argtypes = [C.c_void_p, C.POINTER(OrcDiag)]
        L.orc_rhs.argtypes = [C.c_int, C.c_double, C.c_int, dp, dp, dp]
        L.orc_thom.argtypes = [C.c_int, C.c_double, C.c_int, dp, dp]
        L.orc_sor.argtypes = [C.c_int, C.c_double, C.c_int, dp, dp, C.c_int]
        L.orc_set_sweep.argtypes = [C.c_void_p, C.c_int]
        L.orc_jacobi.argtypes = [C.c_int, C.c_double, C.c_int, dp, dp, C.c_int]
        L.orc_compact.argtypes = [C.c_int, C.c_double, C.c_int, dp, dp, C.c_int]
        L.orc_compact_lex.argtypes = [C.c_int, C.c_double, C.c_int, dp, dp, C.c_int]
        L.orc_step_res.argtypes = [C.c_void_p, dp, dp]
        L.orc_run_to_steady.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.POINTER(C.c_int), dp, dp,
                                        C.POINTER(C.c_int)]
        L.orc_ssprk54_scalar.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int, C.c_int]
        L.orc_ssprk54_scalar.restype = C.c_double
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError("%s failed with code %d" % (what, rc))


def _field(a, N, name):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.shape != (N + 1, N + 1):
        raise ValueError("%s must have shape (N+1, N+1) = (%d, %d), row j = y index" % (name, N + 1, N + 1))
    return a


class OracleCavity:
    """Same call sequence as the C-ABI of include/cavity.h, on the CPU oracle.

    Fields are numpy (N+1, N+1) float64 arrays indexed [j, i] (j = y index, row N = lid)."""

    def __init__(self, N, Re, dt, sor_omega, sweeps_per_stage, mode=MODE_PLAIN):
        self.N = int(N)
        self._h = C.c_void_p()
        _chk(lib().orc_create(C.byref(self._h), N, Re, dt, sor_omega, sweeps_per_stage), "orc_create")
        _chk(lib().orc_set_mode(self._h, mode), "orc_set_mode")

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_sweep(self, kind):
        """SWEEP_REDBLACK (default), SWEEP_JACOBI or SWEEP_COMPACT9."""
        _chk(lib().orc_set_sweep(self._h, kind), "orc_set_sweep")

    def step_res(self):
        """One time step; returns (RES_psi, RES_omega) of that step (eq 26-27)."""
        rp, rw = C.c_double(), C.c_double()
        _chk(lib().orc_step_res(self._h, C.byref(rp), C.byref(rw)), "orc_step_res")
        return rp.value, rw.value

    def run_to_steady(self, max_steps, check_every, tol_psi, tol_omega):
        n, conv, rp, rw = C.c_int(), C.c_int(), C.c_double(), C.c_double()
        _chk(lib().orc_run_to_steady(self._h, max_steps, check_every, tol_psi, tol_omega, C.byref(n), C.byref(rp),
                                     C.byref(rw), C.byref(conv)), "orc_run_to_steady")
        return {"steps": n.value, "res_psi": rp.value, "res_omega": rw.value, "converged": bool(conv.value)}

    def set_lid(self, U):
        _chk(lib().orc_set_lid(self._h, U), "orc_set_lid")

    def set_fields(self, psi, omega):
        psi = None if psi is None else _field(psi, self.N, "psi")
        omega = _field(omega, self.N, "omega")
        _chk(lib().orc_set_fields(self._h, _p(psi), _p(omega)), "orc_set_fields")

    def get_fields(self):
        psi = np.empty((self.N + 1, self.N + 1))
        w = np.empty((self.N + 1, self.N + 1))
        _chk(lib().orc_get_fields(self._h, _p(psi), _p(w)), "orc_get_fields")
        return psi, w

    def step(self, nsteps=1):
        _chk(lib().orc_step(self._h, nsteps), "orc_step")

    def poisson(self, nsweeps):
        r = C.c_double()
        _chk(lib().orc_poisson(self._h, nsweeps, C.byref(r)), "orc_poisson")
        return r.value

    def diag(self):
        d = OrcDiag()
        _chk(lib().orc_get_diag(self._h, C.byref(d)), "orc_get_diag")
        return {"t": d.t, "step": d.step, "res_inf": d.res_inf, "res_l2": d.res_l2,
                "kinetic_energy": d.kinetic_energy, "enstrophy": d.enstrophy}


def rhs(N, Re, psi, omega, mode=MODE_PLAIN):
    psi, omega = _field(psi, N, "psi"), _field(omega, N, "omega")
    out = np.empty_like(psi)
    _chk(lib().orc_rhs(N, Re, mode, _p(psi), _p(omega), _p(out)), "orc_rhs")
    return out


def thom(N, U, psi, omega, mode=MODE_PLAIN):
    psi = _field(psi, N, "psi")
    w = _field(omega, N, "omega").copy()
    _chk(lib().orc_thom(N, U, mode, _p(psi), _p(w)), "orc_thom")
    return w


def sor(N, beta, psi, omega, nsweeps, mode=MODE_PLAIN):
    p = _field(psi, N, "psi").copy()
    omega = _field(omega, N, "omega")
    _chk(lib().orc_sor(N, beta, mode, _p(p), _p(omega), nsweeps), "orc_sor")
    return p


def jacobi(N, beta, psi, omega, nsweeps, mode=MODE_PLAIN):
    p = _field(psi, N, "psi").copy()
    omega = _field(omega, N, "omega")
    _chk(lib().orc_jacobi(N, beta, mode, _p(p), _p(omega), nsweeps), "orc_jacobi")
    return p


def compact(N, beta, psi, omega, nsweeps, mode=MODE_PLAIN):
    """Four-colour sweeps of the paper's 4th-order compact operator (eq 14-21)."""
    p = _field(psi, N, "psi").copy()
    omega = _field(omega, N, "omega")
    _chk(lib().orc_compact(N, beta, mode, _p(p), _p(omega), nsweeps), "orc_compact")
    return p


def compact_lex(N, beta, psi, omega, nsweeps, mode=MODE_PLAIN):
    """Lexicographic sweeps of the compact operator, the paper's own order; oracle only (NEXT-3)."""
    p = _field(psi, N, "psi").copy()
    omega = _field(omega, N, "omega")
    _chk(lib().orc_compact_lex(N, beta, mode, _p(p), _p(omega), nsweeps), "orc_compact_lex")
    return p


def ssprk54_scalar(lam, dt, y0, nsteps, mode=MODE_PLAIN):
    return lib().orc_ssprk54_scalar(lam, dt, y0, nsteps, mode)
