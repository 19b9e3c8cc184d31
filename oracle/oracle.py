"""ctypes wrapper of the CPU oracle (oracle/oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Never imported by the product package and shares no
code with it.  `build()` compiles the C file with gcc (building the checker is not using it).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = [os.path.join(_HERE, f) for f in ("oracle.c", "oracle_source.inc", "oracle_mech.h")]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(_SO)
            and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC)):
        return _SO
    cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wno-unknown-pragmas",
           os.path.join(_HERE, "oracle.c"), "-o", _SO, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


_pd = C.POINTER(C.c_double)
_pi = C.POINTER(C.c_int)


class _OrcMech(C.Structure):
    _fields_ = [("ns", C.c_int), ("nr", C.c_int),
                ("mw", _pd), ("nasa_lo", _pd), ("nasa_hi", _pd), ("t_mid", _pd),
                ("reac_ptr", _pi), ("reac_spec", _pi), ("reac_nu", _pi),
                ("prod_ptr", _pi), ("prod_spec", _pi), ("prod_nu", _pi),
                ("rxn_type", _pi), ("rev_type", _pi),
                ("arr_hi", _pd), ("arr_lo", _pd), ("arr_rev", _pd),
                ("falloff_form", _pi), ("falloff_par", _pd), ("tb_species", _pi),
                ("eff_ptr", _pi), ("eff_spec", _pi), ("eff_val", _pd),
                ("plog_ptr", _pi), ("plog_p", _pd), ("plog_arr", _pd),
                ("cheb_ptr", _pi), ("cheb_nT", _pi), ("cheb_nP", _pi),
                ("cheb_lim", _pd), ("cheb_eta", _pd)]


def _dp(a):
    return a.ctypes.data_as(_pd)


def _ip(a):
    return a.ctypes.data_as(_pi)


class Oracle:
    """Evaluates the paper's equations on the CPU for one mechanism."""

    def __init__(self, mech, threads: int | None = None):
        self.lib = C.CDLL(build())
        self.mech = mech.normalized()
        m = self.mech
        self.ns, self.nr = m.n_species, m.n_reactions
        s = _OrcMech()
        s.ns, s.nr = self.ns, self.nr
        for name in ("mol_wt:mw", "nasa_lo", "nasa_hi", "t_mid", "arr_hi", "arr_lo", "arr_rev",
                     "falloff_par", "eff_val", "plog_p", "plog_arr", "cheb_lim", "cheb_eta"):
            src, _, dst = name.partition(":")
            setattr(s, dst or src, _dp(getattr(m, src)))
        for name in ("reac_ptr", "reac_spec", "reac_nu", "prod_ptr", "prod_spec", "prod_nu",
                     "rxn_type", "rev_type", "falloff_form", "tb_species", "eff_ptr", "eff_spec",
                     "plog_ptr", "cheb_ptr", "cheb_nT", "cheb_nP"):
            setattr(s, name, _ip(getattr(m, name)))
        self._s = s
        self.lib.orc_num_threads.restype = C.c_int
        if threads:
            self.lib.orc_set_num_threads(C.c_int(int(threads)))
        self.threads = int(self.lib.orc_num_threads())

    # -- helpers
    @staticmethod
    def _state(T, P, Y):
        T = np.ascontiguousarray(T, dtype=np.float64).reshape(-1)
        P = np.ascontiguousarray(P, dtype=np.float64).reshape(-1)
        Y = np.ascontiguousarray(Y, dtype=np.float64)
        if Y.ndim == 1:
            Y = Y.reshape(1, -1)
        assert T.shape[0] == P.shape[0] == Y.shape[0]
        return T, P, Y

    def source(self, T, P, Y):
        """dict(rf, rr, cmod [n][nr]; wdot [n][ns]; dydt [n][ns+1])"""
        T, P, Y = self._state(T, P, Y)
        n = T.shape[0]
        out = dict(rf=np.empty((n, self.nr)), rr=np.empty((n, self.nr)),
                   cmod=np.empty((n, self.nr)), wdot=np.empty((n, self.ns)),
                   dydt=np.empty((n, self.ns + 1)))
        rc = self.lib.orc_eval_source(C.byref(self._s), C.c_long(n), _dp(T), _dp(P), _dp(Y),
                                      C.c_long(Y.shape[1]), _dp(out["rf"]), _dp(out["rr"]),
                                      _dp(out["cmod"]), _dp(out["wdot"]), _dp(out["dydt"]))
        if rc != 0:
            raise MemoryError("oracle allocation failed")
        return out

    def details(self, T, P, Y):
        T, P, Y = self._state(T, P, Y)
        n = T.shape[0]
        names = ("kf", "kr", "Kc", "Pr", "F", "Xi")
        out = {k: np.empty((n, self.nr)) for k in names}
        rc = self.lib.orc_eval_details(C.byref(self._s), C.c_long(n), _dp(T), _dp(P), _dp(Y),
                                       C.c_long(Y.shape[1]), *[_dp(out[k]) for k in names])
        if rc != 0:
            raise MemoryError("oracle allocation failed")
        return out

    def species_thermo(self, T: float, T_imag: float = 0.0):
        """(re, im) arrays [5][ns]: Cp/R, H/R, S/R, B, dB/dT at a (complex) temperature."""
        re = np.empty((5, self.ns))
        im = np.empty((5, self.ns))
        self.lib.orc_species_thermo(C.byref(self._s), C.c_double(T), C.c_double(T_imag), _dp(re),
                                    _dp(im))
        return re, im

    def _jac(self, fn, T, P, Y):
        T, P, Y = self._state(T, P, Y)
        n = T.shape[0]
        ld = self.ns + 1
        jac = np.empty((n, ld * ld))
        rc = fn(C.byref(self._s), C.c_long(n), _dp(T), _dp(P), _dp(Y), C.c_long(Y.shape[1]),
                _dp(jac))
        if rc != 0:
            raise MemoryError("oracle allocation failed")
        return jac

    def jacobian(self, T, P, Y):
        """Analytical Jacobian (Section 3 equations, Algorithm 1 order): [n][(ns+1)^2]."""
        return self._jac(self.lib.orc_eval_jacobian, T, P, Y)

    def jacobian_complex_step(self, T, P, Y):
        """J = df/dPhi by complex step on the oracle's own source term."""
        return self._jac(self.lib.orc_eval_jacobian_complex_step, T, P, Y)


    def jacobian_fd(self, T, P, Y, rtol: float = 1e-8, atol: float = 1e-15):
        """First-order forward-difference Jacobian of the oracle's source term with the increments of
        DESIGN.md reading C21 (the paper's comparison method): [n][(ns+1)^2].  rtol and atol must
        be positive: with atol = 0 an unknown that is exactly zero gets the increment D_j = 0 (C21)."""
        if not (rtol > 0.0 and atol > 0.0):
            raise ValueError("jacobian_fd needs rtol > 0 and atol > 0 (DESIGN.md C21: D_j = 0 for a zero unknown otherwise)")
        T, P, Y = self._state(T, P, Y)
        n = T.shape[0]
        ld = self.ns + 1
        jac = np.empty((n, ld * ld))
        rc = self.lib.orc_eval_jacobian_fd(C.byref(self._s), C.c_long(n), _dp(T), _dp(P), _dp(Y),
                                           C.c_long(Y.shape[1]), C.c_double(rtol), C.c_double(atol), _dp(jac))
        if rc != 0:
            raise MemoryError("oracle allocation failed")
        return jac


def as_matrix(jac_flat, ns):
    """[n][(ns+1)^2] column-major -> [n][row][col]"""
    ld = ns + 1
    return np.asarray(jac_flat).reshape(-1, ld, ld).transpose(0, 2, 1)
