"""ORACLE -- TEST INFRASTRUCTURE ONLY.  ctypes access to oracle/libck_oracle.so (built by build()).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  The product package (paper_1608_05794_b200) never does.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libck_oracle.so")
_SRC = [os.path.join(_HERE, f) for f in ("ck_oracle_api.cpp", "ck_oracle_chem.hpp", "ck_oracle_solvers.hpp")]
_libs = {}
# "fma": the SAME sources compiled with fused multiply-add contraction (-mfma -ffp-contract=fast): a second correct
# FP64 execution of the same algorithm that differs from the default build in the last bit of some operations.
# Used only by the CPU test that justifies DESIGN.md's parity reading P3 (tests/test_oracle_p3.py).
_VARIANT_FLAGS = {None: [], "fma": ["-mfma", "-ffp-contract=fast"]}


def _path(variant):
    return _LIB_PATH if variant is None else _LIB_PATH.replace(".so", f"_{variant}.so")


def build(force=False, variant=None):
    """Compile the oracle: plain g++ -O2, no fast-math."""
    path = _path(variant)
    if not force and os.path.exists(path) and all(os.path.getmtime(path) >= os.path.getmtime(s) for s in _SRC):
        return path
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp"] + _VARIANT_FLAGS[variant] + ["-o", path, _SRC[0]]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return path


def lib(variant=None):
    if variant not in _libs:
        L = C.CDLL(build(variant=variant))
        L.cko_mech_create.restype = C.c_void_p
        L.cko_estimate_h0.restype = C.c_double
        _libs[variant] = L
    return _libs[variant]


def _p(a, t=C.c_double):
    return a.ctypes.data_as(C.POINTER(t))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _u8(a):
    return np.ascontiguousarray(a, dtype=np.uint8)


class Mech:
    def __init__(self, d, variant=None, const_volume=False):
        """const_volume: the `p` argument of every call is then the mass density rho."""
        L = self._L = lib(variant)
        self.K, self.R, self.E = int(d["n_species"]), int(d["n_reactions"]), int(d["n_elements"])
        self.N = self.K + 1
        keep = self._keep = dict(
            W=_f64(d["mol_wt"]), elem=_i32(d["elem_comp"]), lo=_f64(d["nasa_lo"]), hi=_f64(d["nasa_hi"]),
            tmid=_f64(d["t_mid"]), rptr=_i32(d["reac_ptr"]), rspec=_i32(d["reac_spec"]), rnu=_i32(d["reac_nu"]),
            pptr=_i32(d["prod_ptr"]), pspec=_i32(d["prod_spec"]), pnu=_i32(d["prod_nu"]),
            A=_f64(d["A"]), beta=_f64(d["beta"]), Ea=_f64(d["Ea"]), rev=_u8(d["reversible"]), type=_u8(d["type"]),
            A0=_f64(d["A0"]), beta0=_f64(d["beta0"]), Ea0=_f64(d["Ea0"]), troe=_f64(d["troe"]),
            eptr=_i32(d["eff_ptr"]), espec=_i32(d["eff_spec"]), eval=_f64(d["eff_val"]))
        k = keep
        self.h = C.c_void_p(L.cko_mech_create(
            self.K, self.R, self.E, _p(k["W"]), _p(k["elem"], C.c_int), _p(k["lo"]), _p(k["hi"]), _p(k["tmid"]),
            _p(k["rptr"], C.c_int), _p(k["rspec"], C.c_int), _p(k["rnu"], C.c_int),
            _p(k["pptr"], C.c_int), _p(k["pspec"], C.c_int), _p(k["pnu"], C.c_int),
            _p(k["A"]), _p(k["beta"]), _p(k["Ea"]), _p(k["rev"], C.c_uint8), _p(k["type"], C.c_uint8),
            _p(k["A0"]), _p(k["beta0"]), _p(k["Ea0"]), _p(k["troe"]),
            _p(k["eptr"], C.c_int), _p(k["espec"], C.c_int), _p(k["eval"])))
        if const_volume:
            L.cko_set_const_volume(self.h, 1)

    def __del__(self):
        try:
            self._L.cko_mech_free(self.h)
        except Exception:
            pass

    # ---- batch calls: y is (N, n) component-major ---------------------------------------------
    def rhs(self, y, p, prec=0, want_scale=False, nthreads=1):
        y = _f64(y); p = _f64(p)
        N, n = y.shape
        assert N == self.N and p.shape == (n,)
        f = np.empty_like(y)
        D = np.empty_like(y) if want_scale else None
        self._L.cko_rhs(self.h, C.c_longlong(n), _p(y), C.c_longlong(n), _p(p), _p(f), C.c_longlong(n),
                      _p(D) if want_scale else None, int(prec), int(nthreads))
        return (f, D) if want_scale else f

    def rates(self, y1, p):
        y1 = _f64(y1)
        qf = np.empty(self.R); qr = np.empty(self.R); rc = np.empty(2)
        self._L.cko_rates(self.h, _p(y1), C.c_double(p), _p(qf), _p(qr), _p(rc))
        return qf, qr, rc[0], rc[1]

    def thermo(self, k, T):
        out = np.empty(3)
        self._L.cko_thermo(self.h, int(k), C.c_double(T), _p(out))
        return out  # cp/R, H/RT, S/R

    def jac(self, y1, p, mode=0, h=0.0, rtol=1e-6, atol=1e-10):
        """One state y1[N] -> J[N,N] (row i = d f_i / d y_j). mode 0 complex-step, 1 FD, 2 (J, Jmag)."""
        y1 = _f64(y1)
        J = np.empty((self.N, self.N)); Jm = np.empty((self.N, self.N))
        self._L.cko_jac(self.h, _p(y1), C.c_double(p), int(mode), C.c_double(h), C.c_double(rtol), C.c_double(atol),
                      _p(J), _p(Jm))
        return (J, Jm) if mode == 2 else J

    def integrate(self, solver, y, p, dt, rtol=1e-6, atol=1e-10, jac_mode=0, h0=0.0, max_steps=100000, nthreads=1):
        """solver 'ros'|'rkf45'.  Returns dict(y, n_accept, n_reject, status, h_last, rhs_evals, jac_evals, lu)."""
        y = _f64(y).copy(); p = _f64(p)
        N, n = y.shape
        assert N == self.N
        na = np.zeros(n, np.int32); nr = np.zeros(n, np.int32); st = np.zeros(n, np.int32)
        hl = np.zeros(n); cnt = np.zeros(3, np.int64)
        self._L.cko_integrate(self.h, 0 if solver == "ros" else 1, C.c_longlong(n), _p(y), C.c_longlong(n), _p(p),
                            C.c_double(dt), C.c_double(rtol), C.c_double(atol), int(jac_mode), C.c_double(h0),
                            int(max_steps), _p(na, C.c_int), _p(nr, C.c_int), _p(st, C.c_int), _p(hl),
                            _p(cnt, C.c_longlong), int(nthreads))
        return dict(y=y, n_accept=na, n_reject=nr, status=st, h_last=hl, rhs_evals=int(cnt[0]),
                    jac_evals=int(cnt[1]), lu=int(cnt[2]))

    def estimate_h0(self, y1, p, dt, rtol=1e-6, atol=1e-10):
        y1 = _f64(y1)
        return float(self._L.cko_estimate_h0(self.h, _p(y1), C.c_double(p), C.c_double(dt), C.c_double(rtol), C.c_double(atol)))

    def rk4(self, y1, p, dt, nsteps):
        y1 = _f64(y1).copy()
        self._L.cko_rk4(self.h, _p(y1), C.c_double(p), C.c_double(dt), C.c_longlong(nsteps))
        return y1


def lu_factor(A):
    A = _f64(A).copy(); N = A.shape[0]
    piv = np.zeros(N, np.int32)
    rc = lib().cko_lu_factor(_p(A), _p(piv, C.c_int), N)
    return A, piv, rc


def lu_solve(LU, piv, b):
    b = _f64(b).copy()
    lib().cko_lu_solve(_p(_f64(LU)), _p(_i32(piv), C.c_int), LU.shape[0], _p(b))
    return b


def onestep_fixed(solver, problem, nsteps, y0, tend=1.0, lam=0.0):
    y0 = _f64(y0); N = y0.shape[0]
    out = np.zeros(2 * N + 1)
    lib().cko_onestep_fixed(0 if solver == "ros" else 1, int(problem), C.c_double(lam), C.c_double(tend), int(nsteps),
                            _p(y0), _p(out))
    return out[:N], out[N:2 * N], int(out[2 * N])


def toy_adaptive(solver, tend, rtol, atol, y0):
    y0 = _f64(y0); out = np.zeros(2); steps = np.zeros(3, np.int32)
    lib().cko_toy_adaptive(0 if solver == "ros" else 1, C.c_double(tend), C.c_double(rtol), C.c_double(atol), _p(y0),
                           _p(out), _p(steps, C.c_int))
    return out, steps


def tableaus():
    a = np.zeros((6, 6)); b = np.zeros(6); bh = np.zeros(6); ros = np.zeros(18)
    lib().cko_tableaus(_p(a), _p(b), _p(bh), _p(ros))
    return a, b, bh, ros


def max_threads():
    return int(lib().cko_max_threads())


def waste(attempts, P):
    """Eq. 20 written out: for each work unit j of P consecutive reactors (static linear mapping,
    PAPER.md:363), W_j = 1 - sum_i N_i / (P max_i N_i).  The ragged last unit divides by the lanes it has; a unit whose
    reactors took no step has W_j = 0 (the readings of include/ck.h).  Plain Python loop, float64.
    Pins (tests/test_oracle_waste.py): equal counts -> 0, one busy lane of P -> 1 - 1/P, counts 1..P ->
    1 - (P + 1) / (2 P), invariance under permutation inside a unit and under scaling of all counts, 0 <= W < 1."""
    a = [int(v) for v in np.asarray(attempts).ravel()]
    out = []
    for b in range(0, len(a), P):
        unit = a[b:b + P]
        mx = max(unit)
        out.append(1.0 - float(sum(unit)) / (float(len(unit)) * float(mx)) if mx > 0 else 0.0)
    return np.array(out, dtype=np.float64)


def waste_tasks(attempts, P, tasks):
    """Eq. 20 with `tasks` reactors per lane (the several-tasks-per-thread mitigation the paper cites from ref. [48],
    PAPER.md:419), written out: unit j = P * tasks consecutive reactors, lane l owns reactors l, l + P, l + 2P, ... of the
    unit, cost_l = sum of their attempts, W_j = 1 - sum_i N_i / (lanes * max_l cost_l), lanes = lanes owning >= 1 reactor.
    tasks = 1 is waste().  Pins (tests/test_oracle_waste.py): reduces to waste() at tasks = 1; equal counts -> 0;
    averaging: W(tasks) of iid counts falls as tasks grows; a unit made of `tasks` copies of one pattern has the W of
    that pattern."""
    a = [int(v) for v in np.asarray(attempts).ravel()]
    per = P * tasks
    out = []
    for b in range(0, len(a), per):
        unit = a[b:b + per]
        cost = [sum(unit[l::P]) for l in range(min(P, len(unit)))]
        mx = max(cost)
        out.append(1.0 - float(sum(unit)) / (float(len(cost)) * float(mx)) if mx > 0 else 0.0)
    return np.array(out, dtype=np.float64)
