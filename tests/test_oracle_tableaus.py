"""Pins for the oracle's coefficient tables and OneStep functions (CPU only).

RKF45: Table B.2 -- exact-rational row sums and order conditions (reading G3).
ROS4:  Table C.3 -- convergence order 4 with gamma=0.57282 (G4), the printed
"b_i" used as the m_i of Eq. 7 (G5), linear test equation, 3 RHS evaluations per attempt (G6).
"""
import os
from fractions import Fraction as Fr

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_rationals(path):
    out = {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        t = line.split()
        out[t[0]] = Fr(int(t[1]), int(t[2]))
    return out


def _read_floats(path):
    out = {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        t = line.split()
        out[t[0]] = float(t[1])
    return out


def _rkf_golden():
    g = _read_rationals(os.path.join(GOLD, "rkf45_table_b2.txt"))
    a = [[Fr(0)] * 6 for _ in range(6)]
    for i in range(2, 7):
        for j in range(1, i):
            a[i - 1][j - 1] = g[f"a{i}{j}"]
    c = [Fr(0)] + [g[f"c{i}"] for i in range(2, 7)]
    b = [g[f"b{i}"] for i in range(1, 7)]
    bh = [g[f"bh{i}"] for i in range(1, 7)]
    return g, a, c, b, bh


def test_rkf45_oracle_uses_golden_table(oracle):
    _, a, c, b, bh = _rkf_golden()
    A, B, BH, _ = oracle.tableaus()
    for i in range(6):
        for j in range(6):
            assert A[i, j] == float(a[i][j]) or abs(A[i, j] - float(a[i][j])) <= 2e-16 * abs(float(a[i][j]))
        assert abs(B[i] - float(b[i])) <= 1e-16 and abs(BH[i] - float(bh[i])) <= 1e-16


def test_rkf45_row_sums_and_printed_a42_is_garbled():
    g, a, c, _, _ = _rkf_golden()
    for i in range(6):
        assert sum(a[i]) == c[i]
    # the cell as printed breaks the row-sum condition -> repaired reading G3
    assert g["a41"] + g["a42_printed"] + g["a43"] != c[3]


def _order_conditions(a, c, w, upto):
    """Exact residuals of the rooted-tree order conditions up to order `upto` for weights w."""
    s = range(6)
    Ac = [sum(a[i][j] * c[j] for j in s) for i in s]
    Ac2 = [sum(a[i][j] * c[j] ** 2 for j in s) for i in s]
    AAc = [sum(a[i][j] * Ac[j] for j in s) for i in s]
    res = {
        "1": sum(w) - 1,
        "2": sum(w[i] * c[i] for i in s) - Fr(1, 2),
        "3a": sum(w[i] * c[i] ** 2 for i in s) - Fr(1, 3),
        "3b": sum(w[i] * Ac[i] for i in s) - Fr(1, 6),
        "4a": sum(w[i] * c[i] ** 3 for i in s) - Fr(1, 4),
        "4b": sum(w[i] * c[i] * Ac[i] for i in s) - Fr(1, 8),
        "4c": sum(w[i] * Ac2[i] for i in s) - Fr(1, 12),
        "4d": sum(w[i] * AAc[i] for i in s) - Fr(1, 24),
    }
    if upto >= 5:
        Ac3 = [sum(a[i][j] * c[j] ** 3 for j in s) for i in s]
        AcAc = [sum(a[i][j] * c[j] * Ac[j] for j in s) for i in s]
        AAc2 = [sum(a[i][j] * Ac2[j] for j in s) for i in s]
        AAAc = [sum(a[i][j] * AAc[j] for j in s) for i in s]
        res.update({
            "5a": sum(w[i] * c[i] ** 4 for i in s) - Fr(1, 5),
            "5b": sum(w[i] * c[i] ** 2 * Ac[i] for i in s) - Fr(1, 10),
            "5c": sum(w[i] * Ac[i] ** 2 for i in s) - Fr(1, 20),
            "5d": sum(w[i] * c[i] * Ac2[i] for i in s) - Fr(1, 15),
            "5e": sum(w[i] * Ac3[i] for i in s) - Fr(1, 20),
            "5f": sum(w[i] * c[i] * AAc[i] for i in s) - Fr(1, 30),
            "5g": sum(w[i] * AcAc[i] for i in s) - Fr(1, 40),
            "5h": sum(w[i] * AAc2[i] for i in s) - Fr(1, 60),
            "5i": sum(w[i] * AAAc[i] for i in s) - Fr(1, 120),
        })
    return res


def test_rkf45_order_conditions_exact():
    _, a, c, b, bh = _rkf_golden()
    r4 = _order_conditions(a, c, b, 5)
    for k in ("1", "2", "3a", "3b", "4a", "4b", "4c", "4d"):
        assert r4[k] == 0, k
    assert r4["5a"] == Fr(-1, 2080)  # the advanced solution is 4th order only
    r5 = _order_conditions(a, c, bh, 5)
    assert all(v == 0 for v in r5.values()), r5
    assert b[5] == 0  # 4th-order solution uses five stages ("five-stage, fourth-order")


def test_ros4_oracle_uses_golden_table(oracle):
    g = _read_floats(os.path.join(GOLD, "ros4_table_c3.txt"))
    _, _, _, ros = oracle.tableaus()
    names = ["gamma", "a21", "a31", "a32", "c21", "c31", "c32", "c41", "c42", "c43", "m1", "m2", "m3", "m4",
             "E1", "E2", "E3", "E4"]
    for v, n in zip(ros, names):
        assert v == g[n], n


# reference solution of the toy problem y1'=-y1 y2, y2'=y1 y2 - y2/2 from (1, 1) over [0,1]:
# a 30-term Taylor series integration in exact-ish arithmetic (mpmath), independent of the oracle.
def _toy_reference():
    import mpmath as mp
    mp.mp.dps = 40
    y = [mp.mpf(1), mp.mpf(1)]
    nseg, order = 64, 30
    h = mp.mpf(1) / nseg
    for _ in range(nseg):
        a = [y[0]]; b = [y[1]]
        for n in range(order):
            conv = sum(a[i] * b[n - i] for i in range(n + 1))
            a.append(-conv / (n + 1))
            b.append((conv - b[n] / 2) / (n + 1))
        y = [sum(a[n] * h ** n for n in range(order + 1)), sum(b[n] * h ** n for n in range(order + 1))]
    return np.array([float(y[0]), float(y[1])])


@pytest.mark.parametrize("solver,lo", [("ros", 3.8), ("rkf45", 3.8)])
def test_onestep_convergence_order(oracle, solver, lo):
    ref = _toy_reference()
    errs = []
    for n in (10, 20, 40, 80):
        y, _, _ = oracle.onestep_fixed(solver, 0, n, [1.0, 1.0])
        errs.append(np.abs(y - ref).max())
    orders = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert np.all(orders > lo) and np.all(orders < 5.4), (errs, orders)


def test_ros4_error_estimator_order_and_rhs_count(oracle):
    e = []
    for n in (10, 20, 40):
        _, est, nrhs = oracle.onestep_fixed("ros", 0, n, [1.0, 1.0])
        e.append(np.abs(est).max())
        assert nrhs == 3 * n  # stage 4 reuses stage 3's evaluation (G6)
    o = np.log2(np.array(e[:-1]) / np.array(e[1:]))
    assert np.all(o > 3.5) and np.all(o < 4.6), o
    _, _, nrhs = oracle.onestep_fixed("rkf45", 0, 7, [1.0, 1.0])
    assert nrhs == 6 * 7


def test_ros4_linear_test_equation(oracle):
    # one step on y'=lam y: y* - exp(h lam) = O(h^5); and L-stability: R(-inf) ~ 0
    d = []
    for h in (0.2, 0.1, 0.05):
        y, _, _ = oracle.onestep_fixed("ros", 1, 1, [1.0], tend=h, lam=-1.0)
        d.append(abs(y[0] - np.exp(-h)))
    o = np.log2(np.array(d[:-1]) / np.array(d[1:]))
    assert np.all(o > 4.6) and np.all(o < 5.5), (d, o)
    y, _, _ = oracle.onestep_fixed("ros", 1, 1, [1.0], tend=1.0, lam=-1e9)
    assert abs(y[0]) < 1e-3


def test_adaptive_driver_error_scales_with_tolerance(oracle):
    ref = _toy_reference()
    for solver in ("ros", "rkf45"):
        errs = []
        for tol in (1e-4, 1e-6, 1e-8):
            y, steps = oracle.toy_adaptive(solver, 1.0, tol, tol * 1e-2, [1.0, 1.0])
            assert steps[2] == 0
            errs.append(np.abs(y - ref).max())
        assert errs[0] < 1e-3 and errs[1] < 1e-5 and errs[2] < 1e-7, errs
        assert errs[2] < errs[1] < errs[0]
