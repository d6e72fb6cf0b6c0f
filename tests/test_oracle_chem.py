"""Pins for the oracle RHS and Jacobian (CPU only; SURVEY.md 8(c) "What pins the oracle").

Each test is something the paper / thermodynamics / calculus fixes, not a retyping of the oracle:
thermo identities (G1), conservation invariants incl. the enthalpy identity (G2), Gibbs-consistent
equilibrium fixed point (G10), closed-form rate for A->B (Eq. 12, 14, 15), falloff limits and the
centre of the Troe curve (G9), brute-force Jacobian by Richardson-extrapolated central differences.
"""
import numpy as np
import pytest

from synth_inputs import make_config, mech_decay
from synth_inputs.configs import get_mech
from helpers import abc_mech, R_U, R_CAL, P_ATM


@pytest.fixture(scope="module", params=["h2", "c1"])
def mech_pair(request, oracle):
    d = get_mech(request.param)
    return d, oracle.Mech(d)


def _states(name, n):
    cfg = {"h2": "C1", "c1": "C2", "c4": "C5"}[name]
    _, y, p, _ = make_config(cfg, n=n)
    return y, p


# ---- 4. thermo identities (pin reading G1 of the garbled Eq. 19) -------------------
def test_thermo_identities_and_continuity(mech_pair):
    d, M = mech_pair
    for k in range(0, d["n_species"], max(1, d["n_species"] // 9)):
        for T in (350.0, 800.0, 1400.0, 2600.0):
            h = 1e-2
            cp, hrt, s = M.thermo(k, T)
            Hp = M.thermo(k, T + h)[1] * (T + h); Hm = M.thermo(k, T - h)[1] * (T - h)
            Sp = M.thermo(k, T + h)[2]; Sm = M.thermo(k, T - h)[2]
            assert abs((Hp - Hm) / (2 * h) - cp) < 1e-6 * abs(cp)        # d(H/R)/dT = cp/R
            assert abs(T * (Sp - Sm) / (2 * h) - cp) < 1e-6 * abs(cp)    # T d(S/R)/dT = cp/R
        tm = d["t_mid"][k]
        lo = M.thermo(k, tm); hi = M.thermo(k, np.nextafter(tm, 1e9))
        assert np.allclose(lo, hi, rtol=1e-9, atol=1e-9)
        assert 2.5 - 1e-9 <= M.thermo(k, 1500.0)[0] <= 8.0 + 1e-9


# ---- 3. invariants on f for random states ------------------------------------------------------------
def test_rhs_invariants(mech_pair):
    d, M = mech_pair
    name = "h2" if d["n_species"] == 9 else "c1"
    y, p = _states(name, 64)
    f, D = M.rhs(y, p, want_scale=True)
    K = d["n_species"]
    # sum_k Ydot_k = 0 and element conservation (W_k are exact element sums)
    scale = np.abs(D[1:]).sum(0) + 1e-300
    assert np.all(np.abs(f[1:].sum(0)) <= 1e-13 * scale)
    wdot_over_rho = f[1:] / d["mol_wt"][:, None]
    for e in range(d["n_elements"]):
        n_e = d["elem_comp"][:, e].astype(float)
        tot = np.abs(n_e @ wdot_over_rho)
        ref = (n_e[:, None] * np.abs(D[1:]) / d["mol_wt"][:, None]).sum(0) + 1e-300
        assert np.all(tot <= 1e-13 * ref)
    # enthalpy identity (pins G2): sum_k f_k h_k + c_p f_T = 0, h_k = R_u T (H_k/RT)/W_k (mass units)
    for r in range(0, 64, 7):
        T = y[0, r]
        th = np.array([M.thermo(k, T) for k in range(K)])
        hk = R_U * T * th[:, 1] / d["mol_wt"]
        cp = R_U * (y[1:, r] * th[:, 0] / d["mol_wt"]).sum()
        lhs = (f[1:, r] * hk).sum() + cp * f[0, r]
        ref = (np.abs(D[1:, r]) * np.abs(hk)).sum() + cp * D[0, r]
        assert abs(lhs) <= 1e-12 * ref


def test_long_double_agrees_within_cancellation_scale(mech_pair):
    d, M = mech_pair
    name = "h2" if d["n_species"] == 9 else "c1"
    y, p = _states(name, 128)
    f, D = M.rhs(y, p, want_scale=True)
    fl = M.rhs(y, p, prec=1)
    assert np.all(np.abs(f - fl) <= 1e-12 * D + 1e-300)
    assert np.all(D >= np.abs(f) * (1 - 1e-12))


# ---- 2. equilibrium fixed point (pins G10: Delta nu sign, K_p = exp(-dg), and Eq. 16-18) ------------
def test_equilibrium_fixed_point(mech_pair):
    d, M = mech_pair
    K, E = d["n_species"], d["n_elements"]
    rng = np.random.default_rng(7)
    for T in (900.0, 1500.0, 2200.0):
        lam = rng.uniform(-12.0, -6.0, size=E)
        g = np.array([M.thermo(k, T)[1] - M.thermo(k, T)[2] for k in range(K)])
        C = (P_ATM / (R_U * T)) * np.exp(-g + d["elem_comp"] @ lam)
        # (a uniform rescale of C would break equilibrium unless dnu=0: the scale lives in lam)
        rho = (C * d["mol_wt"]).sum()
        Y = C * d["mol_wt"] / rho
        p = C.sum() * R_U * T
        y = np.concatenate([[T], Y])[:, None]
        f, D = M.rhs(y, np.array([p]), want_scale=True)
        qf, qr, _, _ = M.rates(y[:, 0], p)
        nz = qf > 0
        assert nz.sum() == d["n_reactions"]
        assert np.all(np.abs(qf - qr)[nz] <= 5e-13 * qf[nz])
        assert np.all(np.abs(f[:, 0]) <= 1e-12 * D[:, 0] + 1e-300)


# ---- 1. closed form: A -> B, beta=E=0, isomers => f_A = -A Y_A, f_B = +A Y_A, f_T = 0 ----------------
def test_first_order_decay_rhs(oracle):
    A = 1234.5
    M = oracle.Mech(mech_decay(A=A))
    y = np.array([[1300.0, 900.0], [0.7, 0.2], [0.3, 0.8]])
    f = M.rhs(y, np.array([P_ATM, 3 * P_ATM]))
    assert np.allclose(f[1], -A * y[1], rtol=1e-14)
    assert np.allclose(f[2], +A * y[1], rtol=1e-14)
    assert np.all(np.abs(f[0]) < 1e-9 * A * 1300)
    # reversible with K_c = exp(dS): f_A = -A (Y_A - Y_B / K_c)
    dS = 0.8
    M = oracle.Mech(mech_decay(A=A, reversible=True, dS=dS))
    f = M.rhs(y, np.array([P_ATM, 3 * P_ATM]))
    assert np.allclose(f[1], -A * (y[1] - y[2] * np.exp(-dS)), rtol=1e-13)


def test_arrhenius_and_density(oracle):
    # A + B -> C irreversible: qf = A T^b exp(-E/(R_cal T)) C_A C_B with C_k = p Y_k / (R_u T W_k sum(Y/W))
    A, b, Ea = 3.0e11, 0.7, 12000.0
    d = abc_mech(0, A=A, beta=b, Ea=Ea)
    M = oracle.Mech(d)
    T, p = 1250.0, 2.5 * P_ATM
    Y = np.array([0.1, 0.5, 0.15, 0.25])
    W = d["mol_wt"]
    rho = p / (R_U * T * (Y / W).sum())
    C = rho * Y / W
    qf, qr, rho_o, _ = M.rates(np.concatenate([[T], Y]), p)
    assert abs(rho_o - rho) < 1e-14 * rho
    assert qr[0] == 0.0
    assert abs(qf[0] - A * T ** b * np.exp(-Ea / (R_CAL * T)) * C[0] * C[1]) < 1e-13 * qf[0]
    f = M.rhs(np.concatenate([[T], Y])[:, None], np.array([p]))
    assert np.allclose(f[1:4, 0], np.array([-1, -1, 1]) * qf[0] * W[:3] / rho, rtol=1e-13)
    assert f[4, 0] == 0.0


# ---- G9: third-body and falloff ----------------------------------------------------------------------
def test_third_body_and_falloff_limits(oracle):
    T, p = 1400.0, 1.7 * P_ATM
    Y = np.array([0.1, 0.5, 0.15, 0.25])
    y1 = np.concatenate([[T], Y])
    base = oracle.Mech(abc_mech(0))
    q0 = base.rates(y1, p)[0][0]            # k_inf C_A C_B
    W = np.array([2.016, 31.998, 34.014, 28.014])
    rho = p / (R_U * T * (Y / W).sum()); C = rho * Y / W
    eff = {2: 6.0, 3: 0.5}
    Mtb = C.sum() + 5.0 * C[2] - 0.5 * C[3]
    # three-body: c_i = [M]
    q = oracle.Mech(abc_mech(1, eff=eff)).rates(y1, p)[0][0]
    assert abs(q - q0 * Mtb) < 1e-13 * q
    # Lindemann: k = k_inf Pr/(1+Pr), Pr = k0 M / k_inf
    for A0 in (1e10, 1e16, 1e22, 1e30):
        Pr = A0 * Mtb / 1e12
        q = oracle.Mech(abc_mech(2, eff=eff, A0=A0)).rates(y1, p)[0][0]
        assert abs(q - q0 * Pr / (1 + Pr)) < 1e-13 * q
    assert abs(oracle.Mech(abc_mech(2, eff=eff, A0=1e40)).rates(y1, p)[0][0] - q0) < 1e-12 * q0   # Pr -> inf
    # Troe with F_cent = 1 (a=1, T* = inf-like) => F = 1 => equals Lindemann
    qT = oracle.Mech(abc_mech(3, eff=eff, A0=1e16, troe=[1.0, 100.0, 1e30, -1.0])).rates(y1, p)[0][0]
    qL = oracle.Mech(abc_mech(2, eff=eff, A0=1e16)).rates(y1, p)[0][0]
    assert abs(qT - qL) < 1e-12 * qL
    # centre of the Troe curve: log10 Pr = -c = 0.4 + 0.67 log10 F_cent  =>  f1 = 0  =>  F = F_cent
    a, T3, T1, T2 = 0.6, 200.0, 1800.0, 5000.0
    Fc = (1 - a) * np.exp(-T / T3) + a * np.exp(-T / T1) + np.exp(-T2 / T)
    Pr = 10.0 ** (0.4 + 0.67 * np.log10(Fc))
    A0 = Pr * 1e12 / Mtb
    q = oracle.Mech(abc_mech(3, eff=eff, A0=A0, troe=[a, T3, T1, T2])).rates(y1, p)[0][0]
    assert abs(q - q0 * Pr / (1 + Pr) * Fc) < 1e-12 * q
    # away from the centre F approaches 1 (f1^2 large) and never leaves [F_cent, 1]
    Fc2 = (1 - a) * np.exp(-T / T3) + a * np.exp(-T / T1)
    for A0 in (1e17, 1e20, 1e24, 1e30, 1e40):
        Pr = A0 * Mtb / 1e12
        q = oracle.Mech(abc_mech(3, eff=eff, A0=A0, troe=[a, T3, T1, -1.0])).rates(y1, p)[0][0]
        F = q / (q0 * Pr / (1 + Pr))
        assert Fc2 < F < 1.0 and (A0 < 1e24 or F > 0.9)


# ---- 6. Jacobian: complex step vs brute-force central differences (Richardson) ------------------------
def _brute_jac(M, y1, p):
    N = y1.size
    J = np.zeros((N, N))
    for j in range(N):
        h = 1e-3 * y1[j] if j == 0 else 1e-3 * max(abs(y1[j]), 1e-2)
        def cd(hh):
            yp = np.repeat(y1[:, None], 2, axis=1); yp[j, 0] += hh; yp[j, 1] -= hh
            hh_eff = (yp[j, 0] - yp[j, 1]) / 2
            f = M.rhs(yp, np.array([p, p]), prec=1)
            return (f[:, 0] - f[:, 1]) / (2 * hh_eff)
        d1, d2 = cd(h), cd(h / 2)
        J[:, j] = (4 * d2 - d1) / 3
    return J


def test_jacobian_complex_step_vs_brute_force(mech_pair):
    d, M = mech_pair
    name = "h2" if d["n_species"] == 9 else "c1"
    y, p = _states(name, 4)
    for r in range(2):
        Jc = M.jac(y[:, r], p[r], mode=0)
        Jd, Jm = M.jac(y[:, r], p[r], mode=2)
        Jb = _brute_jac(M, y[:, r], p[r])
        assert np.all(np.abs(Jc - Jd) <= 1e-11 * Jm + 1e-300)           # two derivations agree to rounding
        colscale = np.abs(Jm).max(axis=0, keepdims=True)
        assert np.all(np.abs(Jc - Jb) <= 2e-6 * Jm + 1e-9 * colscale)    # and match brute force
        # linear invariants w.f = 0 for all y  =>  w.J = 0
        w = d["mol_wt"] * 0 + 1.0
        assert np.all(np.abs(w @ Jc[1:, :]) <= 1e-11 * (np.abs(Jm[1:, :])).sum(0))


def test_fd_jacobian_close_to_complex_step(mech_pair):
    d, M = mech_pair
    name = "h2" if d["n_species"] == 9 else "c1"
    y, p = _states(name, 2)
    Jc, Jm = M.jac(y[:, 0], p[0], mode=2)
    Jf = M.jac(y[:, 0], p[0], mode=1, h=1e-8)
    colscale = np.abs(Jm).max(axis=0, keepdims=True)
    # first-order differences with sigma_j ~ sqrt(eps)|y_j| are rounding-noise dominated for trace species
    # (noise eps*D_i/sigma_j, reading G12), so the pin is on the columns of T and of the major species
    major = np.abs(y[:, 0]) > 1e-3
    assert major.sum() >= 3
    assert np.all((np.abs(Jf - Jc) <= 1e-4 * colscale + 1e-6 * Jm)[:, major])
