"""Pins for the oracle on the reaction kinds the BASELINE recipes never draw:
irreversible rows, Lindemann rows, termolecular sides and nu = 2 (Eq. 14),
a species on both sides, three distinct NASA range breaks, more than six efficiencies.
Closed forms are typed out here from Eq. 12-18; invariants hold for any mechanism."""
import numpy as np
import pytest

from synth_inputs import states as S
from synth_inputs.configs import get_mech
from helpers import custom_mech, R_U, R_CAL, P_ATM


@pytest.fixture(scope="module", params=["h2co", "c1irr", "rk20", "rk14"])
def mech_pair(request, oracle):
    d = get_mech(request.param)
    return d, oracle.Mech(d)


def _states(d, n, seed=17):
    return S.ignition_states(d, n, seed, (900.0, 1900.0), p_range_atm=(1.0, 8.0))


def test_generated_mechanisms_hold_the_row_kinds():
    d = get_mech("rk20")
    t, rev = d["type"], d["reversible"]
    assert (t == 2).sum() >= 2 and (t == 3).sum() >= 1 and (t == 1).sum() >= 2
    assert 0 < rev.sum() < d["n_reactions"]
    order = lambda ptr, nu, i: int(nu[ptr[i]:ptr[i + 1]].sum())
    assert max(order(d["reac_ptr"], d["reac_nu"], i) for i in range(d["n_reactions"])) == 3
    assert d["reac_nu"].max() == 2 or d["prod_nu"].max() == 2
    both = [i for i in range(d["n_reactions"])
            if set(d["reac_spec"][d["reac_ptr"][i]:d["reac_ptr"][i + 1]]) & set(d["prod_spec"][d["prod_ptr"][i]:d["prod_ptr"][i + 1]])]
    assert len(both) >= 1
    assert np.diff(d["eff_ptr"]).max() >= 8 and len(np.unique(d["t_mid"])) == 3
    irr = get_mech("c1irr")
    assert irr["n_species"] == 53 and irr["n_reactions"] == 634 and irr["reversible"].sum() == 0
    h = get_mech("h2co")
    assert h["n_species"] == 14 and h["n_reactions"] == 38 and (h["type"] == 2).sum() == 1


def test_invariants_on_mixed_mechanisms(mech_pair):
    d, M = mech_pair
    y, p = _states(d, 48)
    f, D = M.rhs(y, p, want_scale=True)
    fl = M.rhs(y, p, prec=1)
    assert np.isfinite(f).all()
    assert np.all(np.abs(f - fl) <= 1e-12 * D + 1e-300)
    K = d["n_species"]
    scale = np.abs(D[1:]).sum(0) + 1e-300
    assert np.all(np.abs(f[1:].sum(0)) <= 1e-13 * scale)                       # mass
    wdot_over_rho = f[1:] / d["mol_wt"][:, None]
    for e in range(d["n_elements"]):                                           # elements
        n_e = d["elem_comp"][:, e].astype(float)
        ref = (n_e[:, None] * np.abs(D[1:]) / d["mol_wt"][:, None]).sum(0) + 1e-300
        assert np.all(np.abs(n_e @ wdot_over_rho) <= 1e-13 * ref)
    for r in range(0, 48, 5):                                                  # enthalpy identity (reading G2)
        T = y[0, r]
        th = np.array([M.thermo(k, T) for k in range(K)])
        hk = R_U * T * th[:, 1] / d["mol_wt"]
        cp = R_U * (y[1:, r] * th[:, 0] / d["mol_wt"]).sum()
        lhs = (f[1:, r] * hk).sum() + cp * f[0, r]
        assert abs(lhs) <= 1e-12 * ((np.abs(D[1:, r]) * np.abs(hk)).sum() + cp * D[0, r])


def test_thermo_continuity_at_every_range_break(oracle):
    d = get_mech("rk20")
    M = oracle.Mech(d)
    for k in range(d["n_species"]):
        tm = d["t_mid"][k]
        assert np.allclose(M.thermo(k, tm), M.thermo(k, np.nextafter(tm, 1e9)), rtol=1e-9, atol=1e-9)
        for T in (tm - 50.0, tm + 50.0):
            h = 1e-2
            cp = M.thermo(k, T)[0]
            dH = (M.thermo(k, T + h)[1] * (T + h) - M.thermo(k, T - h)[1] * (T - h)) / (2 * h)
            assert abs(dH - cp) < 1e-6 * abs(cp)


def test_equilibrium_on_mixed_mechanism_reversible_rows_balance_irreversible_rows_do_not(oracle):
    d = get_mech("rk20")
    M = oracle.Mech(d)
    K, E = d["n_species"], d["n_elements"]
    rng = np.random.default_rng(3)
    for T in (950.0, 1200.0, 2100.0):     # one temperature inside each of the three NASA interval patterns
        lam = rng.uniform(-12.0, -6.0, size=E)
        g = np.array([M.thermo(k, T)[1] - M.thermo(k, T)[2] for k in range(K)])
        C = (P_ATM / (R_U * T)) * np.exp(-g + d["elem_comp"] @ lam)
        rho = (C * d["mol_wt"]).sum()
        y1 = np.concatenate([[T], C * d["mol_wt"] / rho])
        qf, qr, _, _ = M.rates(y1, C.sum() * R_U * T)
        rev = d["reversible"].astype(bool)
        assert np.all(qf > 0)
        assert np.all(np.abs(qf - qr)[rev] <= 5e-13 * qf[rev])     # Eq. 16-18 with K_c from Gibbs energies
        assert np.all(qr[~rev] == 0.0)                             # k_r = 0


def test_closed_form_rates_termolecular_nu2_and_both_sides(oracle):
    """Eq. 14 typed out: q = k_f prod C^nu' - k_r prod C^nu''; K_c from Eq. 17-18 with constant cp."""
    W = [2.0, 16.0, 18.0, 20.0, 36.0]                 # E = A + C (18 + ... ) see below
    # species: 0 A (W 2), 1 B (16), 2 C = A + B (18), 3 D (20, inert collider), 4 E = 2 A + 2 B (36)
    elem = [[1, 0, 0], [0, 1, 0], [1, 1, 0], [0, 0, 1], [2, 2, 0]]
    a7 = [20.0, 25.0, 30.0, 22.0, 41.0]
    a6 = [0.0, 0.0, -12000.0, 0.0, -30000.0]
    nasa = [[3.5, 0, 0, 0, 0, a6[k], a7[k]] for k in range(5)]
    kA, kb, kE = 2.0e15, 0.5, 3000.0
    rx = [dict(reac={0: 2, 1: 1}, prod={0: 1, 2: 1}, A=kA, beta=kb, Ea=kE, rev=True),      # 2A + B <=> A + C
          dict(reac={0: 1, 1: 1, 2: 1}, prod={4: 1}, A=kA, beta=kb, Ea=kE, rev=True),      # A + B + C <=> E
          dict(reac={0: 1, 1: 1, 2: 1}, prod={4: 1}, A=kA, beta=kb, Ea=kE, rev=False)]     # same, irreversible
    d = custom_mech(W, nasa, rx, elem_comp=elem)
    M = oracle.Mech(d)
    T, p = 1350.0, 3.0 * P_ATM
    Y = np.array([0.05, 0.35, 0.2, 0.3, 0.1])
    Wn = np.array(W)
    rho = p / (R_U * T * (Y / Wn).sum())
    C = rho * Y / Wn
    kf = kA * T ** kb * np.exp(-kE / (R_CAL * T))
    # constant cp/R = 3.5 for all: g_k = H/RT - S/R = 3.5 + a6/T - 3.5 ln T - a7
    g = 3.5 + np.array(a6) / T - 3.5 * np.log(T) - np.array(a7)
    Kc1 = np.exp(-(g[0] + g[2] - 2 * g[0] - g[1])) * (P_ATM / (R_U * T)) ** (2 - 3)
    Kc2 = np.exp(-(g[4] - g[0] - g[1] - g[2])) * (P_ATM / (R_U * T)) ** (1 - 3)
    qf, qr, _, _ = M.rates(np.concatenate([[T], Y]), p)
    assert abs(qf[0] - kf * C[0] ** 2 * C[1]) < 1e-13 * qf[0]
    assert abs(qr[0] - kf / Kc1 * C[0] * C[2]) < 1e-12 * qr[0]
    assert abs(qf[1] - kf * C[0] * C[1] * C[2]) < 1e-13 * qf[1]
    assert abs(qr[1] - kf / Kc2 * C[4]) < 1e-12 * qr[1]
    assert qf[2] == qf[1] and qr[2] == 0.0
    # production rates: species 0 loses 2 and gains 1 in row 0
    f = M.rhs(np.concatenate([[T], Y])[:, None], np.array([p]))[:, 0]
    q = qf - qr
    w = np.array([-q[0] - q[1] - q[2], -q[0] - q[1] - q[2], q[0] - q[1] - q[2], 0.0, q[1] + q[2]])
    assert np.allclose(f[1:], w * Wn / rho, rtol=1e-11, atol=0.0)


def test_more_than_six_efficiencies_closed_form(oracle):
    K = 10
    W = [2.0, 30.0, 32.0] + [10.0 + k for k in range(7)]
    elem = [[1, 0, 0], [0, 1, 0], [1, 1, 0]] + [[0, 0, 1 + k] for k in range(7)]
    nasa = [[3.5, 0, 0, 0, 0, 0.0, 20.0 + k] for k in range(K)]
    eff = {k: 0.5 + k for k in range(1, 10)}            # nine non-unit efficiencies
    rx = [dict(reac={0: 1, 1: 1}, prod={2: 1}, A=1e12, rev=False, type=1, eff=eff)]
    M = oracle.Mech(custom_mech(W, nasa, rx, elem_comp=elem))
    T, p = 1100.0, 2.0 * P_ATM
    Y = np.linspace(1.0, 2.0, K); Y /= Y.sum()
    Wn = np.array(W)
    C = p / (R_U * T * (Y / Wn).sum()) * Y / Wn
    Mtb = C.sum() + sum((v - 1.0) * C[k] for k, v in eff.items())
    qf = M.rates(np.concatenate([[T], Y]), p)[0]
    assert abs(qf[0] - 1e12 * C[0] * C[1] * Mtb) < 1e-13 * qf[0]


def test_jacobian_on_mixed_mechanism_two_derivations_and_brute_force(oracle):
    d = get_mech("rk14")
    M = oracle.Mech(d)
    y, p = _states(d, 3)
    for r in range(2):
        y1 = y[:, r]
        Jc = M.jac(y1, p[r], mode=0)
        Jd, Jm = M.jac(y1, p[r], mode=2)
        assert np.all(np.abs(Jc - Jd) <= 1e-11 * Jm + 1e-300)
        N = y1.size
        Jb = np.zeros((N, N))
        for j in range(N):
            h = 1e-3 * y1[j] if j == 0 else 1e-3 * max(abs(y1[j]), 1e-2)
            def cd(hh):
                yp = np.repeat(y1[:, None], 2, axis=1); yp[j, 0] += hh; yp[j, 1] -= hh
                f = M.rhs(yp, np.array([p[r], p[r]]), prec=1)
                return (f[:, 0] - f[:, 1]) / (yp[j, 0] - yp[j, 1])
            Jb[:, j] = (4 * cd(h / 2) - cd(h)) / 3
        colscale = np.abs(Jm).max(axis=0, keepdims=True)
        assert np.all(np.abs(Jc - Jb) <= 2e-6 * Jm + 1e-9 * colscale)


def test_integrators_on_mixed_mechanisms_conserve_and_agree(oracle):
    """ROS4 (both Jacobians) and RKF45 on the row-kinds model: linear invariants conserved, and the two solvers agree
    at tolerance level (they share only the RHS)."""
    d = get_mech("rk14")
    M = oracle.Mech(d)
    y, p = _states(d, 16)
    dt = 2e-6
    a = M.integrate("ros", y, p, dt, nthreads=4)
    b = M.integrate("ros", y, p, dt, jac_mode=1, nthreads=4)
    c = M.integrate("rkf45", y, p, dt, nthreads=4)
    t = M.integrate("rkf45", y, p, dt, rtol=1e-10, atol=1e-14, nthreads=4)
    for r in (a, b, c):
        assert np.all(r["status"] == 0)
        assert np.all(np.abs(r["y"][1:].sum(0) - 1.0) < 1e-8)
        assert np.all(np.abs(r["y"][0] - t["y"][0]) <= 2e-5 * t["y"][0])
        assert np.all(np.abs(r["y"][1:] - t["y"][1:]) <= 1e-4 * np.abs(t["y"][1:]) + 1e-8)
    N = d["n_species"] + 1
    att = b["n_accept"] + b["n_reject"]
    assert b["rhs_evals"] == (N + 3) * att.sum() + 2 * 16      # N + 1 evaluations per FD Jacobian
