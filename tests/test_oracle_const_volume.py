"""Pins for the oracle's constant-volume reactor (rho constant, c_p -> c_v and h_k -> u_k
in Eq. 13).  Each is something thermodynamics fixes, not a retyping of the oracle: the species equations do not depend
on the closure (same concentrations => same Ydot as the constant-pressure reactor at the matching pressure), the
temperature equations of the two closures differ by the ratio (sum u_k w_k / c_v) / (sum h_k w_k / c_p), internal
energy is the conserved quantity (identically on f, to tolerance after integration), a Gibbs-consistent composition is
a fixed point, isomerisation with Delta U = 0 leaves T alone, and the pressure rises by the ideal-gas law."""
import numpy as np
import pytest

from synth_inputs import make_config, mech_decay
from synth_inputs.configs import get_mech
from helpers import R_U, P_ATM


def _rho(d, y, p):
    S = (y[1:] / d["mol_wt"][:, None]).sum(0)
    return p / (R_U * y[0] * S)


@pytest.mark.parametrize("name,cfg", [("h2", "C1"), ("c1", "C2"), ("rk20", None)])
def test_species_equations_match_constant_pressure_and_temperature_ratio(oracle, name, cfg):
    d = get_mech(name)
    if cfg:
        _, y, p, _ = make_config(cfg, n=24)
    else:
        from synth_inputs import states as S
        y, p = S.ignition_states(d, 24, 5, (900.0, 1900.0), p_range_atm=(1.0, 8.0))
    Mp, Mv = oracle.Mech(d), oracle.Mech(d, const_volume=True)
    rho = _rho(d, y, p)
    fp, Dp = Mp.rhs(y, p, want_scale=True)
    fv, Dv = Mv.rhs(y, rho, want_scale=True)
    assert np.all(np.abs(fv[1:] - fp[1:]) <= 1e-13 * Dp[1:] + 1e-300)        # same C_k => same Ydot_k
    K = d["n_species"]
    for r in range(0, 24, 5):
        T = y[0, r]
        th = np.array([Mp.thermo(k, T) for k in range(K)])
        W = d["mol_wt"]
        w = fp[1:, r] * rho[r] / W                                              # omega_k
        cp = R_U * (y[1:, r] * th[:, 0] / W).sum()
        cv = cp - R_U * (y[1:, r] / W).sum()
        hsum = (R_U * T * th[:, 1] * w).sum()
        usum = (R_U * T * (th[:, 1] - 1.0) * w).sum()
        assert abs(fv[0, r] - (-usum / (rho[r] * cv))) <= 1e-11 * Dv[0, r]
        # internal-energy identity: sum_k f_k u_k + c_v f_T = 0 (u_k mass units)
        uk = R_U * T * (th[:, 1] - 1.0) / W
        lhs = (fv[1:, r] * uk).sum() + cv * fv[0, r]
        assert abs(lhs) <= 1e-12 * ((np.abs(Dv[1:, r]) * np.abs(uk)).sum() + cv * Dv[0, r])
        # and the enthalpy identity does NOT hold for the constant-volume closure (the two closures differ)
        if abs(hsum) > 1e-6 * abs(usum) and abs(usum - hsum) > 1e-3 * abs(hsum):
            assert abs(fv[0, r] - fp[0, r]) > 1e-6 * abs(fp[0, r])


def test_equilibrium_fixed_point_constant_volume(oracle):
    d = get_mech("h2")
    M = oracle.Mech(d, const_volume=True)
    K, E = d["n_species"], d["n_elements"]
    rng = np.random.default_rng(3)
    for T in (1000.0, 1800.0):
        lam = rng.uniform(-12.0, -6.0, size=E)
        Mp = oracle.Mech(d)
        g = np.array([Mp.thermo(k, T)[1] - Mp.thermo(k, T)[2] for k in range(K)])
        C = (P_ATM / (R_U * T)) * np.exp(-g + d["elem_comp"] @ lam)
        rho = (C * d["mol_wt"]).sum()
        y = np.concatenate([[T], C * d["mol_wt"] / rho])[:, None]
        f, D = M.rhs(y, np.array([rho]), want_scale=True)
        assert np.all(np.abs(f[:, 0]) <= 1e-12 * D[:, 0] + 1e-300)
        r = M.integrate("ros", y, np.array([rho]), 1e-5)
        assert np.allclose(r["y"], y, rtol=1e-9, atol=1e-14)


def test_internal_energy_and_density_conserved_after_integration(oracle):
    d = get_mech("h2")
    _, y, p, cfg = make_config("C1", n=12)
    rho = _rho(d, y, p)
    M = oracle.Mech(d, const_volume=True)
    Mp = oracle.Mech(d)
    K, W = d["n_species"], d["mol_wt"]

    def energy(col):
        th = np.array([Mp.thermo(k, col[0]) for k in range(K)])
        return (col[1:] * R_U * col[0] * (th[:, 1] - 1.0) / W).sum()

    for solver in ("ros", "rkf45"):
        dt = 2e-6 if solver == "ros" else 2e-7
        r = M.integrate(solver, y, rho, dt, nthreads=4)
        rp = Mp.integrate(solver, y, p, dt, nthreads=4)
        assert np.all(r["status"] == 0)
        assert np.all(np.abs(r["y"][1:].sum(0) - 1.0) < 1e-9)
        for j in range(12):
            u0, u1 = energy(y[:, j]), energy(r["y"][:, j])
            scale = abs(u0) + R_U * y[0, j] / W.mean()
            assert abs(u1 - u0) <= 2e-5 * scale                     # conserved to tolerance (nonlinear invariant)
            # the constant-pressure reactor conserves enthalpy instead: its internal energy moves when T does
        moved = np.abs(r["y"][0] - y[0]) > 1.0
        if moved.any():   # heat release at constant volume raises T more than at constant pressure (c_v < c_p)
            dTv = (r["y"][0] - y[0])[moved]; dTp = (rp["y"][0] - y[0])[moved]
            assert np.all(np.abs(dTv) > np.abs(dTp))
        # pressure by the ideal-gas law at the fixed density
        Sn = (r["y"][1:] / W[:, None]).sum(0)
        pn = rho * R_U * r["y"][0] * Sn
        assert np.all(np.isfinite(pn)) and np.all(pn > 0)


def test_isomerisation_with_zero_energy_change_keeps_temperature(oracle):
    A = 2500.0
    d = mech_decay(A=A)
    M = oracle.Mech(d, const_volume=True)
    y = np.array([[1200.0], [0.8], [0.2]])
    rho = np.array([P_ATM / (R_U * 1200.0 * (1.0 / 2.016))])
    f = M.rhs(y, rho)
    assert np.allclose(f[1], -A * y[1], rtol=1e-14) and abs(f[0, 0]) < 1e-9 * A * 1200
    r = M.integrate("rkf45", y, rho, 4e-4)
    assert abs(r["y"][1, 0] - 0.8 * np.exp(-A * 4e-4)) < 2e-6
    assert abs(r["y"][0, 0] - 1200.0) < 1e-6
