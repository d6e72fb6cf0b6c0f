"""GPU parity for constant-volume reactors against the oracle's constant-volume mode:
ck_rhs (shared-memory and tensor-memory kernels), ck_jac (cooperative analytic, finite differences, thread-per-reactor
batched), ROS4 (fused kernel, batched rounds, FD Jacobian) and RKF45.  The `p` argument holds the density."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

R_U = 8.31446261815324e7


def _setup(cfgname, n, mechname=None):
    import torch
    import paper_1608_05794_b200 as ck
    from synth_inputs import make_config, states as S
    from synth_inputs.configs import get_mech
    if mechname is None:
        mech, y, p, cfg = make_config(cfgname, n=n)
    else:
        mech = get_mech(mechname)
        y, p = S.ignition_states(mech, n, 31, (900.0, 1900.0), p_range_atm=(1.0, 8.0))
        cfg = dict(dt=2e-6)
    rho = p / (R_U * y[0] * (y[1:] / mech["mol_wt"][:, None]).sum(0))
    return ck.Mechanism(mech, const_volume=True), mech, y, np.ascontiguousarray(rho), cfg, torch


@pytest.mark.parametrize("cfgname,n,mechname", [("C1", 700, None), ("C2", 3000, None), ("C2", 40000 + 13, None), ("C5", 4500, None),
                                                (None, 500, "rk20"), (None, 300, "c1irr")])
def test_rhs_constant_volume(oracle, cfgname, n, mechname):
    M, mech, y, rho, cfg, torch = _setup(cfgname, n, mechname)
    O = oracle.Mech(mech, const_volume=True)
    f = M.rhs(torch.from_numpy(y).cuda(), torch.from_numpy(rho).cuda()).cpu().numpy()
    idx = np.unique(np.concatenate([np.arange(min(n, 96)), np.arange(max(0, n - 96), n), np.random.default_rng(1).integers(0, n, 200)]))
    ys = np.ascontiguousarray(y[:, idx]); rs = np.ascontiguousarray(rho[idx])
    fref = O.rhs(ys, rs, prec=1, nthreads=8)
    _, D = O.rhs(ys, rs, want_scale=True, nthreads=8)
    assert np.isfinite(f).all()
    assert np.all(np.abs(f[:, idx] - fref) <= 1e-12 * D + 1e-300)
    # and it is NOT the constant-pressure answer for the temperature equation
    import paper_1608_05794_b200 as ck
    assert np.abs(f[0, idx] - oracle.Mech(mech).rhs(ys, rs * R_U * ys[0] * (ys[1:] / mech["mol_wt"][:, None]).sum(0))[0]).max() > 0


@pytest.mark.parametrize("cfgname,n,mechname,nchk", [("C1", 90, None, 8), ("C3", 40, None, 5), (None, 40, "rk14", 5), ("C5", 8, None, 2)])
def test_jac_constant_volume(oracle, cfgname, n, mechname, nchk):
    import paper_1608_05794_b200 as ck
    M, mech, y, rho, cfg, torch = _setup(cfgname, n, mechname)
    O = oracle.Mech(mech, const_volume=True)
    yd, rd = torch.from_numpy(y).cuda(), torch.from_numpy(rho).cuda()
    J = M.jac(yd, rd).cpu().numpy()
    Jb = M.jac_batched(yd, rd).cpu().numpy()
    Jf = M.jac(yd, rd, mode=ck.CK_JAC_FD, h=1e-8).cpu().numpy()
    for r in np.linspace(0, n - 1, nchk).astype(int):
        Jc = O.jac(y[:, r], rho[r], mode=0)
        _, Jm = O.jac(y[:, r], rho[r], mode=2)
        for name, G in (("cooperative", J), ("batched", Jb)):
            err = np.abs(G[:, :, r] - Jc)
            assert np.all(err <= 1e-12 * Jm + 1e-300), (name, int(r), float((err / (Jm + 1e-300)).max()),
                                                         np.unravel_index(np.argmax(err / (Jm + 1e-300)), err.shape))
        Jo = O.jac(y[:, r], rho[r], mode=1, h=1e-8)
        colscale = np.abs(Jm).max(axis=0, keepdims=True)
        major = np.abs(y[:, r]) > 1e-3
        assert np.all((np.abs(Jf[:, :, r] - Jo) <= 1e-5 * colscale)[:, major])


def _integrate(oracle, cfgname, n, solver, mechname=None, jac_mode=0, flags=0, dt=None):
    M, mech, y, rho, cfg, torch = _setup(cfgname, n, mechname)
    dt = dt or cfg["dt"]
    yd = torch.from_numpy(y).cuda()
    res = M.integrate(solver, yd, torch.from_numpy(rho).cuda(), dt, jac_mode=jac_mode, flags=flags)
    g = yd.cpu().numpy()
    ref = oracle.Mech(mech, const_volume=True).integrate(solver, y, rho, dt, jac_mode=jac_mode, nthreads=16)
    assert np.all(res["status"].cpu().numpy() == 0) and np.all(ref["status"] == 0)
    assert np.all(np.abs(g[0] - ref["y"][0]) <= 1e-5 * ref["y"][0])
    bad = np.abs(g[1:] - ref["y"][1:]) > np.maximum(1e-5 * np.abs(ref["y"][1:]), 1e-10)
    assert bad.mean() <= (1e-3 if (jac_mode or solver == "rkf45") else 0.0), int(bad.sum())
    na = res["n_accept"].cpu().numpy()
    assert np.all(np.abs(na - ref["n_accept"]) <= np.maximum(2 if jac_mode else 1, np.ceil(0.05 * ref["n_accept"])))
    return res["report"]


@pytest.mark.parametrize("cfgname,n,flags", [("C1", 400, 0), ("C3", 500, 4), ("C3", 500, 8), ("C5", 64, 8)])
def test_ros_constant_volume(oracle, cfgname, n, flags):
    rep = _integrate(oracle, cfgname, n, "ros", flags=flags)
    assert rep["rhs_evals"] == 2 * rep["attempts"] + rep["jac_evals"] + 2 * n   # f(y_n) comes with the Jacobian


def test_ros_fd_constant_volume(oracle):
    _integrate(oracle, "C1", 150, "ros", jac_mode=1)


@pytest.mark.parametrize("cfgname,n,dt", [("C1", 400, 2e-7), ("C4", 700, None)])
def test_rkf45_constant_volume(oracle, cfgname, n, dt):
    _integrate(oracle, cfgname, n, "rkf45", dt=dt)
