"""GPU parity on the input kinds include/ck.h accepts but BASELINE's five recipes never draw (VERDICT r1 "What's
missing" #6, "weak" #3): Lindemann rows and third-body rows with more than six efficiencies
(PAPER.md:113), irreversible rows, termolecular sides, nu = 2 and a species on both sides (Eq. 14,
PAPER.md:111), three distinct NASA range breaks, the model sizes K = 14 (N = 15), K = 20 (generic
N <= 32 path), K = 130 (N > 128 path), Table 1's H2/CO-sized 14/38 model and a 53-species / 634-irreversible-row model
(PAPER.md:149, 271-279).  Every call goes through the C ABI; bounds are north_star's (P1, P2)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

MECHS = ["rk14", "rk20", "h2co", "c1irr", "rk130"]


def _setup(name, n, seed=23):
    import torch
    import paper_1608_05794_b200 as ck
    from synth_inputs import states as S
    from synth_inputs.configs import get_mech
    mech = get_mech(name)
    y, p = S.ignition_states(mech, n, seed, (900.0, 1900.0), p_range_atm=(1.0, 8.0))
    return ck.Mechanism(mech), mech, y, p, torch


def _rhs_check(oracle, M, mech, y, p, torch, idx=None):
    f = M.rhs(torch.from_numpy(y).cuda(), torch.from_numpy(p).cuda()).cpu().numpy()
    assert np.isfinite(f).all()
    if idx is None:
        idx = np.arange(y.shape[1])
    O = oracle.Mech(mech)
    ys = np.ascontiguousarray(y[:, idx]); ps = np.ascontiguousarray(p[idx])
    fref = O.rhs(ys, ps, prec=1, nthreads=8)
    _, D = O.rhs(ys, ps, want_scale=True, nthreads=8)
    err = np.abs(f[:, idx] - fref)
    assert np.all(err <= 1e-12 * D + 1e-300), float((err / (D + 1e-300)).max())


@pytest.mark.parametrize("name", MECHS)
def test_rhs_small_batch(oracle, name):
    M, mech, y, p, torch = _setup(name, 333)
    _rhs_check(oracle, M, mech, y, p, torch)


@pytest.mark.parametrize("name", ["rk14", "rk20", "h2co", "c1irr"])
def test_rhs_large_batch_tensor_memory_kernel(oracle, name):
    """n >= 37,888 selects the tensor-memory kernel for K + 1 <= 64; sampled columns against the oracle."""
    n = 40000 + 77
    M, mech, y, p, torch = _setup(name, n)
    y = y.copy()
    y[0, 3::97] = 230.0        # a few warps outside the bounded-exponent window: the range-checked path
    idx = np.unique(np.concatenate([np.arange(96), np.arange(n - 96, n), np.arange(3, n, 970),
                                    np.random.default_rng(2).integers(0, n, 400)]))
    _rhs_check(oracle, M, mech, y, p, torch, idx)


@pytest.mark.parametrize("name,n,nchk", [("rk14", 65, 9), ("rk20", 40, 6), ("h2co", 40, 6), ("c1irr", 24, 4), ("rk130", 6, 2)])
def test_jac_both_modes(oracle, name, n, nchk):
    import paper_1608_05794_b200 as ck
    M, mech, y, p, torch = _setup(name, n)
    O = oracle.Mech(mech)
    yd, pd = torch.from_numpy(y).cuda(), torch.from_numpy(p).cuda()
    J = M.jac(yd, pd).cpu().numpy()
    h = 1e-8
    Jf = M.jac(yd, pd, mode=ck.CK_JAC_FD, h=h).cpu().numpy()
    assert np.isfinite(J).all() and np.isfinite(Jf).all()
    for r in np.linspace(0, n - 1, nchk).astype(int):
        Jc = O.jac(y[:, r], p[r], mode=0)
        _, Jm = O.jac(y[:, r], p[r], mode=2)
        err = np.abs(J[:, :, r] - Jc)
        assert np.all(err <= 1e-12 * Jm + 1e-300), (int(r), float((err / (Jm + 1e-300)).max()))
        Jo = O.jac(y[:, r], p[r], mode=1, h=h)
        colscale = np.abs(Jm).max(axis=0, keepdims=True)
        major = np.abs(y[:, r]) > 1e-3
        assert np.all((np.abs(Jf[:, :, r] - Jo) <= 1e-5 * colscale)[:, major])


@pytest.mark.parametrize("name,n,nchk", [("rk14", 700, 6), ("rk20", 700, 6), ("h2co", 700, 5), ("c1irr", 600, 4)])
def test_jac_batched(oracle, name, n, nchk):
    M, mech, y, p, torch = _setup(name, n)
    O = oracle.Mech(mech)
    J = M.jac_batched(torch.from_numpy(y).cuda(), torch.from_numpy(p).cuda()).cpu().numpy()
    assert np.isfinite(J).all()
    for r in np.linspace(0, n - 1, nchk).astype(int):
        Jc = O.jac(y[:, r], p[r], mode=0)
        _, Jm = O.jac(y[:, r], p[r], mode=2)
        err = np.abs(J[:, :, r] - Jc)
        assert np.all(err <= 1e-12 * Jm + 1e-300), (int(r), float((err / (Jm + 1e-300)).max()))


def _integrate_check(oracle, name, n, solver, dt, jac_mode=0, flags=0):
    M, mech, y, p, torch = _setup(name, n)
    yd = torch.from_numpy(y).cuda()
    res = M.integrate(solver, yd, torch.from_numpy(p).cuda(), dt, jac_mode=jac_mode, flags=flags)
    torch.cuda.synchronize()
    g = yd.cpu().numpy()
    ref = oracle.Mech(mech).integrate(solver, y, p, dt, jac_mode=jac_mode, nthreads=16)
    st = res["status"].cpu().numpy()
    assert np.array_equal(st, ref["status"]) and np.all(st == 0)
    assert np.all(np.abs(g[0] - ref["y"][0]) <= 1e-5 * ref["y"][0])
    bad = np.abs(g[1:] - ref["y"][1:]) > np.maximum(1e-5 * np.abs(ref["y"][1:]), 1e-10)
    if jac_mode == 0:
        assert not bad.any(), int(bad.sum())
    elif bad.any():   # FD Jacobian: columns carry rounding noise (reading G12); P3 against a tight analytic solve
        assert bad.mean() <= 1e-3, float(bad.mean())
        rs = np.unique(np.where(bad)[1])
        print("P3 fallback:", int(bad.sum()), "of", bad.size, "entries in", len(rs), "reactors")
        t = oracle.Mech(mech).integrate(solver, np.ascontiguousarray(y[:, rs]), np.ascontiguousarray(p[rs]), dt, rtol=1e-9,
                                        atol=1e-13, nthreads=16)
        for i, r in enumerate(rs):
            col = t["y"][:, i]
            sc = 1e-6 * np.abs(col) + 1e-10
            e_gpu = np.sqrt(np.mean(((g[:, r] - col) / sc) ** 2))
            e_cpu = np.sqrt(np.mean(((ref["y"][:, r] - col) / sc) ** 2))
            lit = np.all(np.abs(g[:, r] - col) <= np.maximum(1e-5 * np.abs(col), np.where(np.arange(col.size) == 0, 0.0, 1e-10)))
            assert lit or e_gpu <= max(2.0 * e_cpu + 1.0, 10.0), (int(r), float(e_gpu), float(e_cpu))
    att = ref["n_accept"] + ref["n_reject"]
    # FD Jacobian: the two CPU builds of the oracle already differ by 2 accepted / 6 rejected attempts per reactor
    # (tests/test_oracle_p3.py), so that is the slack granted here; analytic Jacobian: 1
    slack = {"n_accept": 2 if jac_mode else 1, "n_reject": 6 if jac_mode else 1}
    for key in ("n_accept", "n_reject"):                    # DESIGN.md P2, applied to rejected attempts too
        a, b = res[key].cpu().numpy(), ref[key]
        lim = np.maximum(slack[key], np.ceil(0.05 * (b if key == "n_accept" else att)))
        assert np.all(np.abs(a - b) <= lim), (key, int(np.abs(a - b).max()))
    rep = res["report"]
    N = mech["n_species"] + 1
    per = {("ros", 0): 3, ("ros", 1): N + 3, ("rkf45", 0): 6}[(solver, jac_mode)]
    if solver == "ros" and jac_mode == 0:   # f(y_n) comes with the Jacobian, which the batched rounds keep across a rejected attempt
        assert rep["rhs_evals"] == 2 * rep["attempts"] + rep["jac_evals"] + 2 * n and rep["accepted"] <= rep["jac_evals"] <= rep["attempts"]
    else:
        assert rep["rhs_evals"] == per * rep["attempts"] + 2 * n
    assert rep["rhs_evals"] <= ref["rhs_evals"] or abs(rep["attempts"] - int((ref["n_accept"] + ref["n_reject"]).sum())) <= 0.05 * rep["attempts"]
    return rep


@pytest.mark.parametrize("name,n,dt", [("rk14", 300, 5e-6), ("rk20", 300, 2e-5), ("h2co", 300, 1e-5), ("c1irr", 200, 1e-6),
                                       ("rk130", 24, 1e-6)])
def test_ros_analytic(oracle, name, n, dt):
    _integrate_check(oracle, name, n, "ros", dt)


@pytest.mark.parametrize("name,n,dt", [("rk14", 600, 5e-6), ("rk20", 600, 2e-5), ("h2co", 600, 1e-5), ("c1irr", 400, 1e-6)])
def test_ros_batched_rounds(oracle, name, n, dt):
    """flags bit 3: the batched-rounds driver (thread-per-reactor chemistry, cooperative LU) on small batches."""
    rep = _integrate_check(oracle, name, n, "ros", dt, flags=8)
    assert rep["rounds"] >= 2


@pytest.mark.parametrize("name,n,dt", [("rk14", 150, 5e-6), ("rk20", 150, 2e-5), ("c1irr", 64, 1e-6), ("rk130", 8, 1e-6)])
def test_ros_fd_jacobian(oracle, name, n, dt):
    _integrate_check(oracle, name, n, "ros", dt, jac_mode=1)


@pytest.mark.parametrize("name,n,dt", [("rk14", 500, 1e-6), ("rk20", 500, 5e-6), ("h2co", 500, 1e-6), ("c1irr", 300, 1e-7),
                                       ("rk130", 64, 1e-7)])
def test_rkf45(oracle, name, n, dt):
    _integrate_check(oracle, name, n, "rkf45", dt)
