"""GPU parity: ck_jac vs the oracle.  Analytic mode is compared with the oracle's complex-step Jacobian (a
different derivation) under the cancellation-aware bound |J_gpu - J_ref| <= 1e-12 * Jmag (P1), with
Jmag the sum-of-absolute-terms magnitude from the oracle's forward-mode pass.  FD mode is compared with the
oracle's FD Jacobian at 1e-5 of the column scale (reading G12: FD noise forbids 1e-12)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _setup(name, n):
    import torch
    import paper_1608_05794_b200 as ck
    from synth_inputs import make_config
    mech, y, p, cfg = make_config(name, n=n)
    return ck.Mechanism(mech), mech, y, p, torch


@pytest.mark.parametrize("name,n,nchk", [("C1", 257, 32), ("C3", 96, 12), ("C2", 64, 8), ("C5", 12, 3)])
def test_jac_analytic_matches_complex_step(oracle, name, n, nchk):
    M, mech, y, p, torch = _setup(name, n)
    O = oracle.Mech(mech)
    J = M.jac(torch.from_numpy(y).cuda(), torch.from_numpy(p).cuda()).cpu().numpy()   # (N, N, n)
    assert np.isfinite(J).all()
    worst = 0.0
    for r in np.linspace(0, n - 1, nchk).astype(int):
        Jc = O.jac(y[:, r], p[r], mode=0)
        _, Jm = O.jac(y[:, r], p[r], mode=2)
        err = np.abs(J[:, :, r] - Jc)
        ratio = (err / (Jm + 1e-300)).max()
        worst = max(worst, ratio)
        assert np.all(err <= 1e-12 * Jm + 1e-300), (r, ratio, np.unravel_index(np.argmax(err / (Jm + 1e-300)), err.shape))
    print("worst |dJ|/Jmag", worst)


@pytest.mark.parametrize("name,n", [("C1", 40), ("C3", 10)])
def test_jac_fd_matches_oracle_fd(oracle, name, n):
    M, mech, y, p, torch = _setup(name, n)
    O = oracle.Mech(mech)
    import paper_1608_05794_b200 as ck
    h = 1e-8
    J = M.jac(torch.from_numpy(y).cuda(), torch.from_numpy(p).cuda(), mode=ck.CK_JAC_FD, h=h).cpu().numpy()
    for r in range(0, n, 3):
        Jf = O.jac(y[:, r], p[r], mode=1, h=h)
        _, Jm = O.jac(y[:, r], p[r], mode=2)
        colscale = np.abs(Jm).max(axis=0, keepdims=True)
        major = np.abs(y[:, r]) > 1e-3      # trace-species columns are rounding noise / sigma_j on both sides
        assert np.all((np.abs(J[:, :, r] - Jf) <= 1e-5 * colscale)[:, major])


def test_jac_empty_and_bad_mode():
    import torch
    import paper_1608_05794_b200 as ck
    from synth_inputs.configs import get_mech
    M = ck.Mechanism(get_mech("h2"))
    y = torch.zeros((10, 0), dtype=torch.float64, device="cuda")
    assert M.jac(y, torch.zeros(0, dtype=torch.float64, device="cuda")).shape == (10, 10, 0)
    y = torch.ones((10, 4), dtype=torch.float64, device="cuda")
    with pytest.raises(ck.CkError):
        M.jac(y, torch.ones(4, dtype=torch.float64, device="cuda"), mode=7)


@pytest.mark.parametrize("name,n,nchk", [("C3", 2048 + 77, 10), ("C5", 600, 4), ("C1", 1500, 10)])
def test_jac_batched_thread_per_reactor_matches_complex_step(oracle, name, n, nchk):
    """ck_jac_batched (one reactor per lane, one matrix row at a time in tensor memory; row 0 from the species rows
    through the differentiated enthalpy identity) against the oracle's complex-step Jacobian, and against ck_jac."""
    M, mech, y, p, torch = _setup(name, n)
    O = oracle.Mech(mech)
    yd, pd = torch.from_numpy(y).cuda(), torch.from_numpy(p).cuda()
    J = M.jac_batched(yd, pd).cpu().numpy()
    assert np.isfinite(J).all()
    for r in np.unique(np.concatenate([np.linspace(0, n - 1, nchk).astype(int), [n - 1, n - 2]])):
        Jc = O.jac(y[:, r], p[r], mode=0)
        _, Jm = O.jac(y[:, r], p[r], mode=2)
        err = np.abs(J[:, :, r] - Jc)
        assert np.all(err <= 1e-12 * Jm + 1e-300), (int(r), float((err / (Jm + 1e-300)).max()),
                                                     np.unravel_index(np.argmax(err / (Jm + 1e-300)), err.shape))
