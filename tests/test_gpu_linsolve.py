"""GPU parity of the batched dense LU + solve against the oracle's textbook LU
with partial pivoting, on its own (the ROS4 tests cover it only end to end): random well- and ill-conditioned
matrices, matrices that force row exchanges at every step, sizes spanning one to four rows per lane and ragged
panels, a singular matrix.  Bound: the solution of a backward-stable factorisation, |x - x_ref| <= c N eps cond |x|
(DESIGN.md), checked through the residual and against the oracle's solution."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("N", [1, 3, 8, 10, 15, 16, 17, 33, 54, 64, 65, 112, 128])
def test_lu_solve_batched_matches_oracle(oracle, N):
    import torch
    import paper_1608_05794_b200 as ck
    rng = np.random.default_rng(100 + N)
    n = 40
    A = rng.standard_normal((n, N, N))
    A[: n // 4] += 5.0 * np.eye(N)                       # diagonally dominant: no exchanges
    for r in range(n // 4, n // 2):                      # reversed dominance: an exchange at every step
        A[r] = A[r][::-1].copy() + 5.0 * np.eye(N)[::-1]
    A[n // 2: 3 * n // 4] *= 10.0 ** rng.uniform(-6, 6, size=(3 * n // 4 - n // 2, 1, N))   # badly scaled columns
    b = rng.standard_normal((n, N))
    x, st = ck.lu_solve_batched(torch.from_numpy(A).cuda(), torch.from_numpy(b).cuda())
    x = x.cpu().numpy()
    assert np.all(st.cpu().numpy() == 0) and np.isfinite(x).all()
    eps = np.finfo(float).eps
    for r in range(n):
        LU, piv, rc = oracle.lu_factor(A[r])
        xo = oracle.lu_solve(LU, piv, b[r])
        res = np.abs(A[r] @ x[r] - b[r]).max()
        scale = (np.abs(A[r]) @ np.abs(x[r])).max() + np.abs(b[r]).max()
        assert res <= 50 * N * eps * scale, (r, res, scale)                    # backward stable
        cond = np.linalg.cond(A[r])
        assert np.abs(x[r] - xo).max() <= 100 * N * eps * cond * np.abs(xo).max() + 1e-300, (r, cond)


def test_lu_solve_batched_pivot_choice_and_singular(oracle):
    """The pivot rule decides an integer: on a matrix whose column maxima are unique the solution must agree with the
    oracle's to rounding of the SAME factorisation (1e-13), and a singular matrix must be flagged."""
    import torch
    import paper_1608_05794_b200 as ck
    N = 54
    rng = np.random.default_rng(7)
    A = rng.uniform(-1, 1, size=(8, N, N))
    b = rng.uniform(-1, 1, size=(8, N))
    A[7, :, 5] = 0.0                                      # singular: zero column
    x, st = ck.lu_solve_batched(torch.from_numpy(A).cuda(), torch.from_numpy(b).cuda())
    st = st.cpu().numpy(); x = x.cpu().numpy()
    assert np.all(st[:7] == 0) and st[7] == 4
    for r in range(7):
        LU, piv, _ = oracle.lu_factor(A[r])
        xo = oracle.lu_solve(LU, piv, b[r])
        assert np.abs(x[r] - xo).max() <= 1e-9 * np.abs(xo).max()
    x0, _ = ck.lu_solve_batched(torch.zeros((0, N, N), dtype=torch.float64, device="cuda"),
                                torch.zeros((0, N), dtype=torch.float64, device="cuda"))
    assert x0.shape == (0, N)
