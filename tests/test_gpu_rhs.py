"""GPU parity: ck_rhs (CUDA, through the C ABI) vs the CPU oracle on the same seeded inputs.

Bound (north_star: "relative error <= 1e-12 per component", read per DESIGN.md P1): |f_gpu - f_ref| <= 1e-12 * D
with f_ref the long-double oracle and D its cancellation-aware scale (sum of |terms|)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-12


def _gpu(mech_dict):
    import torch
    import paper_1608_05794_b200 as ck
    assert torch.cuda.is_available()
    return ck.Mechanism(mech_dict), torch


def _check(oracle, name, n, ld_pad=0):
    from synth_inputs import make_config
    mech, y, p, _ = make_config(name, n=n)
    M, torch = _gpu(mech)
    O = oracle.Mech(mech)
    yd = torch.zeros((y.shape[0], n + ld_pad), dtype=torch.float64, device="cuda")
    yd[:, :n] = torch.from_numpy(y)
    out = torch.full_like(yd, float("nan"))
    M.rhs(yd[:, :n], torch.from_numpy(p).cuda(), out=out[:, :n])
    torch.cuda.synchronize()
    f = out[:, :n].cpu().numpy()
    if ld_pad:
        assert torch.isnan(out[:, n:]).all()          # nothing written past n
    fref = O.rhs(y, p, prec=1, nthreads=8)
    _, D = O.rhs(y, p, want_scale=True, nthreads=8)
    err = np.abs(f - fref)
    assert np.isfinite(f).all()
    assert np.all(err <= TOL * D + 1e-300), float((err / (D + 1e-300)).max())
    rel = err / (np.abs(fref) + 1e-300)
    return np.median(rel), rel.max()


@pytest.mark.parametrize("name,n", [("C1", 1024), ("C1", 1), ("C1", 129), ("C2", 1000), ("C2", 4096 + 37), ("C5", 300),
                                    ("C5", 4096 + 19), ("C1", 2048 + 5)])
def test_rhs_matches_oracle(oracle, name, n):
    med, mx = _check(oracle, name, n)
    assert med < 1e-13


def test_rhs_padded_leading_dimension(oracle):
    _check(oracle, "C2", 1000, ld_pad=24)


def test_rhs_empty_batch():
    from synth_inputs.configs import get_mech
    M, torch = _gpu(get_mech("h2"))
    y = torch.zeros((10, 0), dtype=torch.float64, device="cuda")
    out = M.rhs(y, torch.zeros(0, dtype=torch.float64, device="cuda"))
    assert out.shape == (10, 0)


def test_rhs_full_size_sampled(oracle):
    """BASELINE config 2 at full size (1,048,576 states), in the launch configuration bench.py times;
    sampled columns are checked one by one against the oracle."""
    from synth_inputs import make_config
    mech, y, p, _ = make_config("C2")
    M, torch = _gpu(mech)
    yd = torch.from_numpy(y).cuda(); pd = torch.from_numpy(p).cuda()
    f = M.rhs(yd, pd).cpu().numpy()
    assert np.isfinite(f).all()
    idx = np.unique(np.concatenate([np.arange(0, 64), np.arange(y.shape[1] - 64, y.shape[1]),
                                    np.random.default_rng(5).integers(0, y.shape[1], 1024)]))
    O = oracle.Mech(mech)
    ys = np.ascontiguousarray(y[:, idx]); ps = np.ascontiguousarray(p[idx])
    fref = O.rhs(ys, ps, prec=1, nthreads=8)
    _, D = O.rhs(ys, ps, want_scale=True, nthreads=8)
    assert np.all(np.abs(f[:, idx] - fref) <= TOL * D + 1e-300)
    # property at any size: mass conservation sum_k Ydot_k = 0 within the cancellation scale
    assert np.all(np.abs(f[1:].sum(0)) <= 1e-9 * np.abs(f[1:]).sum(0) + 1e-6)


def test_rhs_host_entry_point(oracle):
    from synth_inputs import make_config
    mech, y, p, _ = make_config("C2", n=5000)
    M, torch = _gpu(mech)
    f = M.rhs_host(y, p)
    fd = M.rhs(torch.from_numpy(y).cuda(), torch.from_numpy(p).cuda()).cpu().numpy()
    assert np.array_equal(f, fd)


def test_rhs_temperature_outside_safe_window(oracle):
    """Warps holding a reactor outside the temperature window for which the packer bounded the exponentials'
    arguments (250..4500 K) take the range-checked path; exercised at a size that runs the tensor-memory kernel."""
    from synth_inputs import make_config
    mech, y, p, _ = make_config("C2", n=40000)
    y = y.copy()
    y[0, 5::64] = 205.0
    y[0, 37::64] = 4950.0
    M, torch = _gpu(mech)
    f = M.rhs(torch.from_numpy(y).cuda(), torch.from_numpy(p).cuda()).cpu().numpy()
    idx = np.unique(np.concatenate([np.arange(0, 192), np.arange(5, 40000, 640), np.arange(37, 40000, 640)]))
    O = oracle.Mech(mech)
    ys = np.ascontiguousarray(y[:, idx]); ps = np.ascontiguousarray(p[idx])
    fref = O.rhs(ys, ps, prec=1, nthreads=8)
    _, D = O.rhs(ys, ps, want_scale=True, nthreads=8)
    assert np.isfinite(f).all()
    assert np.all(np.abs(f[:, idx] - fref) <= TOL * D + 1e-300)
