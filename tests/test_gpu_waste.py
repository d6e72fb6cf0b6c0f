"""GPU parity: ck_waste (Eq. 20) vs the oracle's written-out definition.  The kernel and the oracle
evaluate 1 - sum / (lanes * max) with the same IEEE operations on exact integers, so the comparison is bit-exact."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("P", [1, 4, 8, 16, 32, 64, 1000])
@pytest.mark.parametrize("n", [1, 31, 1601, 65536 + 17])
def test_waste_matches_oracle_bit_exact(oracle, P, n):
    import torch
    import paper_1608_05794_b200 as ck
    rng = np.random.default_rng(1000 * P + n)
    na = rng.integers(0, 40000, size=n).astype(np.int32)       # heavy tail like config 4 (max ~ 39,000 attempts)
    na[rng.random(n) < 0.7] //= 300
    nr = rng.integers(0, 50, size=n).astype(np.int32)
    if n > 40:
        na[:P] = 0; nr[:P] = 0                                  # an idle unit
    W = ck.Mechanism.waste(torch.from_numpy(na).cuda(), torch.from_numpy(nr).cuda(), P).cpu().numpy()
    ref = oracle.waste(na.astype(np.int64) + nr, P)
    assert W.shape == ref.shape and np.array_equal(W, ref)
    W1 = ck.Mechanism.waste(torch.from_numpy(na).cuda(), None, P).cpu().numpy()   # n_reject may be null
    assert np.array_equal(W1, oracle.waste(na, P))
    for tasks in (2, 7):                                                            # several reactors per lane
        Wt = ck.Mechanism.waste(torch.from_numpy(na).cuda(), torch.from_numpy(nr).cuda(), P, tasks=tasks).cpu().numpy()
        assert np.array_equal(Wt, oracle.waste_tasks(na.astype(np.int64) + nr, P, tasks))


def test_waste_of_a_real_run_and_report_agree(oracle):
    """Step counts of a ROS4 run (config-3 recipe): ck_waste at P = 32 averages to the report's waste_p32, equals the
    oracle on the same counts, and the flame-ordered copy of the batch wastes less than the shuffled one."""
    import torch
    import paper_1608_05794_b200 as ck
    from synth_inputs import make_config
    means = {}
    for flame in (False, True):
        mech, y, p, cfg = make_config("C3", n=2048, flame_ordered=flame)
        M = ck.Mechanism(mech)
        r = M.integrate("ros", torch.from_numpy(y).cuda(), torch.from_numpy(p).cuda(), cfg["dt"])
        W = M.waste(r["n_accept"], r["n_reject"], 32).cpu().numpy()
        att = (r["n_accept"] + r["n_reject"]).cpu().numpy()
        assert np.array_equal(W, oracle.waste(att, 32))
        assert abs(W.mean() - r["report"]["waste_p32"]) < 1e-12
        means[flame] = W.mean()
    assert means[True] < means[False]


def test_waste_rejects_bad_arguments():
    import torch
    import paper_1608_05794_b200 as ck
    a = torch.zeros(8, dtype=torch.int32, device="cuda")
    for P in (0, -1, 1025):
        with pytest.raises(ck.CkError):
            ck.Mechanism.waste(a, None, P)
    assert ck.Mechanism.waste(a[:0], None, 32).numel() == 0
