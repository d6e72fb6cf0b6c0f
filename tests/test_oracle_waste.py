"""Pins for the oracle's Eq. 20 against what the definition fixes in closed form."""
import numpy as np
import pytest

from oracle import ck_oracle


@pytest.mark.parametrize("P", [4, 8, 16, 32])
def test_waste_closed_forms(P):
    assert ck_oracle.waste([7] * (3 * P), P).tolist() == [0.0, 0.0, 0.0]                      # no variability, no waste
    one = [0] * P; one[P // 2] = 13
    assert ck_oracle.waste(one, P)[0] == pytest.approx(1.0 - 1.0 / P, abs=1e-15)              # one busy lane of P
    ramp = list(range(1, P + 1))
    assert ck_oracle.waste(ramp, P)[0] == pytest.approx(1.0 - (P + 1) / (2.0 * P), abs=1e-15)  # sum 1..P = P(P+1)/2
    assert ck_oracle.waste([0] * P, P)[0] == 0.0                                               # idle unit (reading)


def test_waste_invariances_and_ragged_tail():
    rng = np.random.default_rng(7)
    a = rng.integers(1, 500, size=5 * 32 + 11)
    W = ck_oracle.waste(a, 32)
    assert W.shape == (6,) and np.all(W >= 0) and np.all(W < 1)
    b = a.copy(); b[:32] = rng.permutation(b[:32])                 # order inside a unit does not matter
    assert ck_oracle.waste(b, 32)[0] == pytest.approx(W[0], abs=1e-15)
    assert np.allclose(ck_oracle.waste(3 * a, 32), W, atol=1e-15)  # homogeneous of degree 0
    tail = a[5 * 32:]
    assert W[5] == pytest.approx(1.0 - tail.sum() / (11.0 * tail.max()), abs=1e-15)  # ragged unit: its own lane count
    # wider units can only see more of the spread: the mean waste does not decrease with P on the same counts
    means = [ck_oracle.waste(a[:160], P).mean() for P in (4, 8, 16, 32)]
    assert all(x <= y + 1e-15 for x, y in zip(means, means[1:]))


def test_waste_tasks_per_lane_pins(oracle):
    rng = np.random.default_rng(5)
    a = rng.integers(1, 500, size=4096)
    for P in (4, 32):
        assert np.array_equal(oracle.waste_tasks(a, P, 1), oracle.waste(a, P))              # tasks = 1 is Eq. 20
        assert np.all(oracle.waste_tasks(np.full(640, 7), P, 5) == 0.0)                      # equal counts: no waste
        pat = rng.integers(1, 100, size=P)
        w1 = oracle.waste(pat, P)[0]
        assert abs(oracle.waste_tasks(np.tile(pat, 6), P, 6)[0] - w1) < 1e-15                # copies of one pattern
        means = [oracle.waste_tasks(a, P, m).mean() for m in (1, 4, 16)]
        assert means[0] > means[1] > means[2] > 0                                            # averaging over tasks helps
    # ragged tail: 10 reactors, P = 4, 2 tasks per lane -> units of 8: second unit has 2 reactors on 2 lanes
    w = oracle.waste_tasks(np.array([1, 2, 3, 4, 5, 6, 7, 8, 9, 3]), 4, 2)
    assert abs(w[0] - (1 - 36 / (4 * 12))) < 1e-15 and abs(w[1] - (1 - 12 / (2 * 9))) < 1e-15
