"""BASELINE.json's five configurations as (mechanism, states, call) recipes.

C1 tiny ROS4 (9 sp / 20 rxn, 1,024 reactors, dt=1e-5)       C2 RHS-only (53/325, 1,048,576 states)
C3 ROS4 (53/325, 65,536 reactors, dt=1e-6)                   C4 RKF45 (53/325, 65,536 reactors, dt=1e-7)
C5 ROS4 (111/784, 32,768 reactors, dt=1e-6)
C6 ROS4 (14/38 H2/CO-sized, 16,384 reactors, dt=1e-5)      C7 ROS4 (53 species / 634 irreversible rows, 65,536 reactors)
All: rtol=1e-6, atol=1e-10, FP64.  Seeds: mechanisms 0/1/2, states 101..105.
"""
from __future__ import annotations

import functools

from . import mechanism as _m
from . import states as _s

CONFIGS = {
    "C1": dict(mech="h2", n=1024, call="ros", dt=1e-5, seed=101),
    "C2": dict(mech="c1", n=1048576, call="rhs", dt=None, seed=102),
    "C3": dict(mech="c1", n=65536, call="ros", dt=1e-6, seed=103),
    "C4": dict(mech="c1", n=65536, call="rkf45", dt=1e-7, seed=104),
    "C5": dict(mech="c4", n=32768, call="ros", dt=1e-6, seed=105),
    # Table 1's third model shape (H2/CO-sized, 14/38) and an irreversible-only 53-species model
    "C6": dict(mech="h2co", n=16384, call="ros", dt=1e-5, seed=106),
    "C7": dict(mech="c1irr", n=65536, call="ros", dt=1e-6, seed=107),
}
RTOL, ATOL = 1e-6, 1e-10


@functools.lru_cache(maxsize=None)
def get_mech(name):
    return {"h2": _m.mech_h2, "c1": _m.mech_c1, "c4": _m.mech_c4, "h2co": _m.mech_h2co, "c1irr": _m.mech_c1_irrev,
            "rk20": _m.mech_rowkinds, "rk14": lambda: _m.mech_rowkinds(14, 30, seed=6),
            "rk130": lambda: _m.mech_rowkinds(130, 400, seed=7, max_c=4)}[name]()


def make_config(name, n=None, flame_ordered=False):
    """Return (mech, y[N,n], p[n], cfg). `n` overrides the reactor count (same recipe, same seed:
    the first n columns of a larger draw are NOT reproduced; a fresh draw of size n is made)."""
    cfg = dict(CONFIGS[name])
    mech = get_mech(cfg["mech"])
    if n is not None:
        cfg["n"] = int(n)
    n = cfg["n"]
    if name == "C1":
        y, p = _s.ignition_states(mech, n, cfg["seed"], (1000.0, 1500.0), s_range=(0.0, 0.3),
                                  flame_ordered=flame_ordered)
    elif name in ("C2", "C4"):
        y, p = _s.dirichlet_states(mech, n, cfg["seed"])
    elif name == "C3":
        y, p = _s.ignition_states(mech, n, cfg["seed"], (1000.0, 1800.0), flame_ordered=flame_ordered)
    elif name == "C5":
        y, p = _s.ignition_states(mech, n, cfg["seed"], (900.0, 1800.0), p_range_atm=(1.0, 10.0),
                                  flame_ordered=flame_ordered)
    elif name == "C6":
        y, p = _s.ignition_states(mech, n, cfg["seed"], (1000.0, 1600.0), flame_ordered=flame_ordered)
    elif name == "C7":
        y, p = _s.ignition_states(mech, n, cfg["seed"], (1000.0, 1800.0), flame_ordered=flame_ordered)
    else:
        raise KeyError(name)
    cfg["rtol"], cfg["atol"] = RTOL, ATOL
    return mech, y, p, cfg
