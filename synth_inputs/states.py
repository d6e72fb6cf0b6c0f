"""Seeded synthetic reactor states (inputs only; no method arithmetic).

Stand-ins for the paper's RHS-benchmark states (uniform composition, T swept across
the NASA range break) and its premixed-flame state data [41] (unburnt -> flame ->
burnt, so step counts diverge across reactors, Fig. 4), neither of which is available here.
Recipes follow BASELINE.json `configs` and SURVEY.md 8(d).  Layout is component-major:
y[0, r] = T (K), y[1+k, r] = Y_k; p[r] in dyn/cm^2.
"""
from __future__ import annotations

import numpy as np

P_ATM = 1.01325e6  # dyn/cm^2


def _reactant_product(mech, phi):
    """Mass-fraction vectors (K, n) of fresh fuel/air at equivalence ratio phi and of its
    complete-combustion products (bookkeeping by element counts only)."""
    K = mech["n_species"]
    roles = mech["roles"]
    el = mech["elements"]
    comp = mech["elem_comp"]
    W = mech["mol_wt"]
    n = phi.shape[0]
    f = roles["fuel"]
    c = comp[f][el.index("C")] if "C" in el else 0
    h = comp[f][el.index("H")]
    o = comp[f][el.index("O")] if "O" in el else 0
    o2_st = c + h / 4.0 - o / 2.0  # moles O2 per mole fuel (stoichiometric; oxygen in the fuel counts)
    X = np.zeros((K, n))
    X[f] = 1.0
    o2 = o2_st / phi
    X[roles["O2"]] = o2
    X[roles["N2"]] = 3.76 * o2
    if "Ar" in roles:
        X[roles["Ar"]] = 0.045 * o2
    # products of complete combustion (moles per mole of fuel in the fresh mixture)
    P = np.zeros((K, n))
    burnt = np.minimum(1.0, 1.0 / phi)  # fraction of fuel that can burn
    if "CO2" in roles:
        P[roles["CO2"]] = c * burnt
    P[roles["H2O"]] = (h / 2.0) * burnt
    P[f] += 1.0 - burnt
    P[roles["O2"]] = np.maximum(0.0, o2 - o2_st * burnt)
    P[roles["N2"]] = X[roles["N2"]]
    if "Ar" in roles:
        P[roles["Ar"]] = X[roles["Ar"]]
    Yr = X * W[:, None]
    Yp = P * W[:, None]
    return Yr / Yr.sum(0), Yp / Yp.sum(0)


def _pack(T, Y):
    Y = Y / Y.sum(0)
    return np.ascontiguousarray(np.vstack([T[None, :], Y]), dtype=np.float64)


def ignition_states(mech, n, seed, T_range, p_range_atm=(1.0, 1.0), phi_range=(0.5, 2.0),
                    s_range=(0.0, 1.0), trace=(-12.0, -6.0), flame_ordered=False):
    """Blend of reactant and product compositions at progress s, plus trace radicals
    (configs 1, 3, 5). flame_ordered=True lays s out as a tanh front along the index in
    lines of 1024 reactors, mirroring the replicated 1-D flame of PAPER.md:319-329."""
    rng = np.random.default_rng(seed)
    K = mech["n_species"]
    phi = rng.uniform(*phi_range, size=n)
    Yr, Yp = _reactant_product(mech, phi)
    if flame_ordered:
        x = (np.arange(n) % 1024) / 1023.0
        s = s_range[0] + (s_range[1] - s_range[0]) * 0.5 * (1.0 + np.tanh((x - 0.5) * 12.0))
        T = T_range[0] + (T_range[1] - T_range[0]) * 0.5 * (1.0 + np.tanh((x - 0.5) * 12.0))
    else:
        s = rng.uniform(*s_range, size=n)
        T = rng.uniform(*T_range, size=n)
    Y = (1.0 - s) * Yr + s * Yp
    tr = 10.0 ** rng.uniform(trace[0], trace[1], size=(K, n))
    tr[mech["inert"]] = 0.0
    Y = Y + tr
    p = rng.uniform(*p_range_atm, size=n) * P_ATM
    return _pack(T, Y), np.ascontiguousarray(p)


def dirichlet_states(mech, n, seed, T_range=(800.0, 2500.0), p_range_atm=(1.0, 20.0), eps_max=0.1):
    """Config 2/4 states: reactant/product blend, then a Dirichlet perturbation over all species."""
    rng = np.random.default_rng(seed)
    K = mech["n_species"]
    phi = rng.uniform(0.5, 2.0, size=n)
    Yr, Yp = _reactant_product(mech, phi)
    s = rng.uniform(0.0, 1.0, size=n)
    Y = (1.0 - s) * Yr + s * Yp
    g = rng.standard_exponential(size=(K, n))  # Dirichlet(1,...,1) = normalised exponentials
    g /= g.sum(0)
    eps = rng.uniform(0.0, eps_max, size=n)
    Y = (1.0 - eps) * Y + eps * g
    T = rng.uniform(*T_range, size=n)
    p = rng.uniform(*p_range_atm, size=n) * P_ATM
    return _pack(T, Y), np.ascontiguousarray(p)


def paper_rhs_states(mech, n):
    """The paper's own RHS-benchmark recipe: uniform composition, T linear over 500..1500 K
    (PAPER.md:287-289), p = 1 atm."""
    K = mech["n_species"]
    T = np.linspace(500.0, 1500.0, n)
    Y = np.full((K, n), 1.0 / K)
    return _pack(T, Y), np.full(n, P_ATM)
