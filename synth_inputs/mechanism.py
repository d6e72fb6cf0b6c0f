"""Seeded synthetic kinetic-mechanism generator (inputs only; no method arithmetic).

Stand-ins for the paper's three models (Table 1): the real files are
not available, so mechanisms with their *shape* are drawn from a seeded RNG following
BASELINE.json `configs` and SURVEY.md section 8(d):
  * species are element-count vectors, W_k = sum_e n_ek * (atomic mass)  -> exact mass balance
  * reactions are elementally balanced A+B<=>C+D or C+D(+M)<=>A, all reversible
  * Arrhenius A log-uniform 1e8..1e14 (cgs), beta ~ U[-1.5,2], Ea ~ U[0,50] kcal/mol
  * ~10 % third-body rows with efficiencies ~U[0.5,12], ~8 % Troe falloff rows
  * NASA-7 thermo, two ranges joined at T_mid=1000 K, cp/R monotone in [2.5,8] on 300..3000 K

This module serves BOTH the oracle tests and the CUDA path. It evaluates no reaction rate,
no RHS, no Jacobian.  The only formulas it contains are the ones needed to *construct* the
coefficient tables (polynomial least squares; integration constants that make the two NASA
ranges continuous).  The output is a plain dict of numpy arrays whose keys mirror the
`ck_mech_desc` struct of include/ck.h.
"""
from __future__ import annotations

import itertools
import numpy as np

ATOMIC_MASS = {"H": 1.008, "C": 12.011, "O": 15.999, "N": 14.007, "Ar": 39.948}

T_LOW, T_MID, T_HIGH = 300.0, 1000.0, 3000.0
T_STD = 298.15

# reaction types (include/ck.h)
PLAIN, THREE_BODY, LINDEMANN, TROE = 0, 1, 2, 3


def _formula(elements, comp):
    return "".join(f"{e}{int(c)}" for e, c in zip(elements, comp) if c)


def _candidate_species(elements, max_c, rng):
    """Enumerate small compositions over `elements` (valence-plausible, small)."""
    idx = {e: i for i, e in enumerate(elements)}
    out = []
    has = lambda e: e in idx
    cmax = max_c if has("C") else 0
    for c in range(cmax + 1):
        for h in range(0, 2 * c + 3):
            for o in range(0, 4):
                for n in range(0, 3 if (has("N") and cmax > 0) else 1):
                    atoms = c + h + o + n
                    if atoms == 0 or atoms > 3 * max(c, 1) + 4:
                        continue
                    if h > 2 * c + 2 + n:
                        continue
                    if c == 0 and o == 3 and h > 0:
                        continue
                    if n and (c + o + h) > 3:
                        continue
                    comp = np.zeros(len(elements), dtype=np.int32)
                    if c:
                        comp[idx["C"]] = c
                    if h:
                        comp[idx["H"]] = h
                    if o:
                        comp[idx["O"]] = o
                    if n:
                        comp[idx["N"]] = n
                    out.append(comp)
    return out


def _anchors(elements, fuel):
    idx = {e: i for i, e in enumerate(elements)}

    def mk(**kw):
        comp = np.zeros(len(elements), dtype=np.int32)
        for e, c in kw.items():
            comp[idx[e]] = c
        return comp

    anchors = []  # (role, comp, Hf/R [K] or None)
    anchors.append(("fuel", mk(**fuel), 0.0 if set(fuel) == {"H"} else -9000.0))
    anchors.append(("O2", mk(O=2), 0.0))
    anchors.append(("N2", mk(N=2), 0.0))
    anchors.append(("H2O", mk(H=2, O=1), -29000.0))
    if "C" in idx:
        anchors.append(("CO2", mk(C=1, O=2), -47000.0))
        if set(fuel) != {"H"}:
            anchors.append(("H2", mk(H=2), 0.0))
    if "Ar" in idx:
        anchors.append(("Ar", mk(Ar=1), 0.0))
    return anchors


def _cp_target(T, c_lo, c_hi, pw):
    x = np.clip((T - T_LOW) / (T_HIGH - T_LOW), 0.0, 1.0)
    return c_lo + (c_hi - c_lo) * (1.0 - (1.0 - x) ** pw)


def _fit_nasa(c_lo, c_hi, pw, hf_over_R, s298_over_R, T_MID=T_MID):
    """Two quartic fits of cp/R joined C0/C1 at T_MID; a6,a7 from Hf(298)/R, S(298)/R and continuity."""
    if c_hi - c_lo < 1e-12:  # monatomic: constant cp
        lo = np.array([c_lo, 0, 0, 0, 0], dtype=np.float64)
        hi = lo.copy()
    else:
        # scaled variable x = T/1000 for conditioning
        Tl = np.linspace(T_LOW, T_MID, 71)
        Vl = np.vander(Tl / 1000.0, 5, increasing=True)
        cl, *_ = np.linalg.lstsq(Vl, _cp_target(Tl, c_lo, c_hi, pw), rcond=None)
        # high range: constrain value and slope at T_MID (x=xm): p(x) = v + s (x-xm) + (x-xm)^2 (d0 + d1 (x-xm) + d2 (x-xm)^2)
        xm = T_MID / 1000.0
        v = (cl * xm ** np.arange(5)).sum()
        s = (cl[1:] * np.arange(1, 5) * xm ** np.arange(4)).sum()
        Th = np.linspace(T_MID, T_HIGH, 201)
        z = Th / 1000.0 - xm
        B = np.stack([z**2, z**3, z**4], axis=1)
        rhs = _cp_target(Th, c_lo, c_hi, pw) - v - s * z
        d, *_ = np.linalg.lstsq(B, rhs, rcond=None)
        # expand in powers of x
        pz = np.array([v, s, d[0], d[1], d[2]])  # coefficients in z
        ch = np.zeros(5)
        for k, ck in enumerate(pz):  # (x-xm)^k binomial expansion
            for j in range(k + 1):
                from math import comb
                ch[j] += ck * comb(k, j) * (-xm) ** (k - j)
        lo = cl / (1000.0 ** np.arange(5))
        hi = ch / (1000.0 ** np.arange(5))

    def hpoly(a, T):  # H/R minus a6
        return a[0] * T + a[1] * T**2 / 2 + a[2] * T**3 / 3 + a[3] * T**4 / 4 + a[4] * T**5 / 5

    def spoly(a, T):  # S/R minus a7
        return a[0] * np.log(T) + a[1] * T + a[2] * T**2 / 2 + a[3] * T**3 / 3 + a[4] * T**4 / 4

    a6_lo = hf_over_R - hpoly(lo, T_STD)
    a7_lo = s298_over_R - spoly(lo, T_STD)
    a6_hi = hpoly(lo, T_MID) + a6_lo - hpoly(hi, T_MID)
    a7_hi = spoly(lo, T_MID) + a7_lo - spoly(hi, T_MID)
    return np.concatenate([lo, [a6_lo, a7_lo]]), np.concatenate([hi, [a6_hi, a7_hi]])


def _cp_ok(lo, hi, T_MID=T_MID):
    Tl = np.arange(T_LOW, T_MID + 1, 10.0)
    Th = np.arange(T_MID, T_HIGH + 1, 10.0)
    cl = sum(lo[i] * Tl**i for i in range(5))
    ch = sum(hi[i] * Th**i for i in range(5))
    c = np.concatenate([cl, ch])
    return c.min() >= 2.5 - 1e-9 and c.max() <= 8.0 + 1e-9 and np.all(np.diff(c) >= -1e-9)


def make_mechanism(n_species, n_reactions, elements, seed, fuel, max_c=2,
                   n_third=None, n_troe=None, n_lindemann=0, k_cap=3.0e13, k_cap_uni=1.0e10, t_mid_choices=None, exclude_from_pool=()):
    """Return a dict describing a synthetic mechanism (keys mirror ck_mech_desc).
    t_mid_choices: draw each species' NASA range break from this list (own RNG stream; default: 1000 K for all)."""
    rng = np.random.default_rng(seed)
    rng_tm = np.random.default_rng([seed, 7919])
    elements = list(elements)
    E = len(elements)
    mass = np.array([ATOMIC_MASS[e] for e in elements])
    if n_third is None:
        n_third = int(round(0.10 * n_reactions))
    if n_troe is None:
        n_troe = int(round(0.08 * n_reactions))

    # ---- species -------------------------------------------------------------------------
    anchors = _anchors(elements, fuel)
    comps = [a[1] for a in anchors]
    roles = {a[0]: i for i, a in enumerate(anchors)}
    hf = [a[2] for a in anchors]
    have = {tuple(c) for c in comps}
    cands = [c for c in _candidate_species(elements, max_c, rng) if tuple(c) not in have]
    if exclude_from_pool:  # e.g. no nitrogen chemistry in a small model (N2 stays as an inert anchor)
        bad = [elements.index(e) for e in exclude_from_pool]
        cands = [c for c in cands if not any(c[b] for b in bad)]
    # light species first so that the small H/O radical pool is always present
    cands.sort(key=lambda c: (int(c.sum()), tuple(c)))
    need = n_species - len(comps)
    if need > len(cands):
        raise ValueError("not enough candidate compositions")
    n_light = min(need, max(5, need // 3))
    pick = list(range(n_light))
    rest = np.arange(n_light, len(cands))
    if need > n_light:
        pick += list(rng.choice(rest, size=need - n_light, replace=False))
    for i in pick:
        comps.append(cands[i])
        hf.append(None)
    comps = np.array(comps, dtype=np.int32)
    K = n_species
    assert comps.shape == (K, E)
    mol_wt = comps @ mass
    natoms = comps.sum(axis=1)
    names = [_formula(elements, c) for c in comps]
    inert = np.zeros(K, dtype=bool)
    inert[roles["N2"]] = True
    if "Ar" in roles:
        inert[roles["Ar"]] = True

    # ---- thermo --------------------------------------------------------------------------
    nasa_lo = np.zeros((K, 7))
    nasa_hi = np.zeros((K, 7))
    hf_R = np.zeros(K)
    s_R = np.zeros(K)
    t_mid = np.full(K, T_MID)
    if t_mid_choices is not None:
        t_mid = np.asarray(rng_tm.choice(np.asarray(t_mid_choices, dtype=np.float64), size=K), dtype=np.float64)
    for k in range(K):
        hf_R[k] = hf[k] if hf[k] is not None else rng.uniform(-2.5e4, 3.5e4)
        s_R[k] = float(np.clip(18.0 + 2.5 * natoms[k] + rng.uniform(-3, 3), 15.0, 40.0))
        if natoms[k] == 1:
            c_lo = c_hi = 2.5
        else:
            c_lo = 3.5 if natoms[k] == 2 else min(4.0 + 0.1 * natoms[k], 4.5)
            c_hi = min(8.0, c_lo + rng.uniform(0.35, 0.6) * natoms[k])
        for _ in range(100):
            pw = rng.uniform(1.5, 3.0)
            lo, hi = _fit_nasa(c_lo, c_hi, pw, hf_R[k], s_R[k], float(t_mid[k]))
            if _cp_ok(lo, hi, float(t_mid[k])):
                break
            c_hi = c_lo + 0.9 * (c_hi - c_lo)
        else:
            raise RuntimeError("thermo fit failed")
        nasa_lo[k], nasa_hi[k] = lo, hi

    # ---- reactions -----------------------------------------------------------------------
    active = [k for k in range(K) if not inert[k]]
    key = lambda c: tuple(int(x) for x in c)
    pair_buckets = {}
    for a, b in itertools.combinations_with_replacement(active, 2):
        pair_buckets.setdefault(key(comps[a] + comps[b]), []).append((a, b))
    single = {}
    for a in active:
        single.setdefault(key(comps[a]), []).append(a)
    bimol = []  # (A,B) <=> (C,D)
    for comp_sum, pairs in pair_buckets.items():
        for (p1, p2) in itertools.combinations(pairs, 2):
            if set(p1) & set(p2):
                continue
            bimol.append((p1, p2))
    assoc = []  # (C,D) <=> (A,)
    for comp_sum, pairs in pair_buckets.items():
        for a in single.get(comp_sum, []):
            for pr in pairs:
                assoc.append((pr, (a,)))
    rng.shuffle(bimol)
    rng.shuffle(assoc)
    n_special = n_third + n_troe + n_lindemann
    if len(assoc) < n_special:
        raise ValueError(f"only {len(assoc)} association reactions available, need {n_special}")
    n_assoc_plain = min(len(assoc) - n_special, max(0, int(0.05 * n_reactions)))
    n_bimol = n_reactions - n_special - n_assoc_plain
    if len(bimol) < n_bimol:
        raise ValueError(f"only {len(bimol)} bimolecular reactions available, need {n_bimol}")
    chosen = [(r, PLAIN) for r in bimol[:n_bimol]]
    spare_bimol = bimol[n_bimol:]
    types = [THREE_BODY] * n_third + [TROE] * n_troe + [LINDEMANN] * n_lindemann + [PLAIN] * n_assoc_plain
    chosen += [(r, t) for r, t in zip(assoc, types)]
    spare_assoc = assoc[len(types):]

    # patch: every non-inert species occurs at least once
    def occurs(k):
        return any(k in lhs or k in rhs for (lhs, rhs), _ in chosen)

    for k in active:
        if occurs(k):
            continue
        repl = next((r for r in spare_bimol if k in r[0] or k in r[1]), None)
        if repl is None:
            repl = next((r for r in spare_assoc if k in r[0] or k in r[1]), None)
        if repl is None:
            continue  # species cannot react with this species set; stays a spectator
        # replace a plain bimolecular row whose species all occur elsewhere
        for j in range(n_bimol):
            (lhs, rhs), t = chosen[j]
            chosen[j] = (repl, PLAIN)
            if all(occurs(s) for s in lhs + rhs):
                break
            chosen[j] = ((lhs, rhs), t)

    # orientation: forward direction has dG(1500 K) ~ dHf - 1500 dS(298) < 0 (generator-level estimate)
    def orient(lhs, rhs):
        dh = sum(hf_R[s] for s in rhs) - sum(hf_R[s] for s in lhs)
        ds = sum(s_R[s] for s in rhs) - sum(s_R[s] for s in lhs)
        return (lhs, rhs) if (dh - 1500.0 * ds) <= 0 else (rhs, lhs)

    order = rng.permutation(len(chosen))
    R = len(chosen)
    reac_ptr, reac_spec, reac_nu = [0], [], []
    prod_ptr, prod_spec, prod_nu = [0], [], []
    rtype = np.zeros(R, dtype=np.uint8)
    A = np.zeros(R); beta = np.zeros(R); Ea = np.zeros(R)
    A0 = np.zeros(R); beta0 = np.zeros(R); Ea0 = np.zeros(R)
    troe = np.zeros((R, 4))
    eff_ptr, eff_spec, eff_val = [0], [], []
    Rcal = 1.98720425864083

    def side(lst):
        sp, nu = [], []
        for s in sorted(set(lst)):
            sp.append(s); nu.append(lst.count(s))
        return sp, nu

    def draw_rate(cap):
        for _ in range(10000):
            a = 10.0 ** rng.uniform(8, 14)
            b = rng.uniform(-1.5, 2.0)
            e = rng.uniform(0.0, 50.0e3)
            kmax = max(a * T**b * np.exp(-e / (Rcal * T)) for T in (800.0, 1500.0, 2500.0))
            if kmax <= cap:
                return a, b, e
        raise RuntimeError("rate draw failed")

    for i, j in enumerate(order):
        (lhs, rhs), t = chosen[j]
        lhs, rhs = orient(tuple(lhs), tuple(rhs))
        sp, nu = side(list(lhs)); reac_spec += sp; reac_nu += nu; reac_ptr.append(len(reac_spec))
        sp, nu = side(list(rhs)); prod_spec += sp; prod_nu += nu; prod_ptr.append(len(prod_spec))
        rtype[i] = t
        uni = len(lhs) == 1
        A[i], beta[i], Ea[i] = draw_rate(k_cap_uni if (uni and t != THREE_BODY) else k_cap)
        if t in (THREE_BODY, LINDEMANN, TROE):
            ne = int(rng.integers(2, 5))
            who = rng.choice(K, size=min(ne, K), replace=False)
            for s in sorted(who):
                eff_spec.append(int(s)); eff_val.append(float(rng.uniform(0.5, 12.0)))
        eff_ptr.append(len(eff_spec))
        if t in (LINDEMANN, TROE):
            A0[i] = A[i] * 10.0 ** rng.uniform(4, 6)
            beta0[i] = beta[i] - rng.uniform(0, 2)
            Ea0[i] = rng.uniform(0.0, 50.0e3)
        if t == TROE:
            troe[i, 0] = rng.uniform(0.3, 0.9)
            troe[i, 1] = rng.uniform(50, 500)
            troe[i, 2] = rng.uniform(500, 3000)
            troe[i, 3] = rng.uniform(2000, 8000) if rng.random() < 0.5 else -1.0

    mech = dict(
        n_species=K, n_reactions=R, n_elements=E,
        elements=elements, species_names=names,
        mol_wt=np.ascontiguousarray(mol_wt, dtype=np.float64),
        elem_comp=np.ascontiguousarray(comps, dtype=np.int32),
        nasa_lo=np.ascontiguousarray(nasa_lo), nasa_hi=np.ascontiguousarray(nasa_hi),
        t_mid=t_mid,
        reac_ptr=np.array(reac_ptr, dtype=np.int32), reac_spec=np.array(reac_spec, dtype=np.int32),
        reac_nu=np.array(reac_nu, dtype=np.int32),
        prod_ptr=np.array(prod_ptr, dtype=np.int32), prod_spec=np.array(prod_spec, dtype=np.int32),
        prod_nu=np.array(prod_nu, dtype=np.int32),
        A=A, beta=beta, Ea=Ea,
        reversible=np.ones(R, dtype=np.uint8), type=rtype,
        A0=A0, beta0=beta0, Ea0=Ea0, troe=np.ascontiguousarray(troe),
        eff_ptr=np.array(eff_ptr, dtype=np.int32), eff_spec=np.array(eff_spec, dtype=np.int32),
        eff_val=np.array(eff_val, dtype=np.float64),
        roles=roles, inert=inert, seed=seed, hf_R=hf_R, s_R=s_R,
    )
    return mech


def with_row_kinds(mech, seed, n_lindemann=0, frac_irreversible=0.0, n_termolecular=0, n_both_sides=0,
                   n_many_eff=0, many_eff=8, split_irreversible=False):
    """Post-process a generated mechanism so that it holds the reaction kinds the paper's formulation covers but
    the BASELINE recipes never draw (PAPER.md:113 third-body "and/or pressure effects"; PAPER.md:119 irreversible
    reactions; Eq. 14 with nu > 1; PAPER.md:149 a model of irreversible reactions only).  Own RNG stream.
      n_lindemann        Troe rows turned into Lindemann rows (same low-pressure limit, F = 1)
      frac_irreversible  share of rows marked irreversible (k_r = 0)
      n_termolecular     appended balanced rows A + B + C <=> D (+E), all species distinct
      n_both_sides       appended rows 2A + B <=> A + C (nu = 2 and a species on both sides)
      n_many_eff         third-body / falloff rows given `many_eff` non-unit efficiencies
      split_irreversible every reversible row becomes TWO irreversible rows, forward and backward, the backward one
                         with Arrhenius parameters of its own (the shape of an explicit-reverse model)."""
    rng = np.random.default_rng([int(seed), 104729])
    K = mech["n_species"]
    comps, inert = mech["elem_comp"], mech["inert"]
    hf_R, s_R = mech["hf_R"], mech["s_R"]
    Rcal = 1.98720425864083
    rows = []
    for i in range(mech["n_reactions"]):
        rs = slice(mech["reac_ptr"][i], mech["reac_ptr"][i + 1]); ps = slice(mech["prod_ptr"][i], mech["prod_ptr"][i + 1])
        es = slice(mech["eff_ptr"][i], mech["eff_ptr"][i + 1])
        rows.append(dict(reac=dict(zip(mech["reac_spec"][rs].tolist(), mech["reac_nu"][rs].tolist())),
                         prod=dict(zip(mech["prod_spec"][ps].tolist(), mech["prod_nu"][ps].tolist())),
                         A=float(mech["A"][i]), beta=float(mech["beta"][i]), Ea=float(mech["Ea"][i]),
                         rev=int(mech["reversible"][i]), type=int(mech["type"][i]), A0=float(mech["A0"][i]),
                         beta0=float(mech["beta0"][i]), Ea0=float(mech["Ea0"][i]), troe=mech["troe"][i].copy(),
                         eff=dict(zip(mech["eff_spec"][es].tolist(), mech["eff_val"][es].tolist()))))
    active = [k for k in range(K) if not inert[k]]
    key = lambda c: tuple(int(x) for x in c)

    def orient(lhs, rhs):
        dh = sum(hf_R[s] for s in rhs) - sum(hf_R[s] for s in lhs)
        ds = sum(s_R[s] for s in rhs) - sum(s_R[s] for s in lhs)
        return (lhs, rhs) if (dh - 1500.0 * ds) <= 0 else (rhs, lhs)

    def draw_rate(cap):
        for _ in range(10000):
            a = 10.0 ** rng.uniform(8, 14); b = rng.uniform(-1.5, 2.0); e = rng.uniform(0.0, 50.0e3)
            if max(a * T**b * np.exp(-e / (Rcal * T)) for T in (800.0, 1500.0, 2500.0)) <= cap:
                return a, b, e
        raise RuntimeError("rate draw failed")

    def count(lst):
        d = {}
        for s in lst:
            d[s] = d.get(s, 0) + 1
        return d

    def new_row(lhs, rhs, cap):
        a, b, e = draw_rate(cap)
        return dict(reac=count(lhs), prod=count(rhs), A=a, beta=b, Ea=e, rev=1, type=PLAIN, A0=0.0, beta0=0.0, Ea0=0.0,
                    troe=np.zeros(4), eff={})

    if n_termolecular:
        single = {key(comps[a]): a for a in active}
        pairs = {}
        for a, b in itertools.combinations(active, 2):
            pairs.setdefault(key(comps[a] + comps[b]), []).append((a, b))
        found = []
        for tr in itertools.combinations(active, 3):
            ks = key(comps[list(tr)].sum(0))
            if ks in single and single[ks] not in tr:
                found.append((tr, (single[ks],)))
            for pr in pairs.get(ks, []):
                if not set(pr) & set(tr):
                    found.append((tr, pr))
        if len(found) < n_termolecular:
            raise ValueError(f"only {len(found)} termolecular rows available")
        for j in rng.choice(len(found), size=n_termolecular, replace=False):
            lhs, rhs = orient(*found[j])
            rows.append(new_row(lhs, rhs, 1.0e16 if len(lhs) == 3 else 1.0e10))   # cm^6/mol^2/s scale for A+B+C
    if n_both_sides:
        single = {}
        for a in active:
            single.setdefault(key(comps[a]), []).append(a)
        found = []
        for a, b in itertools.permutations(active, 2):
            for c in single.get(key(comps[a] + comps[b]), []):
                found.append(((a, a, b), (a, c)))
        if len(found) < n_both_sides:
            raise ValueError(f"only {len(found)} both-sides rows available")
        for j in rng.choice(len(found), size=n_both_sides, replace=False):
            lhs, rhs = orient(*found[j])
            rows.append(new_row(lhs, rhs, 1.0e16 if len(lhs) == 3 else 3.0e13))
    troe_rows = [i for i, r in enumerate(rows) if r["type"] == TROE]
    for i in troe_rows[:n_lindemann]:
        rows[i]["type"] = LINDEMANN
    special = [i for i, r in enumerate(rows) if r["type"] != PLAIN]
    for i in special[:n_many_eff]:
        who = rng.choice(K, size=min(many_eff, K), replace=False)
        rows[i]["eff"] = {int(s): float(rng.uniform(0.5, 12.0)) for s in sorted(who)}
    if frac_irreversible > 0:
        for i in rng.choice(len(rows), size=int(round(frac_irreversible * len(rows))), replace=False):
            rows[i]["rev"] = 0
    if split_irreversible:
        out = []
        for r in rows:
            f = dict(r); f["rev"] = 0
            out.append(f)
            if r["rev"]:
                a, b, e = draw_rate(1.0e10 if sum(r["prod"].values()) == 1 else 3.0e13)
                g = dict(r); g.update(reac=r["prod"], prod=r["reac"], A=a, beta=b, Ea=e, rev=0)
                if r["type"] >= LINDEMANN:
                    g["A0"] = a * 10.0 ** rng.uniform(4, 6); g["beta0"] = b - rng.uniform(0, 2); g["Ea0"] = rng.uniform(0.0, 50.0e3)
                out.append(g)
        rows = out
    R = len(rows)
    i32 = lambda a: np.array(a, dtype=np.int32)
    rp, rs_, rn, pp, ps_, pn, ep, es_, ev = [0], [], [], [0], [], [], [0], [], []
    for r in rows:
        for k, nu in sorted(r["reac"].items()):
            rs_.append(k); rn.append(nu)
        rp.append(len(rs_))
        for k, nu in sorted(r["prod"].items()):
            ps_.append(k); pn.append(nu)
        pp.append(len(ps_))
        for k, v in sorted(r["eff"].items()):
            es_.append(k); ev.append(v)
        ep.append(len(es_))
    out = dict(mech)
    out.update(n_reactions=R, reac_ptr=i32(rp), reac_spec=i32(rs_), reac_nu=i32(rn), prod_ptr=i32(pp), prod_spec=i32(ps_),
               prod_nu=i32(pn), A=np.array([r["A"] for r in rows]), beta=np.array([r["beta"] for r in rows]),
               Ea=np.array([r["Ea"] for r in rows]), reversible=np.array([r["rev"] for r in rows], dtype=np.uint8),
               type=np.array([r["type"] for r in rows], dtype=np.uint8), A0=np.array([r["A0"] for r in rows]),
               beta0=np.array([r["beta0"] for r in rows]), Ea0=np.array([r["Ea0"] for r in rows]),
               troe=np.ascontiguousarray(np.array([r["troe"] for r in rows], dtype=np.float64).reshape(R, 4)),
               eff_ptr=i32(ep), eff_spec=i32(es_), eff_val=np.array(ev, dtype=np.float64))
    return out


def mech_h2(seed=0):
    """Config 1: 9 species over {H,O,N}, 20 reversible reactions, 4 third-body + 1 Troe."""
    return make_mechanism(9, 20, ["H", "O", "N"], seed, fuel=dict(H=2), max_c=0, n_third=4, n_troe=1)


def mech_c1(seed=1):
    """Configs 2-4: 53 species / 325 reactions over {C,H,O,N,Ar}, methane-air shaped."""
    return make_mechanism(53, 325, ["C", "H", "O", "N", "Ar"], seed, fuel=dict(C=1, H=4), max_c=2)


def mech_c4(seed=2):
    """Config 5: 111 species / 784 reactions, C1-C4 shaped."""
    return make_mechanism(111, 784, ["C", "H", "O", "N", "Ar"], seed, fuel=dict(C=2, H=4), max_c=4)


def mech_h2co(seed=3):
    """Table 1's smallest model shape (H2/CO, 14 species / 38 reactions) over {C,H,O,N,Ar}: CO-rich
    syngas-like fuel, 4 third-body + 3 Troe rows, one of them turned into a Lindemann row."""
    m = make_mechanism(14, 38, ["C", "H", "O", "N", "Ar"], seed, fuel=dict(C=1, O=1), max_c=1, n_third=4, n_troe=3,
                       exclude_from_pool=("N",))
    return with_row_kinds(m, seed, n_lindemann=1)


def mech_c1_irrev(seed=4):
    """53 species, irreversible reactions only (ref. [20]'s model of 53 species / 634 irreversible
    reactions): 317 reversible-shaped rows of the methane-air-shaped recipe, each written as a forward and a backward
    irreversible row with Arrhenius parameters of its own."""
    m = make_mechanism(53, 317, ["C", "H", "O", "N", "Ar"], seed, fuel=dict(C=1, H=4), max_c=2)
    return with_row_kinds(m, seed, split_irreversible=True)


def mech_rowkinds(n_species=20, n_reactions=48, seed=5, max_c=1, **kw):
    """Every row kind include/ck.h accepts in one small model: Lindemann rows, irreversible rows, termolecular sides
    (A + B + C, 2A + B), a species on both sides, third-body rows with 8 efficiencies, three distinct t_mid values."""
    m = make_mechanism(n_species, n_reactions, ["C", "H", "O", "N", "Ar"], seed, fuel=dict(C=1, O=1) if max_c < 2 else dict(C=1, H=4),
                       max_c=max_c, n_third=max(3, n_reactions // 10), n_troe=max(4, n_reactions // 10),
                       t_mid_choices=(900.0, 1000.0, 1400.0), exclude_from_pool=("N",) if n_species < 40 else ())
    opts = dict(n_lindemann=2, frac_irreversible=0.25, n_termolecular=3, n_both_sides=3, n_many_eff=2)
    opts.update(kw)
    return with_row_kinds(m, seed, **opts)


def mech_decay(A=1.0e3, reversible=False, dS=0.0):
    """Two isomers A<=>B with identical W and cp (dH=0): the closed-form pin of SURVEY 8(c)-1.

    With reversible=True the two species differ only in a7 (entropy) by dS, so K_c = exp(dS).
    """
    lo = np.array([3.5, 0, 0, 0, 0, -1000.0, 4.0])
    nasa = np.stack([lo, lo.copy()])
    nasa[1, 6] += dS
    return dict(
        n_species=2, n_reactions=1, n_elements=1, elements=["H"], species_names=["A", "B"],
        mol_wt=np.array([2.016, 2.016]), elem_comp=np.array([[2], [2]], dtype=np.int32),
        nasa_lo=nasa.copy(), nasa_hi=nasa.copy(), t_mid=np.array([1000.0, 1000.0]),
        reac_ptr=np.array([0, 1], dtype=np.int32), reac_spec=np.array([0], dtype=np.int32),
        reac_nu=np.array([1], dtype=np.int32),
        prod_ptr=np.array([0, 1], dtype=np.int32), prod_spec=np.array([1], dtype=np.int32),
        prod_nu=np.array([1], dtype=np.int32),
        A=np.array([A]), beta=np.zeros(1), Ea=np.zeros(1),
        reversible=np.array([1 if reversible else 0], dtype=np.uint8), type=np.zeros(1, dtype=np.uint8),
        A0=np.zeros(1), beta0=np.zeros(1), Ea0=np.zeros(1), troe=np.zeros((1, 4)),
        eff_ptr=np.array([0, 0], dtype=np.int32), eff_spec=np.zeros(0, dtype=np.int32),
        eff_val=np.zeros(0), roles={}, inert=np.zeros(2, dtype=bool), seed=-1,
    )
