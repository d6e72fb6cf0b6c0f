"""Test-only input builders (no method arithmetic): tiny hand-made mechanisms as ck_mech_desc-shaped dicts."""
import numpy as np

R_U = 8.31446261815324e7
R_CAL = 1.98720425864083
P_ATM = 1.01325e6


def custom_mech(W, nasa, reactions, elem_comp=None, t_mid=1000.0, nasa_hi=None):
    """reactions: list of dicts(reac={k:nu}, prod={k:nu}, A, beta, Ea, rev, type, A0, beta0, Ea0, troe, eff={k:val})."""
    K = len(W)
    R = len(reactions)
    nasa = np.asarray(nasa, dtype=np.float64).reshape(K, 7)
    hi = nasa.copy() if nasa_hi is None else np.asarray(nasa_hi, dtype=np.float64).reshape(K, 7)
    if elem_comp is None:
        elem_comp = np.ones((K, 1), dtype=np.int32)
    elem_comp = np.asarray(elem_comp, dtype=np.int32)
    rp, rs, rn, pp, ps, pn, ep, es, ev = [0], [], [], [0], [], [], [0], [], []
    g = lambda r, k, d: r.get(k, d)
    for r in reactions:
        for k, nu in sorted(r["reac"].items()):
            rs.append(k); rn.append(nu)
        rp.append(len(rs))
        for k, nu in sorted(r["prod"].items()):
            ps.append(k); pn.append(nu)
        pp.append(len(ps))
        for k, v in sorted(g(r, "eff", {}).items()):
            es.append(k); ev.append(v)
        ep.append(len(es))
    i32 = lambda a: np.array(a, dtype=np.int32)
    return dict(
        n_species=K, n_reactions=R, n_elements=elem_comp.shape[1],
        mol_wt=np.asarray(W, dtype=np.float64), elem_comp=elem_comp,
        nasa_lo=nasa.copy(), nasa_hi=hi, t_mid=np.full(K, float(t_mid)),
        reac_ptr=i32(rp), reac_spec=i32(rs), reac_nu=i32(rn),
        prod_ptr=i32(pp), prod_spec=i32(ps), prod_nu=i32(pn),
        A=np.array([r["A"] for r in reactions], dtype=np.float64),
        beta=np.array([g(r, "beta", 0.0) for r in reactions], dtype=np.float64),
        Ea=np.array([g(r, "Ea", 0.0) for r in reactions], dtype=np.float64),
        reversible=np.array([1 if g(r, "rev", True) else 0 for r in reactions], dtype=np.uint8),
        type=np.array([g(r, "type", 0) for r in reactions], dtype=np.uint8),
        A0=np.array([g(r, "A0", 0.0) for r in reactions], dtype=np.float64),
        beta0=np.array([g(r, "beta0", 0.0) for r in reactions], dtype=np.float64),
        Ea0=np.array([g(r, "Ea0", 0.0) for r in reactions], dtype=np.float64),
        troe=np.array([g(r, "troe", [0.0, 1.0, 1.0, -1.0]) for r in reactions], dtype=np.float64).reshape(R, 4),
        eff_ptr=i32(ep), eff_spec=i32(es), eff_val=np.array(ev, dtype=np.float64),
    )


def abc_mech(rtype=0, **kw):
    """A + B (+M) <=> C with W_C = W_A + W_B; 4th species D is an inert collider. Constant cp (no T-dependence)."""
    W = [2.016, 31.998, 34.014, 28.014]
    nasa = [[3.5, 0, 0, 0, 0, 0.0, 15.0], [3.5, 0, 0, 0, 0, 0.0, 24.0], [5.0, 0, 0, 0, 0, -15000.0, 28.0],
            [3.5, 0, 0, 0, 0, 0.0, 22.0]]
    elem = [[2, 0, 0], [0, 2, 0], [2, 2, 0], [0, 0, 2]]
    r = dict(reac={0: 1, 1: 1}, prod={2: 1}, A=1e12, beta=0.0, Ea=0.0, rev=False, type=rtype)
    r.update(kw)
    return custom_mech(W, nasa, [r], elem_comp=elem)
