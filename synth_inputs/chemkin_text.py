"""Serialise a synthetic mechanism (dict with the keys of ck_mech_desc) as CHEMKIN-II style text -- an input writer
for the parser tests of ck_mech_parse.  No method arithmetic; no third-party mechanism data: what is
written is what synth_inputs.mechanism drew.  The THERMO cards use the format's fixed 15-column fields (E15.8), so the
NASA-7 coefficients carry nine significant digits in the text; Arrhenius parameters are written with 17."""
from __future__ import annotations


def _side(spec, nu, names, extra=""):
    terms = [(f"{int(n)}" if n != 1 else "") + names[int(s)] for s, n in zip(spec, nu)]
    return "+".join(terms) + extra


def write_chemkin(m):
    names = [n.upper() for n in m["species_names"]]
    el = [e.upper() for e in m["elements"]]
    K, R = m["n_species"], m["n_reactions"]
    out = ["ELEMENTS " + " ".join(el) + " END", "SPECIES"]
    for i in range(0, K, 6):
        out.append("  " + " ".join(f"{n:<12s}" for n in names[i:i + 6]))
    out += ["END", "THERMO ALL", "   300.000  1000.000  5000.000"]
    for k in range(K):
        comp = [(el[e], int(c)) for e, c in enumerate(m["elem_comp"][k]) if c]
        assert len(comp) <= 4
        atoms = "".join(f"{s:<2s}{c:>3d}" for s, c in comp).ljust(20)
        l1 = f"{names[k]:<18s}SYNTH " + atoms + "G" + f"{300.0:10.3f}{5000.0:10.3f}{float(m['t_mid'][k]):10.3f}"
        out.append(l1.ljust(79) + "1")
        a = list(m["nasa_hi"][k]) + list(m["nasa_lo"][k])
        out.append("".join(f"{v:15.8E}" for v in a[0:5]).ljust(79) + "2")
        out.append("".join(f"{v:15.8E}" for v in a[5:10]).ljust(79) + "3")
        out.append("".join(f"{v:15.8E}" for v in a[10:14]).ljust(79) + "4")
    out += ["END", "REACTIONS   CAL/MOLE"]
    for i in range(R):
        rs = slice(m["reac_ptr"][i], m["reac_ptr"][i + 1]); ps = slice(m["prod_ptr"][i], m["prod_ptr"][i + 1])
        t = int(m["type"][i])
        extra = {0: "", 1: "+M", 2: "(+M)", 3: "(+M)"}[t]
        arrow = "<=>" if m["reversible"][i] else "=>"
        eq = _side(m["reac_spec"][rs], m["reac_nu"][rs], names, extra) + arrow + _side(m["prod_spec"][ps], m["prod_nu"][ps], names, extra)
        out.append(f"{eq:<48s} {m['A'][i]:.16E} {m['beta'][i]:.16E} {m['Ea'][i]:.16E}")
        if t >= 2:
            out.append(f"   LOW/ {m['A0'][i]:.16E} {m['beta0'][i]:.16E} {m['Ea0'][i]:.16E} /")
        if t == 3:
            tr = m["troe"][i]
            vals = " ".join(f"{v:.16E}" for v in (tr[:3] if tr[3] < 0 else tr))
            out.append(f"   TROE/ {vals} /")
        es = slice(m["eff_ptr"][i], m["eff_ptr"][i + 1])
        if t >= 1 and es.stop > es.start:
            out.append("   " + " ".join(f"{names[int(s)]}/{v:.16E}/" for s, v in zip(m["eff_spec"][es], m["eff_val"][es])))
        if i % 17 == 3:
            out.append("   DUPLICATE   ! ignored by the parser")
    out.append("END")
    return "\n".join(out) + "\n"
