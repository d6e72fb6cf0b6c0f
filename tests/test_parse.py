"""ck_mech_parse (CHEMKIN-II style text -> ck_mech_desc): host-only tests.  A synthetic
mechanism is written as text by synth_inputs.chemkin_text and must come back: integer structure and Arrhenius / falloff
parameters exactly, NASA-7 coefficients to the nine digits of the format's E15.8 fields, molar masses from the element
fields.  Malformed input must be refused with a line number."""
import numpy as np
import pytest

from synth_inputs.chemkin_text import write_chemkin
from synth_inputs.configs import get_mech


@pytest.mark.parametrize("name", ["h2", "c1", "rk20", "h2co", "c1irr"])
def test_round_trip(name):
    import paper_1608_05794_b200 as ck
    m = get_mech(name)
    d = ck.parse_mechanism(write_chemkin(m))
    assert (d["n_species"], d["n_reactions"], d["n_elements"]) == (m["n_species"], m["n_reactions"], m["n_elements"])
    assert [s.upper() for s in m["species_names"]] == d["species_names"]
    for key in ("elem_comp", "reac_ptr", "reac_spec", "reac_nu", "prod_ptr", "prod_spec", "prod_nu", "reversible", "type",
                "eff_ptr", "eff_spec"):
        assert np.array_equal(np.asarray(d[key]).ravel(), np.asarray(m[key]).ravel()), key
    for key in ("A", "beta", "Ea", "eff_val"):
        assert np.array_equal(d[key], m[key]), key                       # 17 significant digits: exact
    fall = m["type"] >= 2
    for key in ("A0", "beta0", "Ea0"):
        assert np.array_equal(d[key][fall], m[key][fall]), key
    troe = m["type"] == 3
    assert np.array_equal(d["troe"][troe][:, :3], m["troe"][troe][:, :3])
    assert np.array_equal(d["troe"][troe][:, 3] < 0, m["troe"][troe][:, 3] < 0)
    assert np.allclose(d["mol_wt"], m["mol_wt"], rtol=1e-14)
    assert np.array_equal(d["t_mid"], m["t_mid"])
    for key in ("nasa_lo", "nasa_hi"):
        assert np.allclose(d[key], m[key], rtol=2e-8, atol=1e-300), key     # E15.8


def test_parsed_mechanism_drives_the_oracle(oracle):
    """The parsed description is a complete model: the oracle's RHS on it equals its RHS on the generator's arrays to
    the precision the text carries."""
    import paper_1608_05794_b200 as ck
    from synth_inputs import make_config
    m, y, p, _ = make_config("C1", n=16)
    d = ck.parse_mechanism(write_chemkin(m))
    fa = oracle.Mech(m).rhs(y, p)
    fb, D = oracle.Mech(d).rhs(y, p, want_scale=True)
    assert np.all(np.abs(fa - fb) <= 1e-5 * D + 1e-300)


@pytest.mark.parametrize("bad,what", [
    ("ELEMENTS H END\nSPECIES A END\nREACTIONS\nA<=>B 1 0 0\nEND\n", "unknown species"),
    ("ELEMENTS H END\nSPECIES A B END\nREACTIONS\nA+M<=>B 1 0 0\nEND\n", "third body"),
    ("ELEMENTS H END\nSPECIES A B END\nREACTIONS\nA<=>B 1 0\nEND\n", "three numbers"),
    ("ELEMENTS H END\nSPECIES A A END\n", "twice"),
])
def test_malformed_input_is_refused(bad, what):
    import paper_1608_05794_b200 as ck
    with pytest.raises(ck.CkError) as e:
        ck.parse_mechanism(bad)
    assert what in str(e.value) and ("line" in str(e.value) or "no thermo" in str(e.value))
