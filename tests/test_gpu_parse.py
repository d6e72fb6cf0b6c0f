"""A model that went through the text parser drives the GPU path: ck_mech_parse -> ck_mech_load -> ck_rhs / ROS4, compared
with the oracle on the SAME parsed description."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_parsed_model_on_the_gpu(oracle):
    import torch
    import paper_1608_05794_b200 as ck
    from synth_inputs import make_config
    from synth_inputs.chemkin_text import write_chemkin
    m, y, p, cfg = make_config("C3", n=300)
    d = ck.parse_mechanism(write_chemkin(m))
    M, O = ck.Mechanism(d), oracle.Mech(d)
    f = M.rhs(torch.from_numpy(y).cuda(), torch.from_numpy(p).cuda()).cpu().numpy()
    fref = O.rhs(y, p, prec=1, nthreads=8)
    _, D = O.rhs(y, p, want_scale=True, nthreads=8)
    assert np.all(np.abs(f - fref) <= 1e-12 * D + 1e-300)
    yd = torch.from_numpy(y).cuda()
    r = M.integrate("ros", yd, torch.from_numpy(p).cuda(), cfg["dt"])
    ref = O.integrate("ros", y, p, cfg["dt"], nthreads=16)
    g = yd.cpu().numpy()
    assert np.all(r["status"].cpu().numpy() == 0)
    assert np.all(np.abs(g[0] - ref["y"][0]) <= 1e-5 * ref["y"][0])
    assert np.all(np.abs(g[1:] - ref["y"][1:]) <= np.maximum(1e-5 * np.abs(ref["y"][1:]), 1e-10))
