"""CPU-only checks of the boundary: libck.so builds, loads, and exports every symbol include/ck.h declares.
No compute call is made here (there is no GPU); host-side validation paths that fail before touching the
device are exercised."""
import ctypes as C

import numpy as np
import pytest

import paper_1608_05794_b200 as ck
from paper_1608_05794_b200 import _binding as B
from synth_inputs.configs import get_mech


def test_library_exports_every_declared_symbol():
    declared = B.declared_symbols()
    exported = ck.exported_symbols()
    assert len(declared) >= 12
    missing = [s for s in declared if s not in exported]
    assert not missing, missing
    L = ck.lib()
    for s in declared:
        assert hasattr(L, s)
    assert L.ck_version() >= 100


def test_struct_sizes_match_header():
    # ck_mech_desc: 4 int32 + 23 pointers ; ck_opts: 2 int32 + 3 double + 2 int32 ; ck_report: 6 int64 + 2 double + 2 int32
    assert C.sizeof(B.MechDesc) == 16 + 23 * 8
    assert C.sizeof(B.Opts) == 8 + 24 + 8
    assert C.sizeof(B.Report) == 48 + 16 + 8


def test_mech_load_rejects_bad_input_before_touching_the_device():
    L = ck.lib()
    h = C.c_void_p()
    assert L.ck_mech_load(None, 0, C.byref(h)) == 1
    d = B.MechDesc()
    d.struct_size = 3
    assert L.ck_mech_load(C.byref(d), 0, C.byref(h)) == 1
    assert b"struct_size" in L.ck_last_error()
    # unbalanced reaction -> CK_EINVAL (validation happens on the host, before any CUDA call)
    m = dict(get_mech("h2"))
    m["prod_nu"] = m["prod_nu"].copy(); m["prod_nu"][0] += 1
    with pytest.raises(ck.CkError) as ei:
        ck.Mechanism(m)
    assert ei.value.code == 1 and "balance" in str(ei.value)
    m = dict(get_mech("h2")); m["A"] = m["A"].copy(); m["A"][3] = -1.0
    with pytest.raises(ck.CkError):
        ck.Mechanism(m)
    m = dict(get_mech("h2")); m["t_mid"] = np.linspace(900, 1100, 9)
    with pytest.raises(ck.CkError) as ei:
        ck.Mechanism(m)
    assert ei.value.code == 4


def test_null_handles_are_errors_not_crashes():
    L = ck.lib()
    v = C.c_size_t()
    assert L.ck_workspace_bytes(None, 0, C.c_int64(4), C.byref(v)) == 1
    assert L.ck_rhs(None, C.c_int64(4), None, C.c_int64(4), None, None, C.c_int64(4), None) == 1
    assert L.ck_mech_free(None) == 0


def test_product_package_does_not_import_the_oracle():
    import os, re
    root = os.path.dirname(B.__file__)
    for dp, _, fs in os.walk(root):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|ck_oracle|cko_", txt, flags=re.M), f
