"""ctypes binding of libck.so (include/ck.h).  Marshalling only -- no arithmetic of the method here."""
from __future__ import annotations

import ctypes as C
import os
import re

import numpy as np

from . import _build

CK_OP_ROS, CK_OP_RKF45, CK_OP_JAC = 0, 1, 2
CK_JAC_ANALYTIC, CK_JAC_FD = 0, 1
_ERR = {1: "CK_EINVAL", 2: "CK_ECUDA", 3: "CK_EWORKSPACE", 4: "CK_EUNSUPPORTED"}


class CkError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_ERR.get(code, code)}: {msg}")
        self.code = code


_PD, _PI, _PU8 = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_uint8)


class MechDesc(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("n_species", C.c_int32), ("n_reactions", C.c_int32),
                ("n_elements", C.c_int32), ("mol_wt", _PD), ("elem_comp", _PI),
                ("nasa_lo", _PD), ("nasa_hi", _PD), ("t_mid", _PD),
                ("reac_ptr", _PI), ("reac_spec", _PI), ("reac_nu", _PI),
                ("prod_ptr", _PI), ("prod_spec", _PI), ("prod_nu", _PI),
                ("A", _PD), ("beta", _PD), ("Ea", _PD), ("reversible", _PU8), ("type", _PU8),
                ("A0", _PD), ("beta0", _PD), ("Ea0", _PD), ("troe", _PD),
                ("eff_ptr", _PI), ("eff_spec", _PI), ("eff_val", _PD)]


class Opts(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("jac_mode", C.c_int32), ("rtol", C.c_double), ("atol", C.c_double),
                ("h0", C.c_double), ("max_steps", C.c_int32), ("flags", C.c_int32)]


class Report(C.Structure):
    _fields_ = [("attempts", C.c_int64), ("accepted", C.c_int64), ("rejected", C.c_int64), ("rhs_evals", C.c_int64),
                ("jac_evals", C.c_int64), ("lu_factor", C.c_int64), ("simt_efficiency", C.c_double),
                ("waste_p32", C.c_double), ("rounds", C.c_int32), ("n_failed", C.c_int32)]

    def as_dict(self):
        return {f: getattr(self, f) for f, _ in self._fields_}


_lib = None


def lib_path():
    return _build.LIB


def lib():
    """Load libck.so (building it in-tree if the sources are newer).  Raises if it cannot be had."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.ck_last_error.restype = C.c_char_p
        for name in ("ck_mech_load", "ck_mech_free", "ck_mech_sizes", "ck_mech_set_reactor", "ck_workspace_bytes", "ck_rhs", "ck_jac",
                     "ck_integrate_ros", "ck_integrate_rkf45", "ck_rhs_host", "ck_integrate_host", "ck_rhs_slots",
                     "ck_fp64_peak", "ck_fp64_mma_peak", "ck_version", "ck_jac_batched", "ck_jac_batched_static", "ck_jac_static_max_reactors", "ck_lu_solve_batched", "ck_rhs_variant", "ck_waste", "ck_waste_tasks", "ck_mech_parse", "ck_parsed_name",
                     "ck_parsed_free"):
            getattr(L, name).restype = C.c_int32
        L.ck_parsed_desc.restype = C.POINTER(MechDesc)
        _lib = L
    return _lib


def declared_symbols():
    """Function names include/ck.h declares."""
    hdr = os.path.join(os.path.dirname(_build._HERE), "include", "ck.h")
    txt = open(hdr).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(ck_[a-z0-9_]+)\s*\(", txt)))


def exported_symbols():
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", _build.build()], capture_output=True, text=True, check=True).stdout
    return sorted(l.split()[-1] for l in out.splitlines() if l.split()[-1].startswith("ck_"))


def _check(rc):
    if rc != 0:
        raise CkError(rc, lib().ck_last_error().decode())


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _ptr(t):
    """Device pointer of a torch CUDA tensor (or None)."""
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def fp64_peak(device=0):
    v = C.c_double(0)
    _check(lib().ck_fp64_peak(int(device), C.byref(v), None))
    return v.value


def parse_mechanism(text):
    """CHEMKIN-II style text -> dict with the keys of ck_mech_desc (+ species_names, elements), via ck_mech_parse."""
    L = lib()
    h = C.c_void_p()
    _check(L.ck_mech_parse(text.encode(), C.byref(h)))
    try:
        d = L.ck_parsed_desc(h).contents
        K, R, E = d.n_species, d.n_reactions, d.n_elements
        arr = lambda ptr, n, dt: np.ctypeslib.as_array(ptr, shape=(n,)).astype(dt).copy() if n else np.zeros(0, dt)
        out = dict(n_species=K, n_reactions=R, n_elements=E,
                   mol_wt=arr(d.mol_wt, K, np.float64), elem_comp=arr(d.elem_comp, K * E, np.int32).reshape(K, E),
                   nasa_lo=arr(d.nasa_lo, 7 * K, np.float64).reshape(K, 7), nasa_hi=arr(d.nasa_hi, 7 * K, np.float64).reshape(K, 7),
                   t_mid=arr(d.t_mid, K, np.float64), reac_ptr=arr(d.reac_ptr, R + 1, np.int32), prod_ptr=arr(d.prod_ptr, R + 1, np.int32),
                   eff_ptr=arr(d.eff_ptr, R + 1, np.int32), A=arr(d.A, R, np.float64), beta=arr(d.beta, R, np.float64),
                   Ea=arr(d.Ea, R, np.float64), reversible=arr(d.reversible, R, np.uint8), type=arr(d.type, R, np.uint8),
                   A0=arr(d.A0, R, np.float64), beta0=arr(d.beta0, R, np.float64), Ea0=arr(d.Ea0, R, np.float64),
                   troe=arr(d.troe, 4 * R, np.float64).reshape(R, 4))
        nr, npd, ne = int(out["reac_ptr"][-1]), int(out["prod_ptr"][-1]), int(out["eff_ptr"][-1])
        out.update(reac_spec=arr(d.reac_spec, nr, np.int32), reac_nu=arr(d.reac_nu, nr, np.int32),
                   prod_spec=arr(d.prod_spec, npd, np.int32), prod_nu=arr(d.prod_nu, npd, np.int32),
                   eff_spec=arr(d.eff_spec, ne, np.int32), eff_val=arr(d.eff_val, ne, np.float64))
        buf = C.create_string_buffer(64)
        names = []
        for what, n in ((0, K), (1, E)):
            lst = []
            for i in range(n):
                _check(L.ck_parsed_name(h, what, i, buf, 64))
                lst.append(buf.value.decode())
            names.append(lst)
        out["species_names"], out["elements"] = names
        return out
    finally:
        L.ck_parsed_free(h)


def lu_solve_batched(A, b):
    """Solve A[r] x[r] = b[r] for a batch of dense systems (torch CUDA tensors (n, N, N), (n, N)); returns (x, status)."""
    import torch
    n, N = A.shape[0], A.shape[1]
    A = A.contiguous(); b = b.contiguous()
    x = torch.empty_like(b); st = torch.zeros(n, dtype=torch.int32, device=A.device)
    _check(lib().ck_lu_solve_batched(int(N), C.c_int64(n), _ptr(A), _ptr(b), _ptr(x), _ptr(st), _stream()))
    return x, st


def fp64_mma_peak(device=0):
    v = C.c_double(0)
    _check(lib().ck_fp64_mma_peak(int(device), C.byref(v), None))
    return v.value


class Mechanism:
    """A kinetic model loaded on one GPU.  `d` is a dict whose keys mirror ck_mech_desc."""

    def __init__(self, d, device=0, const_volume=False):
        """const_volume: constant-volume reactors -- every `p` argument then holds the mass density (include/ck.h)."""
        L = lib()
        k = self._keep = dict(
            mol_wt=_np(d["mol_wt"], np.float64), elem_comp=_np(d["elem_comp"], np.int32),
            nasa_lo=_np(d["nasa_lo"], np.float64), nasa_hi=_np(d["nasa_hi"], np.float64), t_mid=_np(d["t_mid"], np.float64),
            reac_ptr=_np(d["reac_ptr"], np.int32), reac_spec=_np(d["reac_spec"], np.int32), reac_nu=_np(d["reac_nu"], np.int32),
            prod_ptr=_np(d["prod_ptr"], np.int32), prod_spec=_np(d["prod_spec"], np.int32), prod_nu=_np(d["prod_nu"], np.int32),
            A=_np(d["A"], np.float64), beta=_np(d["beta"], np.float64), Ea=_np(d["Ea"], np.float64),
            reversible=_np(d["reversible"], np.uint8), type=_np(d["type"], np.uint8),
            A0=_np(d["A0"], np.float64), beta0=_np(d["beta0"], np.float64), Ea0=_np(d["Ea0"], np.float64),
            troe=_np(d["troe"], np.float64), eff_ptr=_np(d["eff_ptr"], np.int32), eff_spec=_np(d["eff_spec"], np.int32),
            eff_val=_np(d["eff_val"], np.float64))
        desc = MechDesc()
        desc.struct_size = C.sizeof(MechDesc)
        desc.n_species, desc.n_reactions, desc.n_elements = int(d["n_species"]), int(d["n_reactions"]), int(d["n_elements"])
        for name, typ in MechDesc._fields_[4:]:
            a = k[name]
            setattr(desc, name, a.ctypes.data_as(typ) if a.size else C.cast(None, typ))
        h = C.c_void_p()
        _check(L.ck_mech_load(C.byref(desc), int(device), C.byref(h)))
        self.h = h
        if const_volume:
            _check(L.ck_mech_set_reactor(h, 1))
        self.device = int(device)
        self.K, self.R = desc.n_species, desc.n_reactions
        self.N = self.K + 1

    def close(self):
        if getattr(self, "h", None):
            lib().ck_mech_free(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def rhs_kernel_name(self, n):
        b, t = C.c_int32(0), C.c_int32(0)
        _check(lib().ck_rhs_variant(self.h, C.c_int64(n), C.byref(b), C.byref(t)))
        return f"ck::rhs_kernel_tmem<{b.value}>" if t.value else f"ck::rhs_kernel<{b.value}>"

    def rhs_slots(self):
        v = C.c_double(0)
        _check(lib().ck_rhs_slots(self.h, C.byref(v)))
        return v.value

    # ---- device-pointer entry points (torch CUDA tensors, component-major (N, ld)) ---------------------
    def rhs(self, y, p, out=None):
        import torch
        n = y.shape[1]
        assert y.dtype == torch.float64 and y.is_cuda and y.shape[0] == self.N and y.stride(1) == 1
        if out is None:
            out = torch.empty_like(y)
        _check(lib().ck_rhs(self.h, C.c_int64(n), _ptr(y), C.c_int64(y.stride(0) if n else 0), _ptr(p), _ptr(out),
                            C.c_int64(out.stride(0) if n else 0), _stream()))
        return out

    def jac(self, y, p, mode=CK_JAC_ANALYTIC, h=0.0, rtol=1e-6, atol=1e-10, out=None):
        import torch
        n = y.shape[1]
        if out is None:
            out = torch.empty((self.N * self.N, n), dtype=torch.float64, device=y.device)
        _check(lib().ck_jac(self.h, C.c_int64(n), _ptr(y), C.c_int64(y.stride(0) if n else 0), _ptr(p), int(mode),
                            C.c_double(h), C.c_double(rtol), C.c_double(atol), _ptr(out),
                            C.c_int64(out.stride(0) if n else 0), _stream()))
        return out.view(self.N, self.N, n)

    def jac_batched(self, y, p, out=None):
        """Analytic Jacobian, thread-per-reactor kernel (large batches); same layout as jac()."""
        import torch
        n = y.shape[1]
        if out is None:
            out = torch.empty((self.N * self.N, n), dtype=torch.float64, device=y.device)
        ws = torch.empty(max(self.workspace_bytes(CK_OP_JAC, n), 8), dtype=torch.uint8, device=y.device)
        _check(lib().ck_jac_batched(self.h, C.c_int64(n), _ptr(y), C.c_int64(y.stride(0) if n else 0), _ptr(p), _ptr(out),
                                    C.c_int64(out.stride(0) if n else 0), _ptr(ws), C.c_size_t(ws.numel()), _stream()))
        return out.view(self.N, self.N, n)

    def jac_batched_static(self, y, p, out):
        """ck_jac_batched_static: no allocation inside the call; `out` (N*N, n) must be supplied by the caller."""
        n = y.shape[1]
        _check(lib().ck_jac_batched_static(self.h, C.c_int64(n), _ptr(y), C.c_int64(y.stride(0) if n else 0), _ptr(p), _ptr(out),
                                           C.c_int64(out.stride(0) if n else 0), _stream()))
        return out.view(self.N, self.N, n)

    def jac_static_max_reactors(self):
        v = C.c_int64(0)
        _check(lib().ck_jac_static_max_reactors(self.h, C.byref(v)))
        return v.value

    def workspace_bytes(self, op, n):
        v = C.c_size_t(0)
        _check(lib().ck_workspace_bytes(self.h, int(op), C.c_int64(n), C.byref(v)))
        return v.value

    def integrate(self, solver, y, p, dt, rtol=1e-6, atol=1e-10, jac_mode=CK_JAC_ANALYTIC, h0=0.0, max_steps=0,
                  flags=0, want_report=True, ws=None):
        """Advance y (N, n) in place over dt.  solver 'ros' | 'rkf45'.  Returns dict of per-reactor tensors + report."""
        import torch
        op = CK_OP_ROS if solver == "ros" else CK_OP_RKF45
        n = y.shape[1]
        dev = y.device
        na = torch.zeros(n, dtype=torch.int32, device=dev); nr = torch.zeros_like(na); st = torch.zeros_like(na)
        hl = torch.zeros(n, dtype=torch.float64, device=dev)
        nbytes = self.workspace_bytes(op, n)
        if ws is None or ws.numel() < nbytes:
            ws = torch.empty(max(nbytes, 8), dtype=torch.uint8, device=dev)
        o = Opts(C.sizeof(Opts), int(jac_mode), rtol, atol, h0, int(max_steps), int(flags))
        rep = Report()
        fn = lib().ck_integrate_ros if op == CK_OP_ROS else lib().ck_integrate_rkf45
        _check(fn(self.h, C.c_int64(n), _ptr(y), C.c_int64(y.stride(0) if n else 0), _ptr(p), C.c_double(dt), C.byref(o),
                  _ptr(na), _ptr(nr), _ptr(st), _ptr(hl), _ptr(ws), C.c_size_t(ws.numel()),
                  C.byref(rep) if want_report else None, _stream()))
        return dict(y=y, n_accept=na, n_reject=nr, status=st, h_last=hl, report=rep.as_dict() if want_report else None,
                    ws=ws)

    @staticmethod
    def waste(n_accept, n_reject, P, tasks=1):
        """Eq. 20 per work unit of width P (static mapping, `tasks` reactors per lane) from device step counts."""
        import torch
        n = n_accept.numel()
        per = P * tasks
        W = torch.empty((n + per - 1) // per if per > 0 else 0, dtype=torch.float64, device=n_accept.device)
        _check(lib().ck_waste_tasks(C.c_int64(n), _ptr(n_accept), _ptr(n_reject) if n_reject is not None else None, int(P),
                                    int(tasks), _ptr(W), _stream()))
        return W

    # ---- host-pointer entry points (numpy arrays; transfers inside the call) ---------------------------
    def rhs_host(self, y, p, out=None):
        assert y.dtype == np.float64 and y.flags.c_contiguous and y.shape[0] == self.N
        n = y.shape[1]
        if out is None:
            out = np.empty_like(y)
        _check(lib().ck_rhs_host(self.h, C.c_int64(n), y.ctypes.data_as(_PD), C.c_int64(n), p.ctypes.data_as(_PD),
                                 out.ctypes.data_as(_PD), C.c_int64(n)))
        return out

    def integrate_host(self, solver, y, p, dt, rtol=1e-6, atol=1e-10, jac_mode=CK_JAC_ANALYTIC, h0=0.0, max_steps=0,
                       flags=0):
        op = CK_OP_ROS if solver == "ros" else CK_OP_RKF45
        assert y.dtype == np.float64 and y.flags.c_contiguous and y.shape[0] == self.N
        n = y.shape[1]
        na = np.zeros(n, np.int32); nr = np.zeros(n, np.int32); st = np.zeros(n, np.int32); hl = np.zeros(n)
        o = Opts(C.sizeof(Opts), int(jac_mode), rtol, atol, h0, int(max_steps), int(flags))
        rep = Report()
        _check(lib().ck_integrate_host(self.h, op, C.c_int64(n), y.ctypes.data_as(_PD), C.c_int64(n),
                                       p.ctypes.data_as(_PD), C.c_double(dt), C.byref(o), na.ctypes.data_as(_PI),
                                       nr.ctypes.data_as(_PI), st.ctypes.data_as(_PI), hl.ctypes.data_as(_PD),
                                       C.byref(rep)))
        return dict(y=y, n_accept=na, n_reject=nr, status=st, h_last=hl, report=rep.as_dict())
