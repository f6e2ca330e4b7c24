"""ctypes binding of the CPU oracle (oracle/cn_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It
never imports paper_1901_10975_b200 and shares no code with the CUDA path.

The oracle restates the per-dt operations of PAPER.md L62-68 (see the header
of cn_oracle.c); model descriptions are the plain dicts produced by
cn_workloads (which holds none of the method's arithmetic).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "liborc.so"

# mechanism name -> (oracle type id, per-instance param order, global order)
MECH = {
    "pas": (1, ("g", "e"), ()),
    "hh": (2, ("gnabar", "gkbar", "gl", "el"), ("ena", "ek")),
    "expsyn": (3, ("tau", "e"), ()),
    "exp2syn": (4, ("tau1", "tau2", "e"), ()),
    "iclamp": (5, ("del", "dur", "amp"), ()),
    "hhform": (6, ("gbar",), ("p", "q", "E", "to_ica",
                              "m_vh", "m_k", "m_t0", "m_t1", "m_vt", "m_s",
                              "h_vh", "h_k", "h_t0", "h_t1", "h_vt", "h_s")),
    "sk": (7, ("gbar",), ("E", "Kd", "n", "tau_z")),
    "cadyn": (8, (), ("gamma", "depth", "tau_d", "cai_min")),
    "ampanmda": (9, (), ("tau_r_A", "tau_d_A", "tau_r_N", "tau_d_N", "r_nmda", "mg", "e")),
    "gap": (10, ("g", "peer"), ()),
}
STATES = {
    "pas": (), "hh": ("m", "h", "n"), "expsyn": ("g",), "exp2syn": ("A", "B"), "iclamp": (),
    "hhform": ("m", "h"), "sk": ("z",), "cadyn": (), "ampanmda": ("A_A", "B_A", "A_N", "B_N"), "gap": (),
}


def build(force: bool = False) -> Path:
    """gcc -O2 -ffp-contract=off (R22): plain IEEE fp64, no FMA contraction."""
    src = _HERE / "cn_oracle.c"
    hdr = _HERE / "cn_oracle.h"
    if (not force and _SO.exists()
            and _SO.stat().st_mtime >= max(src.stat().st_mtime, hdr.stat().st_mtime)):
        return _SO
    tmp = _SO.with_suffix(f".so.tmp{os.getpid()}")
    subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-std=c99", "-fPIC", "-shared",
                           "-o", str(tmp), str(src), "-lm"])
    os.replace(tmp, _SO)
    return _SO


class _Mech(C.Structure):
    _fields_ = [("type", C.c_int32), ("n", C.c_int64), ("node", C.c_void_p),
                ("n_param", C.c_int32), ("param", C.c_void_p),
                ("n_global", C.c_int32), ("glob", C.c_void_p)]


class _Desc(C.Structure):
    _fields_ = [("n_cell", C.c_int32), ("n_node", C.c_int64), ("cell_first", C.c_void_p),
                ("parent", C.c_void_p), ("area", C.c_void_p), ("ri", C.c_void_p),
                ("cm", C.c_void_p), ("v_init", C.c_double), ("celsius", C.c_double),
                ("n_mech", C.c_int32), ("mech", C.c_void_p),
                ("n_netcon", C.c_int64), ("nc_src", C.c_void_p), ("nc_tgt_mech", C.c_void_p),
                ("nc_tgt_inst", C.c_void_p), ("nc_weight", C.c_void_p), ("nc_delay", C.c_void_p),
                ("thr", C.c_void_p), ("n_stim", C.c_int64), ("stim_gid", C.c_void_p),
                ("stim_t", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        dp = C.POINTER(C.c_double)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Desc)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_run.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orc_steps_done.restype = C.c_int64
        L.orc_steps_done.argtypes = [C.c_void_p]
        L.orc_get_v.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_n_spikes.restype = C.c_int64
        L.orc_n_spikes.argtypes = [C.c_void_p]
        L.orc_get_spikes.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_min_margin.restype = C.c_double
        L.orc_min_margin.argtypes = [C.c_void_p]
        L.orc_set_probes.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_trace_steps.restype = C.c_int64
        L.orc_trace_steps.argtypes = [C.c_void_p]
        L.orc_get_trace.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_get_state.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_int64]
        L.orc_get_cai.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_get_ab.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_get_last_system.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                          C.c_int64]
        L.orc_assemble_tree.restype = None
        L.orc_assemble_tree.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                        C.c_void_p, C.c_double, C.c_void_p, C.c_void_p,
                                        C.c_void_p]
        L.orc_hines.restype = None
        L.orc_hines.argtypes = [C.c_int64] + [C.c_void_p] * 5
        L.orc_hh_rates.restype = None
        L.orc_hh_rates.argtypes = [C.c_double, C.c_double, dp]
        L.orc_hhform_gate.restype = None
        L.orc_hhform_gate.argtypes = [C.c_double, dp, dp]
        L.orc_n_state.argtypes = [C.c_int32]
        L.orc_n_param.argtypes = [C.c_int32]
        L.orc_mech_init.restype = None
        L.orc_mech_init.argtypes = [C.c_int32, dp, dp, dp, C.c_double, C.c_double]
        L.orc_mech_cur.restype = None
        L.orc_mech_cur.argtypes = [C.c_int32, dp, dp, dp, C.c_double, C.c_double, C.c_double,
                                   dp, dp, dp]
        L.orc_mech_state.restype = None
        L.orc_mech_state.argtypes = [C.c_int32, dp, dp, dp, C.c_double, C.c_double, C.c_double,
                                     dp, C.c_double]
        L.orc_mech_receive.restype = None
        L.orc_mech_receive.argtypes = [C.c_int32, dp, dp, dp, C.c_double]
        L.orc_exp2syn_factor.restype = C.c_double
        L.orc_exp2syn_factor.argtypes = [C.c_double, C.c_double]
        _lib = L
    return _lib


def _arr(x, dtype):
    return np.ascontiguousarray(np.asarray(x, dtype=dtype))


def _ptr(a):
    return a.ctypes.data if a.size else None


def _darr(xs):
    a = (C.c_double * max(len(xs), 1))()
    for i, x in enumerate(xs):
        a[i] = float(x)
    return a


# ---- single-instance mechanism calls (used by the pins) --------------------------------------

def _glob_vec(name, globals_):
    _, _, gorder = MECH[name]
    return _darr([globals_[k] for k in gorder])


def _par_vec(name, params):
    _, porder, _ = MECH[name]
    return _darr([params[k] for k in porder])


def mech_init(name, params, globals_, v, celsius=6.3):
    S = _darr([0.0] * 8)
    lib().orc_mech_init(MECH[name][0], _glob_vec(name, globals_), _par_vec(name, params), S, v,
                        celsius)
    return [S[i] for i in range(len(STATES[name]))]


def mech_cur(name, params, globals_, states, v, cai=1e-4, t_mid=0.0):
    i, g, ica = C.c_double(), C.c_double(), C.c_double()
    lib().orc_mech_cur(MECH[name][0], _glob_vec(name, globals_), _par_vec(name, params),
                       _darr(list(states) + [0.0] * 8), v, cai, t_mid,
                       C.byref(i), C.byref(g), C.byref(ica))
    return i.value, g.value, ica.value


def mech_state(name, params, globals_, states, v, dt, cai=1e-4, ica=0.0, celsius=6.3):
    S = _darr(list(states) + [0.0] * 8)
    c = C.c_double(cai)
    lib().orc_mech_state(MECH[name][0], _glob_vec(name, globals_), _par_vec(name, params), S, v,
                         dt, celsius, C.byref(c), ica)
    return [S[i] for i in range(len(states))], c.value


def mech_receive(name, params, globals_, states, w):
    S = _darr(list(states) + [0.0] * 8)
    lib().orc_mech_receive(MECH[name][0], _glob_vec(name, globals_), _par_vec(name, params), S, w)
    return [S[i] for i in range(len(states))]


def hh_rates(v, celsius=6.3):
    out = (C.c_double * 6)()
    lib().orc_hh_rates(v, celsius, out)
    return list(out)


def hhform_gate(v, g6):
    out = (C.c_double * 2)()
    lib().orc_hhform_gate(v, _darr(g6), out)
    return out[0], out[1]


def exp2syn_factor(tau1, tau2):
    return lib().orc_exp2syn_factor(tau1, tau2)


def hines(parent, a, b, d, rhs):
    """O6+O7 on copies; returns the solution."""
    parent = _arr(parent, np.int32)
    a, b = _arr(a, np.float64), _arr(b, np.float64)
    d, rhs = _arr(d, np.float64).copy(), _arr(rhs, np.float64).copy()
    lib().orc_hines(len(parent), _ptr(parent), _ptr(a), _ptr(b), _ptr(d), _ptr(rhs))
    return rhs


def assemble_tree(parent, a, b, cm, dt, v, d, rhs):
    """O4+O5 on copies; returns (d, rhs)."""
    parent = _arr(parent, np.int32)
    a, b, cm, v = (_arr(x, np.float64) for x in (a, b, cm, v))
    d, rhs = _arr(d, np.float64).copy(), _arr(rhs, np.float64).copy()
    lib().orc_assemble_tree(len(parent), _ptr(parent), _ptr(a), _ptr(b), _ptr(cm), dt, _ptr(v),
                            _ptr(d), _ptr(rhs))
    return d, rhs


# ---- the model ---------------------------------------------------------------------------------

class OracleModel:
    def __init__(self, desc: dict):
        L = lib()
        keep = []
        self.n_node = int(len(desc["parent"]))
        self.n_cell = int(len(desc["cell_first"]) - 1)
        self.mech_names = [m["type"] for m in desc["mechs"]]
        self.mech_n = [int(len(m["node"])) for m in desc["mechs"]]

        def k(a):
            keep.append(a)
            return _ptr(a)

        mechs = (_Mech * max(len(desc["mechs"]), 1))()
        for j, m in enumerate(desc["mechs"]):
            tid, porder, gorder = MECH[m["type"]]
            n = len(m["node"])
            par = np.zeros((len(porder), n), dtype=np.float64)
            for pi, pn in enumerate(porder):
                par[pi, :] = np.asarray(m["params"][pn], dtype=np.float64)
            gl = np.array([float(m.get("globals", {})[g]) for g in gorder], dtype=np.float64)
            mechs[j].type = tid
            mechs[j].n = n
            mechs[j].node = k(_arr(m["node"], np.int32))
            mechs[j].n_param = len(porder)
            mechs[j].param = k(np.ascontiguousarray(par))
            mechs[j].n_global = len(gorder)
            mechs[j].glob = k(gl)
        nc = desc.get("netcons") or {}
        stim = desc.get("stim") or {}
        d = _Desc()
        d.n_cell = self.n_cell
        d.n_node = self.n_node
        d.cell_first = k(_arr(desc["cell_first"], np.int64))
        d.parent = k(_arr(desc["parent"], np.int32))
        d.area = k(_arr(desc["area"], np.float64))
        d.ri = k(_arr(desc["ri"], np.float64))
        d.cm = k(_arr(desc["cm"], np.float64))
        d.v_init = float(desc.get("v_init", -65.0))
        d.celsius = float(desc.get("celsius", 6.3))
        d.n_mech = len(desc["mechs"])
        d.mech = C.cast(mechs, C.c_void_p).value
        d.n_netcon = len(nc.get("src", ()))
        d.nc_src = k(_arr(nc.get("src", ()), np.int32))
        d.nc_tgt_mech = k(_arr(nc.get("tgt_mech", ()), np.int32))
        d.nc_tgt_inst = k(_arr(nc.get("tgt_inst", ()), np.int64))
        d.nc_weight = k(_arr(nc.get("weight", ()), np.float64))
        d.nc_delay = k(_arr(nc.get("delay", ()), np.float64))
        d.thr = k(_arr(desc["thr"], np.float64))
        d.n_stim = len(stim.get("gid", ()))
        d.stim_gid = k(_arr(stim.get("gid", ()), np.int32))
        d.stim_t = k(_arr(stim.get("t", ()), np.float64))
        self._h = L.orc_create(C.byref(d))
        if not self._h:
            raise ValueError("oracle: invalid model description")
        self._n_probe = 0

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            lib().orc_destroy(h)
            self._h = None

    def run(self, tstop, dt):
        if lib().orc_run(self._h, float(tstop), float(dt)) != 0:
            raise ValueError("oracle: orc_run failed (dt changed, dt <= 0 or a delay < 1 step)")

    @property
    def steps_done(self):
        return lib().orc_steps_done(self._h)

    def get_v(self):
        out = np.empty(self.n_node, dtype=np.float64)
        assert lib().orc_get_v(self._h, _ptr(out), self.n_node) == 0
        return out

    def get_spikes(self):
        n = lib().orc_n_spikes(self._h)
        gid = np.empty(n, dtype=np.int32)
        step = np.empty(n, dtype=np.int64)
        lib().orc_get_spikes(self._h, _ptr(gid), _ptr(step), n)
        return gid, step

    @property
    def min_margin(self):
        return lib().orc_min_margin(self._h)

    def set_probes(self, nodes):
        nodes = _arr(nodes, np.int32)
        assert lib().orc_set_probes(self._h, _ptr(nodes), len(nodes)) == 0
        self._n_probe = len(nodes)

    def get_trace(self):
        n = lib().orc_trace_steps(self._h)
        out = np.empty((n, self._n_probe), dtype=np.float64)
        lib().orc_get_trace(self._h, _ptr(out), n)
        return out

    def get_state(self, t, s):
        out = np.empty(self.mech_n[t], dtype=np.float64)
        r = lib().orc_get_state(self._h, t, s, _ptr(out), len(out))
        assert r >= 0
        return out

    def get_cai(self):
        out = np.empty(self.n_node, dtype=np.float64)
        lib().orc_get_cai(self._h, _ptr(out), self.n_node)
        return out

    def get_ab(self):
        a = np.empty(self.n_node, dtype=np.float64)
        b = np.empty(self.n_node, dtype=np.float64)
        lib().orc_get_ab(self._h, _ptr(a), _ptr(b), self.n_node)
        return a, b

    def get_last_system(self):
        d = np.empty(self.n_node, dtype=np.float64)
        rhs = np.empty(self.n_node, dtype=np.float64)
        sol = np.empty(self.n_node, dtype=np.float64)
        assert lib().orc_get_last_system(self._h, _ptr(d), _ptr(rhs), _ptr(sol), self.n_node) == 0
        return d, rhs, sol
