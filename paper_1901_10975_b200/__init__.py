"""paper_1901_10975_b200 -- thin Python binding of libcn (include/cn.h).

Argument marshalling only: every step of the path (event delivery, nrn_cur, Hines solve, voltage
update, nrn_state, threshold detection) runs in the CUDA kernels of
csrc/cn_tape.cuh (interleaved kernel) and csrc/cn_device.cuh (warp-cooperative kernel, event
delivery, point processes).  There is no CPU fallback; without the built library or a CUDA device the
calls raise.  This package never imports the oracle.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "libcn.so"

CN_OK = 0
ERRORS = {-1: "CN_ERR_ARG", -2: "CN_ERR_TOPOLOGY", -3: "CN_ERR_MECH", -4: "CN_ERR_NETCON",
          -5: "CN_ERR_DT", -6: "CN_ERR_CUDA", -7: "CN_ERR_OVERFLOW", -8: "CN_ERR_NOMEM",
          -9: "CN_ERR_UNSUPPORTED"}

# mechanism name -> (CN_* type id, parameter row order, global order); see include/cn.h
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

NOALLOC_MAX_INSTANCES = 65536   # include/cn.h CN_NOALLOC_MAX_INSTANCES

EXPORTS = ("cn_model_create", "cn_model_create_opts", "cn_run", "cn_run_async", "cn_sync", "cn_set_stream", "cn_get_v",
           "cn_get_spikes", "cn_set_probes", "cn_get_trace", "cn_get_state", "cn_get_state_noalloc", "cn_steps_done",
           "cn_launch_count", "cn_last_run_ms", "cn_set_kernel_timing", "cn_select_timed_kernel", "cn_get_kernel_timing", "cn_get_layout_info", "cn_get_run_info", "cn_set_spike_capacity",
           "cn_checkpoint_size", "cn_checkpoint_save", "cn_checkpoint_load",
           "cn_model_destroy", "cn_last_error")


class CnError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")
        self.code = code


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
    """Load libcn.so (built in-tree by build.py); fails loudly when it is missing."""
    global _lib
    if _lib is None:
        if not _SO.exists():
            raise ImportError(f"{_SO} is missing: run `python -m paper_1901_10975_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(str(_SO))
        vp = C.c_void_p
        L.cn_model_create.argtypes = [C.POINTER(_Desc), C.POINTER(vp)]
        L.cn_model_create_opts.argtypes = [C.POINTER(_Desc), C.c_char_p, C.POINTER(vp)]
        L.cn_run.argtypes = [vp, C.c_double, C.c_double]
        L.cn_run_async.argtypes = [vp, C.c_double, C.c_double]
        L.cn_sync.argtypes = [vp]
        L.cn_set_stream.argtypes = [vp, vp]
        L.cn_get_v.argtypes = [vp, vp, C.c_int64]
        L.cn_get_spikes.argtypes = [vp, vp, vp, C.c_int64, C.POINTER(C.c_int64)]
        L.cn_set_probes.argtypes = [vp, vp, C.c_int64, C.c_int64]
        L.cn_get_trace.argtypes = [vp, vp, C.c_int64, C.POINTER(C.c_int64)]
        L.cn_get_state.argtypes = [vp, C.c_int32, C.c_int32, vp, C.c_int64]
        L.cn_get_state_noalloc.argtypes = [vp, C.c_int32, C.c_int32, vp, C.c_int64]
        L.cn_steps_done.restype = C.c_int64
        L.cn_steps_done.argtypes = [vp]
        L.cn_launch_count.restype = C.c_int64
        L.cn_launch_count.argtypes = [vp]
        L.cn_last_run_ms.argtypes = [vp, C.POINTER(C.c_double)]
        L.cn_set_kernel_timing.argtypes = [vp, C.c_int32, C.c_int32]
        L.cn_select_timed_kernel.argtypes = [vp, C.c_int32]
        L.cn_get_kernel_timing.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.cn_get_layout_info.argtypes = [vp, vp]
        L.cn_get_run_info.argtypes = [vp, vp]
        L.cn_set_spike_capacity.argtypes = [vp, C.c_int64]
        L.cn_checkpoint_size.argtypes = [vp, C.POINTER(C.c_int64)]
        L.cn_checkpoint_save.argtypes = [vp, vp, C.c_int64]
        L.cn_checkpoint_load.argtypes = [vp, vp, C.c_int64]
        L.cn_model_destroy.restype = None
        L.cn_model_destroy.argtypes = [vp]
        L.cn_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(rc):
    if rc != CN_OK:
        raise CnError(rc, lib().cn_last_error().decode())


def _arr(x, dtype):
    return np.ascontiguousarray(np.asarray(x, dtype=dtype))


def _ptr(a):
    return a.ctypes.data if a.size else None


def marshal(desc: dict):
    """dict description (see cn_workloads) -> (cn_model_desc, keep-alive list, bytes)."""
    keep = []

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
    keep.append(mechs)
    nc = desc.get("netcons") or {}
    stim = desc.get("stim") or {}
    d = _Desc()
    d.n_cell = int(len(desc["cell_first"]) - 1)
    d.n_node = int(len(desc["parent"]))
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
    nbytes = sum(a.nbytes for a in keep if isinstance(a, np.ndarray))
    return d, keep, nbytes


class Model:
    """cn_model_create / cn_run / cn_get_v / cn_get_spikes with the same names as the C ABI."""

    def __init__(self, desc: dict, marshalled=None, stream=None, options=None):
        """options: dict or "key=value;..." string for cn_model_create_opts (include/cn.h)."""
        L = lib()
        if isinstance(options, dict):
            options = ";".join(f"{k}={v}" for k, v in options.items())
        d, keep, self.desc_bytes = marshalled if marshalled is not None else marshal(desc)
        self.n_node = int(d.n_node)
        self.n_cell = int(d.n_cell)
        self.mech_n = [int(len(m["node"])) for m in desc["mechs"]] if desc is not None else []
        h = C.c_void_p()
        self._h = None
        if options:
            _check(L.cn_model_create_opts(C.byref(d), options.encode(), C.byref(h)))
        else:
            _check(L.cn_model_create(C.byref(d), C.byref(h)))
        self._h = h
        self._n_probe = 0
        if stream is not None:
            self.set_stream(stream)

    def __del__(self):
        try:
            self.destroy()
        except Exception:  # interpreter shutdown: the module globals may be gone already
            pass

    def destroy(self):
        h = getattr(self, "_h", None)
        if h:
            self._h = None
            lib().cn_model_destroy(h)

    def set_stream(self, cuda_stream_handle: int):
        _check(lib().cn_set_stream(self._h, C.c_void_p(int(cuda_stream_handle))))

    def run(self, tstop, dt):
        _check(lib().cn_run(self._h, float(tstop), float(dt)))

    def run_async(self, tstop, dt):
        _check(lib().cn_run_async(self._h, float(tstop), float(dt)))

    def sync(self):
        _check(lib().cn_sync(self._h))

    def get_v(self, out=None):
        if out is None:
            out = np.empty(self.n_node, dtype=np.float64)
        _check(lib().cn_get_v(self._h, _ptr(out), self.n_node))
        return out

    def get_spikes(self):
        n = C.c_int64()
        _check(lib().cn_get_spikes(self._h, None, None, 0, C.byref(n)))
        gid = np.empty(n.value, dtype=np.int32)
        step = np.empty(n.value, dtype=np.int64)
        if n.value:
            _check(lib().cn_get_spikes(self._h, _ptr(gid), _ptr(step), n.value, C.byref(n)))
        return gid, step

    def set_probes(self, nodes, max_steps):
        nodes = _arr(nodes, np.int32)
        _check(lib().cn_set_probes(self._h, _ptr(nodes), len(nodes), int(max_steps)))
        self._n_probe = len(nodes)

    def get_trace(self):
        n = C.c_int64()
        _check(lib().cn_get_trace(self._h, None, 0, C.byref(n)))
        out = np.empty((n.value, self._n_probe), dtype=np.float64)
        if out.size:
            _check(lib().cn_get_trace(self._h, _ptr(out), n.value, C.byref(n)))
        return out

    def get_state(self, t, s):
        out = np.empty(self.mech_n[t], dtype=np.float64)
        _check(lib().cn_get_state(self._h, t, s, _ptr(out), len(out)))
        return out

    def get_state_noalloc(self, t, s, out=None):
        """cn_get_state through the library's static device scratch (no allocation in the call;
        tables of at most NOALLOC_MAX_INSTANCES instances); `out`: caller's buffer."""
        if out is None:
            out = np.empty(self.mech_n[t], dtype=np.float64)
        _check(lib().cn_get_state_noalloc(self._h, t, s, _ptr(out), len(out)))
        return out

    @property
    def steps_done(self):
        return lib().cn_steps_done(self._h)

    @property
    def launch_count(self):
        return lib().cn_launch_count(self._h)

    def last_run_ms(self):
        ms = C.c_double()
        _check(lib().cn_last_run_ms(self._h, C.byref(ms)))
        return ms.value

    def set_kernel_timing(self, every, max_samples=4096):
        _check(lib().cn_set_kernel_timing(self._h, int(every), int(max_samples)))

    def select_timed_kernel(self, which):
        _check(lib().cn_select_timed_kernel(self._h, {"step": 0, "pp": 1, "deliver": 2}[which]))

    def get_kernel_timing(self):
        ms, n = C.c_double(), C.c_int64()
        _check(lib().cn_get_kernel_timing(self._h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def layout_info(self):
        a = np.zeros(8, dtype=np.int64)
        _check(lib().cn_get_layout_info(self._h, _ptr(a)))
        return {"n_class": int(a[0]), "n_group": int(a[1]), "warp_smem_bytes": int(a[2]),
                "max_rounds": int(a[3]), "n_tape_group": int(a[4]), "tape_bytes": int(a[5]),
                "tape_smem_bytes": int(a[6]), "tape_warps": int(a[7]) & 255,
                "tape_ctas": (int(a[7]) >> 8) & 0xFFFF, "tape_sys_rows": int(a[7]) >> 24}

    def run_info(self):
        a = np.zeros(4, dtype=np.int64)
        _check(lib().cn_get_run_info(self._h, _ptr(a)))
        return {"mode": {-1: "unknown", 0: "per-step", 1: "window", 2: "onchip-window"}[int(a[0])],
                "graph_replays": int(a[1]), "window_steps": int(a[2]), "window_ctas": int(a[3])}

    def checkpoint(self) -> np.ndarray:
        """cn_checkpoint_size + cn_checkpoint_save into a fresh uint8 array."""
        n = C.c_int64()
        _check(lib().cn_checkpoint_size(self._h, C.byref(n)))
        buf = np.empty(n.value, dtype=np.uint8)
        _check(lib().cn_checkpoint_save(self._h, _ptr(buf), n.value))
        return buf

    def restore(self, buf: np.ndarray):
        buf = np.ascontiguousarray(buf, dtype=np.uint8)
        _check(lib().cn_checkpoint_load(self._h, _ptr(buf), buf.size))

    def set_spike_capacity(self, cap):
        _check(lib().cn_set_spike_capacity(self._h, int(cap)))
