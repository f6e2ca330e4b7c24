"""Seeded synthetic model descriptions shaped like BASELINE.json's configs.

These are INPUT generators only: topology, geometry -> (area, axial resistance),
mechanism placement / parameters, NetCons.  They hold none of the method's
arithmetic (no currents, no matrix, no solve) and serve both the oracle and the
CUDA path.  The paper's benchmark models (Table 1) are not
reproduced; only their published sizes and shapes are used.

A description is a plain dict:
  cell_first int64[n_cell+1], parent int32[N] (global, -1 roots), area[N] um2,
  ri[N] MOhm (node<->parent), cm[N] uF/cm2, v_init, celsius,
  mechs: list of {type, node int32[n], params {name: f64[n]}, globals {name: float}},
  netcons: {src int32, tgt_mech int32, tgt_inst int64, weight f64 uS, delay f64 ms},
  thr f64[n_cell], stim: {gid int32 (>= n_cell), t f64 ms}  (scripted source spikes)
"""
from __future__ import annotations

import hashlib

import numpy as np

from . import rng

HH_SQUID = dict(gnabar=0.12, gkbar=0.036, gl=0.0003, el=-54.3)
HH_GLOBALS = dict(ena=50.0, ek=-77.0)


# ------------------------------------------------------------------------------------------
# geometry (SURVEY 8(c) "Geometry (done by the generator, not the library)")
# ------------------------------------------------------------------------------------------

def geometry(parent_local: np.ndarray, Lc: np.ndarray, diam: np.ndarray, Ra: float):
    """Lateral area (um2) and centre-to-centre axial resistance to the parent (MOhm).

    Lc, diam: [..., n] compartment length / diameter in um; parent_local: [n], -1 for the root.
    """
    area = np.pi * diam * Lc
    rhalf = 1e-2 * Ra * (Lc / 2.0) / (np.pi * diam * diam / 4.0)
    p = np.where(parent_local < 0, 0, parent_local)
    ri = rhalf + np.take(rhalf, p, axis=-1)
    ri = np.where(parent_local < 0, 1.0, ri)  # ignored for roots; kept positive and finite
    return area, ri


def binary_branches(depth: int) -> np.ndarray:
    """Parent-branch index (-1 = attached to soma) of a full binary tree with `depth` levels."""
    par = []
    level = []
    for lv in range(depth):
        cur = []
        for j in range(2 ** (lv + 1)):
            cur.append(len(par))
            par.append(-1 if lv == 0 else level[j // 2])
        level = cur
    return np.array(par, dtype=np.int64)


def expand_branches(branch_parent: np.ndarray, ncomp: np.ndarray):
    """Local parent[] for soma (node 0) + branches laid out in order, proximal to distal.

    The first compartment of a child branch attaches to the LAST compartment of its parent
    branch, or to the soma (R9).  Returns parent_local, branch_of_node (-1 = soma), first, last.
    """
    nb = len(branch_parent)
    first = np.zeros(nb, dtype=np.int64)
    last = np.zeros(nb, dtype=np.int64)
    pos = 1
    for j in range(nb):
        first[j] = pos
        pos += int(ncomp[j])
        last[j] = pos - 1
    n = pos
    parent = np.arange(-1, n - 1, dtype=np.int64)
    branch_of = np.full(n, -1, dtype=np.int64)
    for j in range(nb):
        branch_of[first[j]:last[j] + 1] = j
        parent[first[j]] = 0 if branch_parent[j] < 0 else last[branch_parent[j]]
    parent[0] = -1
    return parent, branch_of, first, last


def _mech(type_, node, params=None, globals_=None):
    return {"type": type_, "node": np.asarray(node, dtype=np.int32),
            "params": {k: np.ascontiguousarray(v, dtype=np.float64)
                       for k, v in (params or {}).items()},
            "globals": dict(globals_ or {})}


def _const(n, x):
    return np.full(int(n), float(x), dtype=np.float64)


def _netcons(src, tgt_mech, tgt_inst, weight, delay):
    return {"src": np.asarray(src, dtype=np.int32), "tgt_mech": np.asarray(tgt_mech, np.int32),
            "tgt_inst": np.asarray(tgt_inst, dtype=np.int64),
            "weight": np.asarray(weight, dtype=np.float64),
            "delay": np.asarray(delay, dtype=np.float64)}


def _no_stim():
    return {"gid": np.zeros(0, np.int32), "t": np.zeros(0, np.float64)}


def desc_hash(desc: dict) -> str:
    h = hashlib.sha256()
    for k in ("cell_first", "parent", "area", "ri", "cm", "thr"):
        h.update(np.ascontiguousarray(desc[k]).tobytes())
    for m in desc["mechs"]:
        h.update(m["type"].encode())
        h.update(np.ascontiguousarray(m["node"]).tobytes())
        for k in sorted(m["params"]):
            h.update(np.ascontiguousarray(m["params"][k]).tobytes())
        h.update(repr(sorted(m["globals"].items())).encode())
    for k in ("src", "tgt_mech", "tgt_inst", "weight", "delay"):
        h.update(np.ascontiguousarray(desc["netcons"][k]).tobytes())
    h.update(np.ascontiguousarray(desc["stim"]["gid"]).tobytes())
    h.update(np.ascontiguousarray(desc["stim"]["t"]).tobytes())
    return h.hexdigest()


# ------------------------------------------------------------------------------------------
# tiny models for pins and edge cases
# ------------------------------------------------------------------------------------------

def single_compartment(mechs, diam=20.0, L=20.0, cm=1.0, v_init=-65.0, thr=-20.0, celsius=6.3):
    """One cylindrical compartment; `mechs` is a list of (type, params-dict, globals-dict)."""
    parent = np.array([-1], dtype=np.int64)
    area, ri = geometry(parent, np.array([L]), np.array([diam]), 100.0)
    ms = [_mech(t, [0], {k: [v] for k, v in p.items()}, g) for (t, p, g) in mechs]
    return {"cell_first": np.array([0, 1], np.int64), "parent": parent.astype(np.int32),
            "area": area, "ri": ri, "cm": _const(1, cm), "v_init": v_init, "celsius": celsius,
            "mechs": ms, "netcons": _netcons([], [], [], [], []),
            "thr": _const(1, thr), "stim": _no_stim()}


def cable(n, diam=1.0, L=200.0, Ra=100.0, cm=1.0, g_pas=0.001, e_pas=-65.0, v_init=-65.0):
    """Unbranched passive cable of n equal compartments (parent[i] = i-1)."""
    parent = np.arange(-1, n - 1, dtype=np.int64)
    area, ri = geometry(parent, _const(n, L / n), _const(n, diam), Ra)
    ms = []
    if g_pas is not None:
        ms.append(_mech("pas", np.arange(n), {"g": _const(n, g_pas), "e": _const(n, e_pas)}))
    return {"cell_first": np.array([0, n], np.int64), "parent": parent.astype(np.int32),
            "area": area, "ri": ri, "cm": _const(n, cm), "v_init": v_init, "celsius": 6.3,
            "mechs": ms, "netcons": _netcons([], [], [], [], []),
            "thr": _const(1, -20.0), "stim": _no_stim()}


def random_tree_parent(n: int, stream, max_children: int = 3) -> np.ndarray:
    """Random rooted tree with parent[i] < i."""
    parent = np.full(n, -1, dtype=np.int64)
    nchild = np.zeros(n, dtype=np.int64)
    draws = rng.bits(stream, 4 * n)
    j = 0
    for i in range(1, n):
        while True:
            p = int(draws[j % len(draws)] % np.uint64(i))
            j += 1
            if nchild[p] < max_children or j > 3 * n:
                break
        parent[i] = p
        nchild[p] += 1
    return parent


def random_tree_cells(n_cell, n_lo, n_hi, stream="rtree", mech="pas", identical=False,
                      with_ring=True, weight=0.05, delay=1.0, amp=0.5):
    """Cells with seeded random topology; optional ring of ExpSyn NetCons and an IClamp on cell 0.

    mech = "pas" (passive dendrites + HH soma) or "hh" (HH everywhere).
    """
    sizes = rng.randint((stream, "size"), n_cell, n_lo, n_hi + 1)
    if identical:
        sizes[:] = sizes[0]
    cell_first = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    N = int(cell_first[-1])
    parent = np.zeros(N, dtype=np.int64)
    area = np.zeros(N)
    ri = np.zeros(N)
    for c in range(n_cell):
        n = int(sizes[c])
        pl = random_tree_parent(n, (stream, "topo", 0 if identical else c))
        Lc = rng.uniform((stream, "L", c), n, 10.0, 30.0)
        dm = rng.uniform((stream, "d", c), n, 0.8, 2.0)
        Lc[0], dm[0] = 20.0, 20.0
        a_, r_ = geometry(pl, Lc, dm, 100.0)
        f = int(cell_first[c])
        parent[f:f + n] = np.where(pl < 0, -1, pl + f)
        area[f:f + n] = a_
        ri[f:f + n] = r_
    roots = cell_first[:-1]
    is_root = np.zeros(N, dtype=bool)
    is_root[roots] = True
    mechs = []
    if mech == "hh":
        hh_nodes = np.arange(N)
    else:
        hh_nodes = roots
    fac = rng.uniform((stream, "hhfac"), len(hh_nodes), 0.7, 1.0)
    mechs.append(_mech("hh", hh_nodes, {"gnabar": HH_SQUID["gnabar"] * fac,
                                         "gkbar": HH_SQUID["gkbar"] * fac,
                                         "gl": HH_SQUID["gl"] * fac,
                                         "el": _const(len(hh_nodes), HH_SQUID["el"])},
                       HH_GLOBALS))
    if mech != "hh":
        pn = np.nonzero(~is_root)[0]
        mechs.append(_mech("pas", pn, {"g": rng.uniform((stream, "gp"), len(pn), 5e-4, 2e-3),
                                        "e": _const(len(pn), -65.0)}))
    syn_t = len(mechs)
    mechs.append(_mech("expsyn", roots, {"tau": _const(n_cell, 2.0), "e": _const(n_cell, 0.0)}))
    mechs.append(_mech("iclamp", [roots[0]], {"del": [1.0], "dur": [1.0], "amp": [amp]}))
    if with_ring and n_cell > 1:
        src = np.arange(n_cell)
        nc = _netcons(src, np.full(n_cell, syn_t), (src + 1) % n_cell, _const(n_cell, weight),
                      _const(n_cell, delay))
    else:
        nc = _netcons([], [], [], [], [])
    return {"cell_first": cell_first, "parent": parent.astype(np.int32), "area": area, "ri": ri,
            "cm": _const(N, 1.0), "v_init": -65.0, "celsius": 6.3, "mechs": mechs, "netcons": nc,
            "thr": _const(n_cell, -20.0), "stim": _no_stim()}


# ------------------------------------------------------------------------------------------
# shared builder: many cells on branch templates
# ------------------------------------------------------------------------------------------

def _assemble_uniform(parent_local_by_cell, Lc, dm, Ra):
    """All cells have the same node count n.  parent_local_by_cell: [n_cell, n]."""
    n_cell, n = Lc.shape
    area = np.pi * dm * Lc
    rhalf = 1e-2 * Ra * (Lc / 2.0) / (np.pi * dm * dm / 4.0)
    p = np.where(parent_local_by_cell < 0, 0, parent_local_by_cell)
    ri = rhalf + np.take_along_axis(rhalf, p, axis=1)
    ri = np.where(parent_local_by_cell < 0, 1.0, ri)
    offs = (np.arange(n_cell, dtype=np.int64) * n)[:, None]
    parent = np.where(parent_local_by_cell < 0, -1, parent_local_by_cell + offs)
    cell_first = np.arange(n_cell + 1, dtype=np.int64) * n
    return cell_first, parent.reshape(-1).astype(np.int32), area.reshape(-1), ri.reshape(-1)


def _ring_netcons(n_cell, ring_size, syn_mech, weight, delay):
    gid = np.arange(n_cell, dtype=np.int64)
    ring = gid // ring_size
    nxt = ring * ring_size + (gid % ring_size + 1) % ring_size
    return _netcons(gid, np.full(n_cell, syn_mech), nxt, _const(n_cell, weight),
                    _const(n_cell, delay))


# ------------------------------------------------------------------------------------------
# config 1: ring of 8 cells, 61 compartments each
# ------------------------------------------------------------------------------------------

def config1(n_cell: int = 8, weight: float = 0.05, stim_cell: int = 0):
    bp = binary_branches(2)                       # 6 branches
    ncomp = np.full(len(bp), 10, dtype=np.int64)
    pl, branch_of, _, _ = expand_branches(bp, ncomp)
    n = len(pl)                                   # 61
    Lc = np.where(branch_of < 0, 20.0, 200.0 / 10.0)
    dm = np.where(branch_of < 0, 20.0, 1.0)
    cell_first, parent, area, ri = _assemble_uniform(
        np.tile(pl, (n_cell, 1)), np.tile(Lc, (n_cell, 1)), np.tile(dm, (n_cell, 1)), 100.0)
    N = n_cell * n
    roots = cell_first[:-1]
    dend = np.nonzero(np.tile(branch_of >= 0, n_cell))[0]
    mechs = [
        _mech("hh", roots, {k: _const(n_cell, v) for k, v in HH_SQUID.items()}, HH_GLOBALS),
        _mech("pas", dend, {"g": _const(len(dend), 0.001), "e": _const(len(dend), -65.0)}),
        _mech("expsyn", roots, {"tau": _const(n_cell, 2.0), "e": _const(n_cell, 0.0)}),
        _mech("iclamp", [roots[stim_cell]], {"del": [1.0], "dur": [1.0], "amp": [0.5]}),
    ]
    return {"cell_first": cell_first, "parent": parent, "area": area, "ri": ri,
            "cm": _const(N, 1.0), "v_init": -65.0, "celsius": 6.3, "mechs": mechs,
            "netcons": _ring_netcons(n_cell, n_cell, 2, weight, 1.0),
            "thr": _const(n_cell, -20.0), "stim": _no_stim()}


# ------------------------------------------------------------------------------------------
# config 2: 256 cells, HH everywhere, 4 independent rings of 64 (R14)
# ------------------------------------------------------------------------------------------

def config2(n_cell: int = 256, ring_size: int = 64, depth: int = 4, ncomp_branch: int = 20,
            weight: float = 0.02, rings=None):
    bp = binary_branches(depth)
    nb = len(bp)
    ncomp = np.full(nb, ncomp_branch, dtype=np.int64)
    pl, branch_of, _, _ = expand_branches(bp, ncomp)
    n = len(pl)
    # seeded branch-length variation of +-30 % around 200 um, per cell and branch
    Lb = 200.0 * rng.uniform(("c2", "L"), n_cell * nb, 0.7, 1.3).reshape(n_cell, nb)
    Lc = np.where(branch_of[None, :] < 0, 20.0, Lb[:, np.maximum(branch_of, 0)] / ncomp_branch)
    dm = np.tile(np.where(branch_of < 0, 20.0, 1.0), (n_cell, 1))
    cell_first, parent, area, ri = _assemble_uniform(np.tile(pl, (n_cell, 1)), Lc, dm, 100.0)
    N = n_cell * n
    roots = cell_first[:-1]
    fac = rng.uniform(("c2", "hhfac"), N, 0.5, 1.0)
    fac[roots] = 1.0
    mechs = [
        _mech("hh", np.arange(N), {"gnabar": HH_SQUID["gnabar"] * fac,
                                   "gkbar": HH_SQUID["gkbar"] * fac,
                                   "gl": HH_SQUID["gl"] * fac,
                                   "el": _const(N, HH_SQUID["el"])}, HH_GLOBALS),
        _mech("expsyn", roots, {"tau": _const(n_cell, 2.0), "e": _const(n_cell, 0.0)}),
    ]
    stim_cells = roots[::ring_size]
    ns = len(stim_cells)
    mechs.append(_mech("iclamp", stim_cells, {"del": _const(ns, 1.0), "dur": _const(ns, 1.0),
                                              "amp": _const(ns, 0.5)}))
    desc = {"cell_first": cell_first, "parent": parent, "area": area, "ri": ri,
            "cm": _const(N, 1.0), "v_init": -65.0, "celsius": 6.3, "mechs": mechs,
            "netcons": _ring_netcons(n_cell, ring_size, 1, weight, 1.0),
            "thr": _const(n_cell, -20.0), "stim": _no_stim()}
    if rings is not None:
        gids = np.concatenate([np.arange(r * ring_size, (r + 1) * ring_size) for r in rings])
        desc = extract_cells(desc, gids)
    return desc


# ------------------------------------------------------------------------------------------
# config 4: large ring-of-branching-cells workload (Table 1 "Ring": 32,768 x 291, 33,280 NetCons)
# ------------------------------------------------------------------------------------------

def _composition(total: int, parts: int, lo: int, hi: int, stream) -> np.ndarray:
    """Seeded composition of `total` into `parts` integers in [lo, hi]."""
    x = np.full(parts, lo, dtype=np.int64)
    rest = total - lo * parts
    assert 0 <= rest <= (hi - lo) * parts
    draws = rng.bits(stream, 64 * parts)
    j = 0
    while rest > 0:
        q = int(draws[j % len(draws)] % np.uint64(parts))
        j += 1
        if x[q] < hi:
            x[q] += 1
            rest -= 1
    return x


def config4(n_cell: int = 32768, n_types: int = 1024, ring_size: int = 64, depth: int = 5,
            n_dend_comp: int = 290, weight: float = 0.02, shuffle: bool = True, cells=None):
    """R15: n_types seeded branch-length compositions, cells of a type share topology only
    (per-cell geometry jitter), cell order shuffled; 512 rings x 64 + one scripted source/ring.

    `cells`: optional list of ring indices to extract (sampled parity at full size)."""
    bp = binary_branches(depth)                   # 62 branches
    nb = len(bp)
    n = n_dend_comp + 1
    # axon-like path: branch chain 0 -> first child -> ... to a leaf
    children = [[] for _ in range(nb)]
    for j, p in enumerate(bp):
        if p >= 0:
            children[p].append(j)
    pl_t = np.zeros((n_types, n), dtype=np.int64)
    hh_t = np.zeros((n_types, n), dtype=bool)
    for t in range(n_types):
        ncomp = _composition(n_dend_comp, nb, 1, 12, ("c4", "comp", t))
        pl, branch_of, _, _ = expand_branches(bp, ncomp)
        pl_t[t] = pl
        # seeded root-to-leaf path
        path = []
        pick = rng.bits(("c4", "path", t), depth)
        cur = int(pick[0] % np.uint64(2))         # one of the two primary branches
        path.append(cur)
        for lv in range(1, depth):
            cur = children[cur][int(pick[lv] % np.uint64(2))]
            path.append(cur)
        hh_t[t] = (branch_of < 0) | np.isin(branch_of, path)
    if shuffle:
        type_of = (rng.permutation(("c4", "shuffle"), n_cell) % n_types).astype(np.int64)
    else:
        type_of = (np.arange(n_cell) % n_types).astype(np.int64)
    n_ring = n_cell // ring_size
    if cells is not None:
        gid_sel = np.concatenate([np.arange(r * ring_size, (r + 1) * ring_size) for r in cells])
    else:
        gid_sel = np.arange(n_cell)
    nc_sel = len(gid_sel)
    ty = type_of[gid_sel]
    pl_c = pl_t[ty]
    hh_c = hh_t[ty]
    # per-cell geometry jitter: compartment length 20 um +-10 %, dendrite diameter 1 um +-10 %
    jl = np.empty(nc_sel)
    jd = np.empty(nc_sel)
    ul = rng.uniform(("c4", "jl"), n_cell, 0.9, 1.1)
    ud = rng.uniform(("c4", "jd"), n_cell, 0.9, 1.1)
    jl[:] = ul[gid_sel]
    jd[:] = ud[gid_sel]
    Lc = np.empty((nc_sel, n))
    dm = np.empty((nc_sel, n))
    Lc[:, :] = 20.0 * jl[:, None]
    dm[:, :] = 1.0 * jd[:, None]
    Lc[:, 0] = 20.0
    dm[:, 0] = 20.0
    cell_first, parent, area, ri = _assemble_uniform(pl_c, Lc, dm, 100.0)
    N = nc_sel * n
    roots = cell_first[:-1]
    hh_nodes = np.nonzero(hh_c.reshape(-1))[0]
    pas_nodes = np.nonzero(~hh_c.reshape(-1))[0]
    mechs = [
        _mech("hh", hh_nodes, {k: _const(len(hh_nodes), v) for k, v in HH_SQUID.items()},
              HH_GLOBALS),
        _mech("pas", pas_nodes, {"g": _const(len(pas_nodes), 0.001),
                                 "e": _const(len(pas_nodes), -65.0)}),
        _mech("expsyn", roots, {"tau": _const(nc_sel, 2.0), "e": _const(nc_sel, 0.0)}),
    ]
    nc = _ring_netcons(nc_sel, ring_size, 2, weight, 1.0)
    nr = nc_sel // ring_size
    # one scripted source per ring (gids n_cell .. n_cell+n_ring-1), spiking once at t = 0
    s_src = nc_sel + np.arange(nr)
    nc = {k: np.concatenate([nc[k], v]) for k, v in
          _netcons(s_src, np.full(nr, 2), np.arange(nr) * ring_size, _const(nr, 2.5 * weight),
                   _const(nr, 1.0)).items()}
    desc = {"cell_first": cell_first, "parent": parent, "area": area, "ri": ri,
            "cm": _const(N, 1.0), "v_init": -65.0, "celsius": 6.3, "mechs": mechs, "netcons": nc,
            "thr": _const(nc_sel, -20.0),
            "stim": {"gid": s_src.astype(np.int32), "t": np.zeros(nr)}}
    desc["_type_of"] = ty
    desc["_n_ring_total"] = n_ring
    return desc


# ------------------------------------------------------------------------------------------
# sub-model extraction (sampled parity at full size)
# ------------------------------------------------------------------------------------------

def extract_cells(desc: dict, gids) -> dict:
    """Sub-model of the given cells (kept in the given order).  Every NetCon whose target is kept
    must have its source kept too (closed set), else ValueError.  Scripted sources are kept."""
    gids = np.asarray(gids, dtype=np.int64)
    n_cell = len(desc["cell_first"]) - 1
    cf = desc["cell_first"]
    sizes = (cf[1:] - cf[:-1])[gids]
    new_first = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    N = int(new_first[-1])
    old_nodes = np.concatenate([np.arange(cf[g], cf[g + 1]) for g in gids]) if len(gids) else \
        np.zeros(0, np.int64)
    node_map = np.full(int(cf[-1]), -1, dtype=np.int64)
    node_map[old_nodes] = np.arange(N)
    gid_map = np.full(n_cell, -1, dtype=np.int64)
    gid_map[gids] = np.arange(len(gids))
    parent_old = desc["parent"][old_nodes].astype(np.int64)
    parent = np.where(parent_old < 0, -1, node_map[np.maximum(parent_old, 0)])
    mechs = []
    inst_maps = []
    for m in desc["mechs"]:
        keep = node_map[m["node"]] >= 0
        imap = np.full(len(m["node"]), -1, dtype=np.int64)
        imap[keep] = np.arange(int(keep.sum()))
        inst_maps.append(imap)
        mechs.append(_mech(m["type"], node_map[m["node"]][keep],
                           {k: v[keep] for k, v in m["params"].items()}, m["globals"]))
    nc = desc["netcons"]
    src = nc["src"].astype(np.int64)
    # (vectorised: one flat instance map over all tables)
    toff = np.concatenate([[0], np.cumsum([len(x) for x in inst_maps])]).astype(np.int64)
    flat = np.concatenate(inst_maps) if inst_maps else np.zeros(0, np.int64)
    tm_all = nc["tgt_mech"].astype(np.int64)
    new_inst = flat[toff[tm_all] + nc["tgt_inst"].astype(np.int64)] if len(src) else np.zeros(0, np.int64)
    tgt_keep = new_inst >= 0
    is_stim = src >= n_cell
    src_cell_new = np.where(is_stim, -1, gid_map[np.minimum(src, n_cell - 1)]) if n_cell else \
        np.full(len(src), -1, np.int64)
    if np.any(tgt_keep & ~is_stim & (src_cell_new < 0)):
        raise ValueError("extract_cells: a kept target has a dropped source (set not closed)")
    # renumber scripted sources densely after the kept cells
    stim_old = np.unique(src[tgt_keep & is_stim])
    stim_map = {int(g): len(gids) + j for j, g in enumerate(stim_old)}
    new_src = src_cell_new[tgt_keep].copy()
    ks = is_stim[tgt_keep]
    if ks.any():
        new_src[ks] = len(gids) + np.searchsorted(stim_old, src[tgt_keep][ks])
    tm = nc["tgt_mech"][tgt_keep]
    ti = new_inst[tgt_keep]
    new_nc = _netcons(new_src, tm, ti, nc["weight"][tgt_keep], nc["delay"][tgt_keep])
    sk = np.array([int(g) in stim_map for g in desc["stim"]["gid"]], dtype=bool) \
        if len(desc["stim"]["gid"]) else np.zeros(0, bool)
    stim = {"gid": np.array([stim_map[int(g)] for g in desc["stim"]["gid"][sk]], dtype=np.int32),
            "t": desc["stim"]["t"][sk]}
    return {"cell_first": new_first, "parent": parent.astype(np.int32),
            "area": desc["area"][old_nodes], "ri": desc["ri"][old_nodes],
            "cm": desc["cm"][old_nodes], "v_init": desc["v_init"], "celsius": desc["celsius"],
            "mechs": mechs, "netcons": new_nc, "thr": desc["thr"][gids], "stim": stim}


def concat_models(descs) -> dict:
    """Several descriptions side by side as one model: cells, nodes and instances renumbered, no
    connection between the parts.  The parts must have the same list of mechanism tables (type and
    globals) and no scripted sources."""
    d0 = descs[0]
    node_off = np.concatenate([[0], np.cumsum([int(d["cell_first"][-1]) for d in descs])])
    cell_off = np.concatenate([[0], np.cumsum([len(d["cell_first"]) - 1 for d in descs])])
    for d in descs:
        assert len(d["stim"]["gid"]) == 0 and len(d["mechs"]) == len(d0["mechs"])
        assert d["v_init"] == d0["v_init"] and d["celsius"] == d0["celsius"]
    mechs = []
    inst_off = []
    for t, m0 in enumerate(d0["mechs"]):
        parts = [d["mechs"][t] for d in descs]
        assert all(p["type"] == m0["type"] and p["globals"] == m0["globals"] for p in parts)
        inst_off.append(np.concatenate([[0], np.cumsum([len(p["node"]) for p in parts])]))
        mechs.append(_mech(m0["type"],
                           np.concatenate([p["node"].astype(np.int64) + node_off[j]
                                           for j, p in enumerate(parts)]),
                           {k: np.concatenate([p["params"][k] for p in parts])
                            for k in m0["params"]}, m0["globals"]))
    cat = lambda key, sub=None: np.concatenate(  # noqa: E731
        [(d[key] if sub is None else d[key][sub]) for d in descs])
    nc = _netcons(
        np.concatenate([d["netcons"]["src"].astype(np.int64) + cell_off[j]
                        for j, d in enumerate(descs)]),
        cat("netcons", "tgt_mech"),
        np.concatenate([d["netcons"]["tgt_inst"].astype(np.int64) +
                        np.array([inst_off[t][j] for t in d["netcons"]["tgt_mech"]], np.int64)
                        for j, d in enumerate(descs)]),
        cat("netcons", "weight"), cat("netcons", "delay"))
    par = np.concatenate([np.where(d["parent"] < 0, -1, d["parent"].astype(np.int64) + node_off[j])
                          for j, d in enumerate(descs)])
    cf = np.concatenate([[0]] + [d["cell_first"][1:] + node_off[j] for j, d in enumerate(descs)])
    return {"cell_first": cf.astype(np.int64), "parent": par.astype(np.int32),
            "area": cat("area"), "ri": cat("ri"), "cm": cat("cm"), "v_init": d0["v_init"],
            "celsius": d0["celsius"], "mechs": mechs, "netcons": nc, "thr": cat("thr"),
            "stim": _no_stim()}


def renumber_nodes(desc: dict, stream="renum") -> dict:
    """Seeded random parent-before-child renumbering inside every cell (roots stay first)."""
    cf = desc["cell_first"]
    N = int(cf[-1])
    parent = desc["parent"].astype(np.int64)
    new_of_old = np.zeros(N, dtype=np.int64)
    for c in range(len(cf) - 1):
        f, l = int(cf[c]), int(cf[c + 1])
        n = l - f
        key = rng.uniform((stream, c), n)
        # random topological order: repeatedly emit the ready node with the smallest key
        children = [[] for _ in range(n)]
        for i in range(f + 1, l):
            children[parent[i] - f].append(i - f)
        import heapq
        heap = [(0.0, 0)]
        order = []
        while heap:
            _, i = heapq.heappop(heap)
            order.append(i)
            for ch in children[i]:
                heapq.heappush(heap, (key[ch], ch))
        new_of_old[f + np.array(order)] = f + np.arange(n)
    old_of_new = np.argsort(new_of_old)
    out = dict(desc)
    out["parent"] = np.where(parent[old_of_new] < 0, -1,
                             new_of_old[np.maximum(parent[old_of_new], 0)]).astype(np.int32)
    for k in ("area", "ri", "cm"):
        out[k] = desc[k][old_of_new]
    out["mechs"] = [_mech(m["type"], new_of_old[m["node"]], m["params"], m["globals"])
                    for m in desc["mechs"]]
    out["_new_of_old"] = new_of_old
    return out


def shuffle_instances(desc: dict, stream="shuf") -> dict:
    """The same model with the instances of every mechanism table in a seeded random order
    (NetCon targets follow); `_new_of_old_inst[t]` maps an old instance index to its new one."""
    out = dict(desc)
    mechs, maps = [], []
    for t, m in enumerate(desc["mechs"]):
        n = len(m["node"])
        old_of_new = rng.permutation((stream, t), n).astype(np.int64) if n else np.zeros(0, np.int64)
        new_of_old = np.empty(n, dtype=np.int64)
        new_of_old[old_of_new] = np.arange(n)
        mechs.append(_mech(m["type"], m["node"][old_of_new],
                           {k: v[old_of_new] for k, v in m["params"].items()}, m["globals"]))
        maps.append(new_of_old)
    out["mechs"] = mechs
    nc = dict(desc["netcons"])
    if len(nc["tgt_inst"]):
        nc["tgt_inst"] = np.array([maps[tm][ti] for tm, ti in zip(nc["tgt_mech"], nc["tgt_inst"])],
                                  dtype=np.int64)
    out["netcons"] = nc
    out["_new_of_old_inst"] = maps
    return out
