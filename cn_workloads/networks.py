"""Seeded synthetic networks shaped like BASELINE.json's configs 3 and 5 (inputs only).

Like configs.py this module holds topology, geometry -> (area, axial resistance), mechanism
placement / parameters and NetCons, and none of the method's arithmetic.  The channel constants
are the SYNTHETIC table of SURVEY.md 8(c) (shaped like the paper's model classes, PAPER.md L39 /
L222; the real channel files are third-party and not in this container).
"""
from __future__ import annotations

import numpy as np

from . import rng
from .configs import (HH_GLOBALS, HH_SQUID, _composition, _const, _mech, _netcons,
                      binary_branches, expand_branches)

# p, q, E, m-gate (v_half, k, tau0, tau1, v_tau, sigma), h-gate (same)
HHFORM_TABLE = {
    "NaT": (3, 1, 50.0, (-38, 6, 0.02, 0.4, -38, 12), (-66, -6, 0.3, 10, -60, 12)),
    "NaP": (3, 1, 50.0, (-52, 5, 0.5, 5, -52, 15), (-49, -10, 100, 4000, -49, 15)),
    "Kv31": (1, 0, -85.0, (18.7, 9.7, 0.2, 8, -46, 44), (0, 1, 1, 0, 0, 1)),
    "Kv1": (2, 1, -85.0, (-11, 12, 1, 10, -11, 30), (-64, -11, 300, 1000, -64, 25)),
    "Ih": (1, 0, -45.0, (-90, -9, 20, 1000, -90, 20), (0, 1, 1, 0, 0, 1)),
    "CaHVA": (2, 1, 132.4579, (-27, 5, 0.5, 3, -27, 15), (-40, -8, 200, 500, -40, 20)),
    "CaLVA": (2, 1, 132.4579, (-40, 6, 5, 25, -40, 15), (-90, -6.4, 20, 70, -75, 15)),
}
SK_GLOBALS = dict(E=-85.0, Kd=4.3e-4, n=4.8, tau_z=1.0)
CADYN_GLOBALS = dict(gamma=0.05, depth=0.1, tau_d=80.0, cai_min=1e-4)
AMPANMDA_GLOBALS = dict(tau_r_A=0.2, tau_d_A=1.7, tau_r_N=0.29, tau_d_N=43.0, r_nmda=0.71,
                        mg=1.0, e=0.0)


def hhform_globals(name: str) -> dict:
    p, q, E, mg, hg = HHFORM_TABLE[name]
    G = {"p": p, "q": q, "E": E, "to_ica": 1.0 if name.startswith("Ca") else 0.0}
    for pre, gate in (("m", mg), ("h", hg)):
        for key, val in zip(("vh", "k", "t0", "t1", "vt", "s"), gate):
            G[f"{pre}_{key}"] = float(val)
    return G


# ------------------------------------------------------------------------------------------
# cells of several morphology types, variable node count
# ------------------------------------------------------------------------------------------

def _branch_levels(bp: np.ndarray) -> np.ndarray:
    lv = np.zeros(len(bp), dtype=np.int64)
    for j, p in enumerate(bp):
        lv[j] = 0 if p < 0 else lv[p] + 1
    return lv


def _morph_types(tag, n_types, n_nodes, depths, comp_hi):
    """Per type: local parent[], level of every node (-1 soma), a seeded root-to-leaf path."""
    types = []
    for t in range(n_types):
        bp = binary_branches(int(depths[t]))
        nb = len(bp)
        ncomp = _composition(int(n_nodes[t]) - 1, nb, 1, comp_hi, (tag, "comp", t))
        pl, branch_of, _, _ = expand_branches(bp, ncomp)
        lv = _branch_levels(bp)
        level = np.where(branch_of < 0, -1, lv[np.maximum(branch_of, 0)])
        children = [[] for _ in range(nb)]
        for j, p in enumerate(bp):
            if p >= 0:
                children[p].append(j)
        pick = rng.bits((tag, "path", t), int(depths[t]))
        cur = int(pick[0] % np.uint64(2))
        path = [cur]
        for d in range(1, int(depths[t])):
            cur = children[cur][int(pick[d] % np.uint64(2))]
            path.append(cur)
        on_path = (branch_of < 0) | np.isin(branch_of, path)
        types.append({"parent": pl, "level": level, "path": on_path, "n": len(pl)})
    return types


def _assemble_typed(tag, types, type_of, diam0=2.0):
    """Cells in gid order, cell g of type type_of[g].  Compartment length 20 um and dendrite
    diameter diam0 / (1 + level / 2) um, each with a seeded +-10 % factor per cell; soma 20 x 20 um;
    Ra = 100 Ohm cm.  Returns cell_first, parent, area, ri and a scatter index per type."""
    n_cell = len(type_of)
    n_of = np.array([types[t]["n"] for t in type_of], dtype=np.int64)
    cell_first = np.zeros(n_cell + 1, dtype=np.int64)
    np.cumsum(n_of, out=cell_first[1:])
    N = int(cell_first[-1])
    parent = np.empty(N, dtype=np.int64)
    area = np.empty(N)
    ri = np.empty(N)
    jl = rng.uniform((tag, "jl"), n_cell, 0.9, 1.1)
    jd = rng.uniform((tag, "jd"), n_cell, 0.9, 1.1)
    idx_of_type = []
    for t, T in enumerate(types):
        gids = np.nonzero(type_of == t)[0]
        n = T["n"]
        idx = cell_first[gids][:, None] + np.arange(n)[None, :]      # [cells of t, n] global nodes
        idx_of_type.append((gids, idx))
        if len(gids) == 0:
            continue
        lvl = T["level"]
        Lc = np.where(lvl[None, :] < 0, 20.0, 20.0 * jl[gids][:, None])
        dm = np.where(lvl[None, :] < 0, 20.0,
                      diam0 / (1.0 + 0.5 * np.maximum(lvl, 0))[None, :] * jd[gids][:, None])
        a = np.pi * dm * Lc
        rhalf = 1e-2 * 100.0 * (Lc / 2.0) / (np.pi * dm * dm / 4.0)
        pl = T["parent"]
        r = rhalf + rhalf[:, np.maximum(pl, 0)]
        r[:, 0] = 1.0
        area[idx] = a
        ri[idx] = r
        parent[idx] = np.where(pl[None, :] < 0, -1, cell_first[gids][:, None] + np.maximum(pl, 0)[None, :])
    return cell_first, parent.astype(np.int32), area, ri, idx_of_type


def _nodes_where(types, idx_of_type, mask_fn):
    """Global nodes (ascending) of all cells whose local node satisfies mask_fn(type dict)."""
    out = []
    for T, (gids, idx) in zip(types, idx_of_type):
        if len(gids):
            out.append(idx[:, np.nonzero(mask_fn(T))[0]].reshape(-1))
    return np.sort(np.concatenate(out)) if out else np.zeros(0, np.int64)


def _cell_of_nodes(cell_first, nodes):
    return np.searchsorted(cell_first, nodes, side="right") - 1


def _poisson_pulses(tag, cells, rate_hz, t_end, dt, amp, dur, roots):
    """IClamp pulses: seeded Poisson onsets (exponential gaps) quantised to steps of dt."""
    node, dels = [], []
    mean_gap = 1000.0 / rate_hz
    for c in cells:
        u = rng.uniform((tag, "gap", int(c)), 64)
        t = np.cumsum(-mean_gap * np.log(1.0 - u))
        t = t[t < t_end]
        k = np.maximum(np.round(t / dt), 1.0)
        node.extend([roots[c]] * len(k))
        dels.extend(list(k * dt))
    n = len(node)
    return _mech("iclamp", node, {"del": np.array(dels), "dur": _const(n, dur), "amp": _const(n, amp)})


def _type_counts(n_cell, n_nodes, total):
    """Cells per type (sum n_cell) such that sum(count * n_nodes) == total (if not None)."""
    nt = len(n_nodes)
    cnt = np.full(nt, n_cell // nt, dtype=np.int64)
    cnt[: n_cell % nt] += 1
    if total is None:
        return cnt
    order = np.argsort(n_nodes)
    lo, hi = int(order[0]), int(order[-1])
    d = int(total - np.sum(cnt * n_nodes))
    big = int(n_nodes[hi] - n_nodes[lo])
    while abs(d) >= big:                      # coarse: move cells between the extreme types
        src, dst = (lo, hi) if d > 0 else (hi, lo)
        if cnt[src] <= 1:
            raise ValueError("cannot reach the requested compartment total")
        cnt[src] -= 1
        cnt[dst] += 1
        d -= big if d > 0 else -big
    # fine: types 0 and 1 differ by exactly one node
    assert n_nodes[1] - n_nodes[0] == 1
    while d != 0:
        src, dst = (0, 1) if d > 0 else (1, 0)
        cnt[src] -= 1
        cnt[dst] += 1
        d -= 1 if d > 0 else -1
    assert np.all(cnt > 0) and np.sum(cnt * n_nodes) == total
    return cnt


def _random_synapses(tag, types, idx_of_type, n_cell, syn_per_cell, by_area=None):
    """syn_per_cell synapse nodes per cell, drawn over the cell's dendritic nodes (uniformly, or
    proportionally to `by_area`); returned grouped by cell in gid order."""
    node = np.empty((n_cell, syn_per_cell), dtype=np.int64)
    for t, (T, (gids, idx)) in enumerate(zip(types, idx_of_type)):
        if len(gids) == 0:
            continue
        dend = np.nonzero(T["level"] >= 0)[0]
        u = rng.uniform((tag, "synnode", t), len(gids) * syn_per_cell).reshape(len(gids), -1)
        if by_area is None:
            k = np.minimum((u * len(dend)).astype(np.int64), len(dend) - 1)
        else:
            a = by_area[idx[:, dend]]
            cdf = np.cumsum(a, axis=1)
            cdf /= cdf[:, -1:]
            k = np.empty_like(u, dtype=np.int64)
            for r in range(len(gids)):
                k[r] = np.minimum(np.searchsorted(cdf[r], u[r]), len(dend) - 1)
        node[gids] = np.take_along_axis(idx[:, dend], k, axis=1)
    return node.reshape(-1)


# ------------------------------------------------------------------------------------------
# config 3: thalamocortical-shaped network (Table 1 "Traub": 3,560 cells, 14 types, 465,740
# compartments -- R20; ~1.1 M Exp2Syn; Ca source added -- R17; Poisson IClamp drive -- R18)
# ------------------------------------------------------------------------------------------

def config3(n_cell: int = 3560, n_types: int = 14, n_comp_total=465740, syn_per_cell: int = 309,
            w_scale: float = 0.1, drive_amp: float = 0.8, t_end: float = 100.0,
            dt: float = 0.025):
    """w_scale: factor on the lognormal(-4, 0.5) uS weights, tuned once in the oracle (0.1: every
    cell fires 1-2 times in 100 ms, mean rate in 1-20 Hz; 1.0 gives population bursts at 30 Hz)
    and frozen.  Weights scale with 309 / syn_per_cell so that scaled-down copies keep the drive."""
    tag = "c3"
    base = rng.randint((tag, "n"), n_types, 70, 200)
    base[1] = base[0] + 1
    depths = np.where(base < 100, 3, 4)
    types = _morph_types(tag, n_types, base, depths, 12)
    n_nodes = np.array([T["n"] for T in types], dtype=np.int64)
    cnt = _type_counts(n_cell, n_nodes, n_comp_total if n_cell == 3560 else None)
    type_of = np.repeat(np.arange(n_types), cnt)[rng.permutation((tag, "shuffle"), n_cell)]
    cell_first, parent, area, ri, iot = _assemble_typed(tag, types, type_of)
    N = int(cell_first[-1])
    roots = cell_first[:-1]
    # active zone: soma + primary branches (HH-like Na/K, Ca_HVA, SK, cai); pas everywhere
    act = _nodes_where(types, iot, lambda T: T["level"] <= 0)
    na = len(act)
    dens = rng.uniform((tag, "dens"), n_types, 0.8, 1.2)[type_of[_cell_of_nodes(cell_first, act)]]
    allnodes = np.arange(N)
    mechs = [
        _mech("hh", act, {"gnabar": HH_SQUID["gnabar"] * dens, "gkbar": HH_SQUID["gkbar"] * dens,
                          "gl": _const(na, HH_SQUID["gl"]), "el": _const(na, HH_SQUID["el"])},
              HH_GLOBALS),
        _mech("hhform", act, {"gbar": 2e-4 * dens}, hhform_globals("CaHVA")),
        _mech("sk", act, {"gbar": 2e-3 * dens}, SK_GLOBALS),
        _mech("cadyn", act, {}, CADYN_GLOBALS),
        _mech("pas", allnodes, {"g": _const(N, 1e-4), "e": _const(N, -65.0)}),
    ]
    ns = n_cell * syn_per_cell
    syn_node = _random_synapses(tag, types, iot, n_cell, syn_per_cell)
    mechs.append(_mech("exp2syn", syn_node, {"tau1": _const(ns, 0.5), "tau2": _const(ns, 5.0),
                                             "e": _const(ns, 0.0)}))
    driven = np.sort(rng.permutation((tag, "driven"), n_cell)[: max(1, n_cell // 10)])
    mechs.append(_poisson_pulses(tag, driven, 40.0, t_end, dt, drive_amp, 2.0, roots))
    src = rng.randint((tag, "pre"), ns, 0, n_cell)
    delay = dt * rng.randint((tag, "delay"), ns, int(round(1.0 / dt)), int(round(5.0 / dt)) + 1)
    weight = w_scale * (309.0 / syn_per_cell) * np.exp(-4.0 + 0.5 * rng.normal((tag, "w"), ns))
    nc = _netcons(src, np.full(ns, 5), np.arange(ns), weight, delay)
    return {"cell_first": cell_first, "parent": parent, "area": area, "ri": ri,
            "cm": _const(N, 1.0), "v_init": -65.0, "celsius": 6.3, "mechs": mechs, "netcons": nc,
            "thr": _const(n_cell, -20.0),
            "stim": {"gid": np.zeros(0, np.int32), "t": np.zeros(0)},
            "_type_of": type_of}


# ------------------------------------------------------------------------------------------
# config 5: cortex-shaped slice (Table 1 "Cortex": 20,000 cells x ~454 compartments, 55 types,
# 10 channel types per cell, ~4,000 AMPA+NMDA synapses per cell -- R19)
# ------------------------------------------------------------------------------------------

def config5(scale: float = 1.0, n_types: int = 55, syn_per_cell=None, w_scale: float = 1.0,
            drive_amp: float = 2.0, dt: float = 0.025, n_cell=None, block=None):
    """scale = 1: 20,000 cells, 4,000 synapses per cell (80 M).  Smaller scales shrink the cell
    count and (unless given) the synapses per cell proportionally; cells keep their full size.
    Weights are lognormal(-4, 0.5) uS x w_scale x 10 / syn_per_cell (tuned once in the oracle on a
    100-cell copy so that about a quarter of the cells fire within the 20 ms, then frozen; the
    1 / syn_per_cell factor keeps the summed drive of a cell independent of the scale).  The config
    names no stimulus: 10 % of the cells get one 2 ms IClamp pulse of drive_amp nA with a seeded
    onset in [0.5, 5) ms (reading R24).
    block: if given, the presynaptic cell of every synapse is drawn among the `block` cells of the
    target's own block (gids [j*block, (j+1)*block)): the network falls into closed sub-networks of
    full-size cells with the full number of synapses per cell, each of which the oracle can
    integrate on its own (extract_cells) -- sampled parity at the stated per-cell size."""
    tag = "c5"
    if n_cell is None:
        n_cell = max(n_types, int(round(20000 * scale)))
    if syn_per_cell is None:
        syn_per_cell = max(8, int(round(4000 * scale)))
    base = rng.randint((tag, "n"), n_types, 330, 580)
    depths = np.where(base < 420, 5, 6)
    types = _morph_types(tag, n_types, base, depths, 12)
    cnt = _type_counts(n_cell, np.array([T["n"] for T in types]), None)
    type_of = np.repeat(np.arange(n_types), cnt)[rng.permutation((tag, "shuffle"), n_cell)]
    cell_first, parent, area, ri, iot = _assemble_typed(tag, types, type_of, diam0=3.0)
    N = int(cell_first[-1])
    roots = cell_first[:-1]
    axo = _nodes_where(types, iot, lambda T: T["path"])                 # soma + axon-like path
    prox = _nodes_where(types, iot, lambda T: T["level"] <= 1)          # soma + two branch levels
    dend = _nodes_where(types, iot, lambda T: T["level"] >= 0)
    tdens = rng.uniform((tag, "dens"), n_types, 0.8, 1.2)

    def dens(nodes):
        return tdens[type_of[_cell_of_nodes(cell_first, nodes)]]

    mechs = [
        _mech("hhform", axo, {"gbar": 0.12 * dens(axo)}, hhform_globals("NaT")),
        _mech("hhform", axo, {"gbar": 2e-4 * dens(axo)}, hhform_globals("NaP")),
        _mech("hhform", axo, {"gbar": 0.05 * dens(axo)}, hhform_globals("Kv31")),
        _mech("hhform", axo, {"gbar": 2e-3 * dens(axo)}, hhform_globals("Kv1")),
        _mech("hhform", dend, {"gbar": 5e-5 * dens(dend)}, hhform_globals("Ih")),
        _mech("hhform", prox, {"gbar": 2e-4 * dens(prox)}, hhform_globals("CaHVA")),
        _mech("hhform", prox, {"gbar": 5e-4 * dens(prox)}, hhform_globals("CaLVA")),
        _mech("sk", prox, {"gbar": 2e-3 * dens(prox)}, SK_GLOBALS),
        _mech("cadyn", prox, {}, CADYN_GLOBALS),
        _mech("pas", np.arange(N), {"g": _const(N, 3e-5), "e": _const(N, -75.0)}),
    ]
    ns = n_cell * syn_per_cell
    syn_node = _random_synapses(tag, types, iot, n_cell, syn_per_cell, by_area=area)
    mechs.append(_mech("ampanmda", syn_node, {}, AMPANMDA_GLOBALS))
    driven = np.sort(rng.permutation((tag, "driven"), n_cell)[: max(1, n_cell // 10)])
    nd = len(driven)
    onset = dt * rng.randint((tag, "onset"), nd, int(round(0.5 / dt)), int(round(5.0 / dt)))
    mechs.append(_mech("iclamp", roots[driven], {"del": onset, "dur": _const(nd, 2.0),
                                                  "amp": _const(nd, drive_amp)}))
    if block is None:
        src = rng.randint((tag, "pre"), ns, 0, n_cell)
    else:
        tgt_cell = np.arange(ns, dtype=np.int64) // syn_per_cell
        b0 = (tgt_cell // block) * block
        bsz = np.minimum(block, n_cell - b0)
        src = b0 + (rng.bits((tag, "pre"), ns) % bsz.astype(np.uint64)).astype(np.int64)
    delay = dt * rng.randint((tag, "delay"), ns, int(round(0.1 / dt)), int(round(10.0 / dt)) + 1)
    weight = w_scale * (10.0 / syn_per_cell) * np.exp(-4.0 + 0.5 * rng.normal((tag, "w"), ns))
    nc = _netcons(src, np.full(ns, 10), np.arange(ns), weight, delay)
    return {"cell_first": cell_first, "parent": parent, "area": area, "ri": ri,
            "cm": _const(N, 1.0), "v_init": -75.0, "celsius": 6.3, "mechs": mechs, "netcons": nc,
            "thr": _const(n_cell, -20.0),
            "stim": {"gid": np.zeros(0, np.int32), "t": np.zeros(0)},
            "_type_of": type_of}


# ------------------------------------------------------------------------------------------
# node-ordering study (Fig. 5F): multiple-ring model, every cell 83 nodes,
# 40 dendrites with a random branching pattern per type, 1..32 identical cells per type
# ------------------------------------------------------------------------------------------

def fig5f(n_cell: int = 131072, per_type: int = 32, ring_size: int = 64, weight: float = 0.02):
    """Seeded stand-in for the paper's node-ordering workload (its model files are not here):
    soma + 40 dendrites (82 compartments, 1..4 per dendrite), each dendrite attached to the soma or
    to the last compartment of a random earlier dendrite; HH soma, passive dendrites, ExpSyn ring
    NetCons with 1 ms delay, one scripted source per ring.  Cell g has type g // per_type."""
    from .configs import _assemble_uniform, _ring_netcons
    tag = "f5"
    n_types = n_cell // per_type
    assert n_types * per_type == n_cell and n_cell % ring_size == 0
    n = 83
    pl_t = np.empty((n_types, n), dtype=np.int64)
    draws = rng.bits((tag, "attach"), n_types * 40).reshape(n_types, 40)
    for t in range(n_types):
        ncomp = _composition(82, 40, 1, 4, (tag, "comp", t))
        bp = np.full(40, -1, dtype=np.int64)
        for j in range(1, 40):
            k = int(draws[t, j] % np.uint64(j + 1))      # 0 = soma, else dendrite k - 1
            bp[j] = k - 1
        pl_t[t], _, _, _ = expand_branches(bp, ncomp)
    type_of = np.arange(n_cell) // per_type
    pl_c = pl_t[type_of]
    jl = rng.uniform((tag, "jl"), n_cell, 0.9, 1.1)
    Lc = np.empty((n_cell, n))
    dm = np.empty((n_cell, n))
    Lc[:, :] = 20.0 * jl[:, None]
    dm[:, :] = 1.0
    Lc[:, 0] = 20.0
    dm[:, 0] = 20.0
    cell_first, parent, area, ri = _assemble_uniform(pl_c, Lc, dm, 100.0)
    N = n_cell * n
    roots = cell_first[:-1]
    dend = np.setdiff1d(np.arange(N), roots, assume_unique=True)
    mechs = [
        _mech("hh", roots, {k: _const(n_cell, v) for k, v in HH_SQUID.items()}, HH_GLOBALS),
        _mech("pas", dend, {"g": _const(len(dend), 0.001), "e": _const(len(dend), -65.0)}),
        _mech("expsyn", roots, {"tau": _const(n_cell, 2.0), "e": _const(n_cell, 0.0)}),
    ]
    nc = _ring_netcons(n_cell, ring_size, 2, weight, 1.0)
    nr = n_cell // ring_size
    s_src = n_cell + np.arange(nr)
    nc = {k: np.concatenate([nc[k], v]) for k, v in
          _netcons(s_src, np.full(nr, 2), np.arange(nr) * ring_size, _const(nr, 2.5 * weight),
                   _const(nr, 1.0)).items()}
    return {"cell_first": cell_first, "parent": parent, "area": area, "ri": ri,
            "cm": _const(N, 1.0), "v_init": -65.0, "celsius": 6.3, "mechs": mechs, "netcons": nc,
            "thr": _const(n_cell, -20.0),
            "stim": {"gid": s_src.astype(np.int32), "t": np.zeros(nr)}, "_type_of": type_of}


# ------------------------------------------------------------------------------------------
# gap junctions: electrical coupling between cells
# ------------------------------------------------------------------------------------------

def with_gap_junctions(desc: dict, n_junction: int, g: float = 0.002, tag="gap",
                       neighbours_only: bool = True) -> dict:
    """`desc` plus n_junction symmetric gap junctions (two `gap` instances each, conductance g uS
    +- 50 % seeded).  The two ends are seeded nodes of different cells; with neighbours_only the
    cells are gid neighbours (c, c+1), the way electrically coupled interneurons sit side by
    side, otherwise any two cells."""
    cf = desc["cell_first"]
    n_cell = len(cf) - 1
    assert n_cell >= 2
    bits = rng.bits((tag, "ends"), 4 * n_junction)
    ca = (bits[0::4] % np.uint64(n_cell)).astype(np.int64)
    if neighbours_only:
        cb = (ca + 1) % n_cell
    else:
        cb = (ca + 1 + (bits[1::4] % np.uint64(n_cell - 1)).astype(np.int64)) % n_cell
    sz = cf[1:] - cf[:-1]
    na = cf[ca] + (bits[2::4] % sz[ca].astype(np.uint64)).astype(np.int64)
    nb = cf[cb] + (bits[3::4] % sz[cb].astype(np.uint64)).astype(np.int64)
    gj = g * rng.uniform((tag, "g"), n_junction, 0.5, 1.5)
    node = np.concatenate([na, nb])
    peer = np.concatenate([nb, na]).astype(np.float64)
    out = dict(desc)
    out["mechs"] = list(desc["mechs"]) + [_mech("gap", node, {"g": np.concatenate([gj, gj]),
                                                            "peer": peer})]
    return out
