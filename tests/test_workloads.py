"""Shape checks of the seeded synthetic workloads against BASELINE.json's configs (CPU only).

The generators hold no arithmetic of the method; what is checked here is that the inputs have the
sizes, distributions and structure the configs state.
"""
import numpy as np

import cn_workloads as W

DT = 0.025


def _forest_ok(desc):
    cf, par = desc["cell_first"], desc["parent"].astype(np.int64)
    for c in range(0, len(cf) - 1, max(1, (len(cf) - 1) // 50)):
        f, l = int(cf[c]), int(cf[c + 1])
        assert par[f] == -1
        p = par[f + 1:l]
        assert np.all(p >= f) and np.all(p < np.arange(f + 1, l))
    assert np.all(desc["area"] > 0) and np.all(desc["ri"] > 0) and np.all(np.isfinite(desc["ri"]))


def test_config3_sizes_and_distributions():
    d = W.config3()
    n_cell = len(d["cell_first"]) - 1
    assert n_cell == 3560 and len(d["parent"]) == 465740          # Table 1 "Traub" (R20)
    assert len(np.unique(d["_type_of"])) == 14
    sizes = np.diff(d["cell_first"])
    assert abs(sizes.mean() - 465740 / 3560) < 1e-9 and len(np.unique(sizes)) >= 10
    _forest_ok(d)
    types = [m["type"] for m in d["mechs"]]
    assert types == ["hh", "hhform", "sk", "cadyn", "pas", "exp2syn", "iclamp"]
    syn = d["mechs"][5]
    assert len(syn["node"]) == 1100040 and np.all(syn["params"]["tau1"] == 0.5)
    assert np.all(syn["params"]["tau2"] == 5.0)
    nc = d["netcons"]
    assert len(nc["src"]) == 1100040 and nc["src"].min() >= 0 and nc["src"].max() < n_cell
    steps = np.round(nc["delay"] / DT)
    assert steps.min() == 40 and steps.max() == 200 and np.allclose(steps * DT, nc["delay"])
    # presynaptic cells uniform: chi-square-ish bound on the per-cell counts
    cnt = np.bincount(nc["src"], minlength=n_cell)
    assert abs(cnt.mean() - 309) < 1e-9 and cnt.std() < 1.3 * np.sqrt(309)
    lw = np.log(nc["weight"] / 0.1)                                # w_scale = 0.1 (tuned, frozen)
    assert abs(lw.mean() + 4.0) < 0.01 and abs(lw.std() - 0.5) < 0.01
    # synapses sit on dendritic nodes of their own cell, 309 per cell
    cell_of_syn = np.searchsorted(d["cell_first"], syn["node"], side="right") - 1
    assert np.all(np.bincount(cell_of_syn, minlength=n_cell) == 309)
    assert not np.any(np.isin(syn["node"], d["cell_first"][:-1]))
    # 10 % of the cells are driven by 2 ms pulses on the step grid
    ic = d["mechs"][6]
    assert 340 <= len(np.unique(ic["node"])) <= 356 and np.all(ic["params"]["dur"] == 2.0)
    k = ic["params"]["del"] / DT
    assert np.allclose(k, np.round(k)) and ic["params"]["del"].max() < 100.0
    rate = len(k) / 356 / 0.1
    assert 30.0 < rate < 50.0                                      # 40 Hz Poisson
    assert W.desc_hash(d) == W.desc_hash(W.config3())              # seeded, reproducible


def test_config5_shape_at_small_scale():
    d = W.config5(n_cell=550, syn_per_cell=40)
    n_cell = len(d["cell_first"]) - 1
    assert n_cell == 550 and len(np.unique(d["_type_of"])) == 55
    sizes = np.diff(d["cell_first"])
    assert 330 <= sizes.min() and sizes.max() < 580 and 420 < sizes.mean() < 490   # "~454"
    _forest_ok(d)
    types = [m["type"] for m in d["mechs"]]
    assert types.count("hhform") == 7 and "sk" in types and "cadyn" in types and "pas" in types
    assert types[10] == "ampanmda" and len(d["mechs"][10]["node"]) == 550 * 40
    # ten channel types on every cell
    for m in d["mechs"][:10]:
        cells = np.unique(np.searchsorted(d["cell_first"], m["node"], side="right") - 1)
        assert len(cells) == n_cell, m["type"]
    steps = np.round(d["netcons"]["delay"] / DT)
    assert steps.min() == 4 and steps.max() == 400
    assert d["netcons"]["src"].max() < n_cell
    # full-scale bookkeeping without building it: 20,000 cells x 4,000 synapses
    full_cells, full_syn = int(round(20000 * 1.0)), int(round(4000 * 1.0))
    assert full_cells * full_syn == 80_000_000


def test_config4_headline_sizes_small_copy():
    d = W.config4(n_cell=2048, n_types=64)
    assert np.all(np.diff(d["cell_first"]) == 291)
    assert len(d["netcons"]["src"]) == 2048 + 2048 // 64          # ring NetCons + one source per ring
    _forest_ok(d)


def test_fig5f_node_ordering_workload_shape():
    d = W.fig5f(n_cell=4096, per_type=4)
    assert np.all(np.diff(d["cell_first"]) == 83)              # 83 nodes per cell
    assert 131072 * 83 == 10878976                             # ... 10,878,976 nodes at full size
    _forest_ok(d)
    par = d["parent"].astype(np.int64)
    # cells of one type share the branching pattern, different types differ
    loc = (par.reshape(4096, 83) - d["cell_first"][:-1, None])[:, 1:]
    assert np.array_equal(loc[0], loc[3]) and not np.array_equal(loc[0], loc[4])
    assert len(np.unique(loc, axis=0)) == 1024
    assert len(d["netcons"]["src"]) == 4096 + 64


def test_concat_models_is_block_diagonal():
    from oracle import OracleModel
    a = W.random_tree_cells(5, 10, 10, stream="cat-a", identical=True, weight=0.2, amp=2.0)
    b = W.random_tree_cells(4, 8, 30, stream="cat-b", weight=0.2, amp=2.0)
    ab = W.concat_models([a, b])
    oa, ob, oab = OracleModel(a), OracleModel(b), OracleModel(ab)
    for o in (oa, ob, oab):
        o.run(20.0, 0.025)
    assert np.array_equal(np.concatenate([oa.get_v(), ob.get_v()]), oab.get_v())
    ga, sa = oa.get_spikes()
    gb, sb = ob.get_spikes()
    gab, sab = oab.get_spikes()
    assert len(ga) > 2 and len(gb) > 2
    assert sorted(zip(sab, gab)) == sorted(list(zip(sa, ga)) + list(zip(sb, gb + 5)))


def test_gap_junction_generator():
    base = W.config2(n_cell=16, ring_size=8, depth=2, ncomp_branch=4)
    d = W.with_gap_junctions(base, 25, g=0.01)
    gj = d["mechs"][-1]
    assert gj["type"] == "gap" and len(gj["node"]) == 50
    node, peer = gj["node"].astype(np.int64), gj["params"]["peer"].astype(np.int64)
    assert np.array_equal(node[:25], peer[25:]) and np.array_equal(node[25:], peer[:25])
    assert np.array_equal(gj["params"]["g"][:25], gj["params"]["g"][25:])
    cf = d["cell_first"]
    ca = np.searchsorted(cf, node, side="right") - 1
    cb = np.searchsorted(cf, peer, side="right") - 1
    assert np.all((cb[:25] - ca[:25]) % 16 == 1)          # gid neighbours
    d2 = W.with_gap_junctions(base, 25, g=0.01, neighbours_only=False)
    p2 = d2["mechs"][-1]["params"]["peer"].astype(np.int64)
    n2 = d2["mechs"][-1]["node"].astype(np.int64)
    assert np.all(np.searchsorted(cf, n2, side="right") != np.searchsorted(cf, p2, side="right"))
    assert len(base["mechs"]) + 1 == len(d["mechs"])      # the input is left alone
