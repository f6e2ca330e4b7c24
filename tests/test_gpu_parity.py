"""Parity of the CUDA path (through the C ABI) with the CPU oracle on the same seeded inputs.

Bar (BASELINE.json north_star): identical spike (gid, step) lists and max |dV| <= 1e-6 mV at every
recorded step.  The minimum threshold-detection margin of the oracle run is asserted to be far
above the voltage error, so spike identity is not knife-edge (R16).
"""
import numpy as np
import pytest

import cn_workloads as W

pytestmark = pytest.mark.gpu

DT = 0.025
TOL = 1e-6


@pytest.fixture(autouse=True)
def _gpu(need_gpu):
    pass


@pytest.fixture(params=["coop", "cell", "tape", "tape-step", "tape-w1", "tape-w4", "tape-w8"])
def strategy(request, opts):
    """Both kernels on the same inputs: warp-cooperative groups, or every cell on the interleaved
    (tape) kernel, ragged groups included (tape_min_group=1), with 12 (default for small models), 8, 1 or 4 warps
    (subtree tasks) per group of 32 cells.  The interleaved kernel runs in window mode where the
    model allows it (the probes are then recorded by the kernel itself); "tape-step" forces one
    launch sequence per dt."""
    if request.param.startswith("tape"):
        opts["tape"] = 1
        opts["tape_min_group"] = 1
        if request.param == "tape-step":
            opts["tape_window"] = 0
        if "-w" in request.param:
            opts["tape_w"] = int(request.param.split("-w")[1])
    else:
        # the warp-cooperative layout: one launch sequence per dt (replayed from a CUDA graph), or
        # "cell": the on-chip window kernel, one CTA per cell for a whole min-delay window
        opts["tape"] = 0
        opts["onchip"] = 1 if request.param == "cell" else 0
    return "tape" if request.param.startswith("tape") else "coop"


def run_both(cn, desc, tstop, dt=DT, probes=None, chunks=1, env=None):
    from oracle import OracleModel
    nsteps = int(round(tstop / dt))
    if probes is None:
        probes = np.asarray(desc["cell_first"][:-1], dtype=np.int32)
    o = OracleModel(desc)
    o.set_probes(probes)
    o.run(tstop, dt)
    g = cn.Model(desc)
    g.set_probes(probes, nsteps)
    for j in range(1, chunks + 1):
        g.run(tstop * j / chunks if j < chunks else tstop, dt)
    return o, g


def check(o, g, tol=TOL, min_spikes=0):
    og, os_ = o.get_spikes()
    gg, gs = g.get_spikes()
    assert len(og) >= min_spikes
    tr_o, tr_g = o.get_trace(), g.get_trace()
    assert tr_o.shape == tr_g.shape
    err_t = np.max(np.abs(tr_o - tr_g)) if tr_o.size else 0.0
    err_v = np.max(np.abs(o.get_v() - g.get_v())) if o.n_node else 0.0
    assert err_t <= tol and err_v <= tol, (err_t, err_v)
    assert list(og) == list(gg) and list(os_) == list(gs)
    if len(og):
        assert o.min_margin > 1e3 * max(err_t, err_v, 1e-12), (o.min_margin, err_t)
    return err_t, err_v


def test_config1_full(cn, strategy):
    desc = W.config1()
    probes = np.concatenate([desc["cell_first"][:-1], [30, 60, 100, 487]]).astype(np.int32)
    o, g = run_both(cn, desc, 100.0, probes=probes)
    check(o, g, min_spikes=60)
    for t, s in ((0, 0), (0, 1), (0, 2), (2, 0)):
        assert np.max(np.abs(o.get_state(t, s) - g.get_state(t, s))) < 1e-9


def test_unique_topologies_one_cell_per_warp(cn, strategy):
    desc = W.random_tree_cells(13, 5, 120, stream="gpu-u", weight=0.2, amp=2.0)
    o, g = run_both(cn, desc, 40.0)
    assert g.layout_info()["n_class"] == 13
    assert g.layout_info()["n_tape_group"] == (13 if strategy == "tape" else 0)
    check(o, g, min_spikes=5)


@pytest.mark.parametrize("mech", ["pas", "hh"])
def test_random_trees_of_every_size(cn, strategy, mech):
    """Fuzz of the tree handling of every kernel: 48 unique random topologies from single nodes to
    330 nodes (up to 3 children per node: stars, long unbranched chains, a root with one child),
    passive dendrites or HH on every node, plus degenerate hand-made shapes (a pure chain of 300
    nodes, a star of 60 leaves on the soma)."""
    a = W.random_tree_cells(48, 1, 330, stream="fuzz-" + mech, mech=mech, weight=0.3, amp=3.0)
    chain = W.random_tree_cells(2, 300, 300, stream="fuzz-chain", mech=mech, identical=True, weight=0.3, amp=3.0)
    chain["parent"] = np.concatenate([np.arange(-1, 299), 300 + np.arange(-1, 299)]).astype(np.int32)
    chain["parent"][300] = -1
    star = W.random_tree_cells(2, 61, 61, stream="fuzz-star", mech=mech, identical=True, weight=0.3, amp=3.0)
    star["parent"] = np.concatenate([[-1], np.zeros(60), [-1], np.full(60, 61)]).astype(np.int32)
    desc = W.concat_models([a, chain, star])
    o, g = run_both(cn, desc, 25.0)
    assert g.layout_info()["n_class"] == 50
    check(o, g, min_spikes=20)


def test_identical_random_cells_grouped(cn, strategy, opts):
    desc = W.random_tree_cells(11, 77, 77, stream="gpu-i", identical=True, weight=0.2, amp=2.0)
    if strategy == "coop":      # (a model this small gets one cell per warp unless told otherwise)
        opts["force_g"] = 4
    o, g = run_both(cn, desc, 40.0)
    info = g.layout_info()
    # coop: 4 + 4 + 3 (ragged tail group); tape: one ragged group of 11 lanes
    assert info["n_class"] == 1 and info["n_group"] == (3 if strategy == "coop" else 1)
    check(o, g, min_spikes=5)
    if strategy == "coop":
        opts.pop("force_g", None)
        assert cn.Model(desc).layout_info()["n_group"] == 11


def test_hh_everywhere_config2_shape(cn, strategy):
    desc = W.config2(n_cell=8, ring_size=4, weight=0.05)
    o, g = run_both(cn, desc, 30.0)
    check(o, g, min_spikes=4)


def test_hh_everywhere_small_cells_on_tape(cn, strategy):
    """61-node cells with HH on every node: every node has a mechanism record, every system row
    sits in shared memory (no tensor-memory rows), two rings of 32 cells = two full groups."""
    desc = W.config2(n_cell=64, ring_size=32, depth=2, ncomp_branch=10, weight=0.05)
    o, g = run_both(cn, desc, 30.0)
    assert g.layout_info()["n_tape_group"] == (2 if strategy == "tape" else 0)
    check(o, g, min_spikes=20)
    for s in (0, 1, 2):
        assert np.max(np.abs(o.get_state(0, s) - g.get_state(0, s))) < 1e-9


def test_config3_shape(cn, strategy):
    """Config 3 scaled to 140 cells (14 morphology types x 10): HH + Ca_HVA + SK + cai + pas,
    Exp2Syn with random presynaptic cells and delays, Poisson IClamp drive."""
    desc = W.config3(n_cell=140, syn_per_cell=60)
    o, g = run_both(cn, desc, 40.0)
    info = g.layout_info()
    assert info["n_class"] == 14 and info["n_tape_group"] == (14 if strategy == "tape" else 0)
    check(o, g, min_spikes=100)
    for t, s in ((0, 0), (0, 2), (1, 0), (1, 1), (2, 0), (5, 0), (5, 1)):
        assert np.max(np.abs(o.get_state(t, s) - g.get_state(t, s))) < 1e-9, (t, s)


def test_config5_shape(cn, strategy):
    """Config 5 scaled to 110 cells (55 types x 2, full-size cells of 330-580 compartments):
    ten channel types, AMPA+NMDA synapses with Mg block, delays from 0.1 ms (4 steps).  Every
    node carries a mechanism (Ih), so these cells always run on the warp-cooperative kernel."""
    desc = W.config5(n_cell=110, syn_per_cell=40)
    o, g = run_both(cn, desc, 20.0)
    assert g.layout_info()["n_class"] == 55
    check(o, g, min_spikes=10)
    for t, s in ((0, 0), (0, 1), (3, 1), (4, 0), (6, 1), (7, 0), (10, 0), (10, 3)):
        assert np.max(np.abs(o.get_state(t, s) - g.get_state(t, s))) < 1e-9, (t, s)


def test_config2_one_ring_of_64(cn, strategy):
    desc = W.config2(rings=[1])
    o, g = run_both(cn, desc, 12.0)
    check(o, g, min_spikes=3)


def test_config2_full_size(cn):
    """All four rings of config 2 (256 cells x 601 compartments, HH on every compartment) for its
    full 200 ms, soma voltages compared at every step; default strategy for this size: the
    warp-cooperative layout run by the on-chip window kernel (the 19 MB model is resident in the
    shared memory of the device; one launch per 40-step window)."""
    desc = W.config2()
    assert len(desc["parent"]) == 153856
    o, g = run_both(cn, desc, 200.0)
    info = g.run_info()
    assert info["mode"] == "onchip-window" and info["window_steps"] == 40
    assert g.launch_count <= 2 * 200 + 8
    check(o, g, min_spikes=400)
    for s in (0, 1, 2):
        assert np.max(np.abs(o.get_state(0, s) - g.get_state(0, s))) < 1e-9


def test_config2_full_size_per_step_graph(cn, opts):
    """The same model with one launch sequence per dt (onchip=0), replayed from a CUDA graph."""
    opts["onchip"] = 0
    desc = W.config2()
    o, g = run_both(cn, desc, 30.0)
    info = g.run_info()
    assert info["mode"] == "per-step" and info["graph_replays"] >= 1200 // 20 - 2
    check(o, g, min_spikes=40)


@pytest.mark.parametrize("which", ["config1", "config2", "config3", "config5", "unique"])
def test_onchip_window_matches_oracle(cn, which, opts):
    """On-chip window mode: one CTA keeps one cell in shared memory for a window of
    up to min-delay steps.  Windows of different lengths (cn_run in uneven pieces), probes inside
    the windows, every mechanism type, AMPA+NMDA synapses (their current depends on v: evaluated in
    the kernel from the cell's own voltage), delays from 4 steps."""
    from oracle import OracleModel
    opts.update({"tape": 0, "onchip": 1})
    desc, tstop = {
        "config1": (W.config1(), 60.0),
        "config2": (W.config2(n_cell=8, ring_size=4, weight=0.05), 30.0),
        "config3": (W.config3(n_cell=140, syn_per_cell=60), 40.0),
        "config5": (W.config5(n_cell=110, syn_per_cell=40), 20.0),
        "unique": (W.random_tree_cells(13, 5, 120, stream="gpu-u", weight=0.2, amp=2.0), 40.0),
    }[which]
    nsteps = int(round(tstop / DT))
    cf = desc["cell_first"]
    probes = np.concatenate([cf[:-1], [cf[1] - 1, cf[2] - 3]]).astype(np.int32)
    o = OracleModel(desc)
    o.set_probes(probes)
    o.run(tstop, DT)
    g = cn.Model(desc)
    g.set_probes(probes, nsteps)
    for t in (0.3 * tstop, 0.3 * tstop + DT, 0.3 * tstop + 8 * DT, tstop):
        g.run(t, DT)
    info = g.run_info()
    assert info["mode"] == "onchip-window"
    assert info["window_steps"] == (4 if which == "config5" else 40)
    assert g.steps_done == nsteps and g.launch_count <= 2 * (nsteps // info["window_steps"] + 4) + 4
    check(o, g, min_spikes=5)
    for t, m in enumerate(desc["mechs"]):
        for st in range({"hh": 3, "hhform": 2, "sk": 1, "expsyn": 1, "exp2syn": 2, "ampanmda": 4}.get(m["type"], 0)):
            assert np.max(np.abs(o.get_state(t, st) - g.get_state(t, st))) < 1e-9, (m["type"], st)


def test_onchip_window_one_step_per_call_and_checkpoint(cn, opts):
    """cn_run once per dt (every window one step long) with delays of up to 200 steps, a checkpoint
    in the middle that is continued by the per-step kernel."""
    from oracle import OracleModel
    opts.update({"tape": 0, "onchip": 1})
    desc = W.config3(n_cell=28, syn_per_cell=40)
    o = OracleModel(desc)
    g = cn.Model(desc)
    for k in range(1, 501):
        g.run(k * DT, DT)
    assert g.run_info()["mode"] == "onchip-window"
    h = cn.Model(desc, options={"onchip": 0})
    h.restore(g.checkpoint())
    h.run(700 * DT, DT)
    g.run(700 * DT, DT)
    o.run(700 * DT, DT)
    for x in (g, h):
        assert np.max(np.abs(o.get_v() - x.get_v())) <= TOL
        assert [list(a) for a in x.get_spikes()] == [list(a) for a in o.get_spikes()]
    assert len(o.get_spikes()[0]) >= 20


def test_graph_replay_equals_direct_launches(cn, opts):
    """Per-dt launch sequences replayed from a CUDA graph (20 steps per graph, a device-side step
    counter) against the same launches issued one by one: bit-identical, on both kernels, with
    probes, in uneven pieces."""
    for base in ({"tape": 0, "onchip": 0}, {"tape": 1, "tape_window": 0, "tape_min_group": 1}):
        desc = W.config4(n_cell=128, n_types=4)
        probes = np.asarray(desc["cell_first"][:8], np.int32)
        res = []
        for graph in (1, 0):
            m = cn.Model(desc, options=dict(base, graph=graph))
            m.set_probes(probes, 700)
            for k in (7, 48, 49, 300, 641, 800):
                m.run(k * DT, DT)
            assert (m.run_info()["graph_replays"] > 25) == (graph == 1)
            res.append((m.get_v(), m.get_spikes(), m.get_trace()))
        assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][2], res[1][2])
        assert res[0][2].shape == (700, 8)
        assert [list(x) for x in res[0][1]] == [list(x) for x in res[1][1]]
        assert len(res[0][1][0]) > 20


def test_config4_small_full_length(cn, strategy):
    desc = W.config4(n_cell=256, n_types=8)
    o, g = run_both(cn, desc, 50.0)
    assert g.layout_info()["n_class"] == 8
    assert g.layout_info()["n_tape_group"] == (8 if strategy == "tape" else 0)
    check(o, g, min_spikes=100)


def test_mixed_strategies_in_one_model(cn, opts):
    """Classes of 40 cells: 32 go to one tape group, the ragged 8 to warp-cooperative groups."""
    opts["tape"] = 1
    opts["force_g"] = 4
    desc = W.config4(n_cell=320, n_types=8, ring_size=64)
    o, g = run_both(cn, desc, 30.0)
    info = g.layout_info()
    assert info["n_tape_group"] == 8 and info["n_group"] == 8 + 8 * 2
    check(o, g, min_spikes=50)


def test_chunked_run_equals_one_shot(cn, strategy):
    desc = W.config1()
    a = cn.Model(desc)
    a.run(20.0, DT)
    b = cn.Model(desc)
    for t in (0.025, 1.0, 1.0, 7.3, 7.325, 20.0):
        b.run(t, DT)
    assert b.steps_done == 800 == a.steps_done
    assert np.array_equal(a.get_v(), b.get_v())
    assert [list(x) for x in a.get_spikes()] == [list(x) for x in b.get_spikes()]


@pytest.mark.parametrize("which", ["config3", "config5"])
def test_runs_with_many_synapses_per_node_are_bit_reproducible(cn, strategy, which):
    """Several synapses per node and several events per step: the conductance / current of a
    node's point processes is summed in fixed point, so the order in which the atomics land
    cannot change a bit."""
    desc = W.config3(n_cell=140, syn_per_cell=300) if which == "config3" else \
        W.config5(n_cell=110, syn_per_cell=400)
    r = []
    for _ in range(3):
        m = cn.Model(desc)
        m.run(15.0, DT)
        r.append((m.get_v(), m.get_spikes(), m.get_state(len(desc["mechs"]) - 2, 1)))
    for x in r[1:]:
        assert np.array_equal(r[0][0], x[0]) and np.array_equal(r[0][2], x[2])
        assert [list(a) for a in r[0][1]] == [list(a) for a in x[1]]
    assert len(r[0][1][0]) >= 5


def test_run_is_deterministic(cn, strategy):
    desc = W.config4(n_cell=128, n_types=4)
    r = []
    for _ in range(2):
        m = cn.Model(desc)
        m.run(30.0, DT)
        r.append((m.get_v(), m.get_spikes()))
    assert np.array_equal(r[0][0], r[1][0])
    assert [list(x) for x in r[0][1]] == [list(x) for x in r[1][1]]


def test_edge_cases(cn, strategy):
    from oracle import OracleModel
    # empty model
    empty = {"cell_first": np.zeros(1, np.int64), "parent": np.zeros(0, np.int32),
             "area": np.zeros(0), "ri": np.zeros(0), "cm": np.zeros(0), "mechs": [],
             "netcons": {k: np.zeros(0) for k in ("src", "tgt_mech", "tgt_inst", "weight", "delay")},
             "thr": np.zeros(0), "stim": {"gid": np.zeros(0, np.int32), "t": np.zeros(0)}}
    m = cn.Model(empty)
    m.run(1.0, DT)
    assert m.steps_done == 40 and len(m.get_v()) == 0 and len(m.get_spikes()[0]) == 0
    # single passive compartment: closed-form backward Euler decay
    d = W.single_compartment([("pas", {"g": 0.001, "e": -65.0}, {})], v_init=-50.0)
    m = cn.Model(d)
    m.set_probes([0], 200)
    m.run(5.0, DT)
    n = np.arange(1, 201)
    assert np.max(np.abs(m.get_trace()[:, 0] - (-65.0 + 15.0 * (1 + DT / 1.0) ** (-n)))) < 1e-11
    # mechanism-free cell next to single-node cells
    d = W.random_tree_cells(3, 1, 1, stream="gpu-e1", weight=0.5)
    o, g = run_both(cn, d, 10.0)
    check(o, g)
    # tstop not after the current time is a no-op; dt change is an error
    g.run(5.0, DT)
    assert g.steps_done == 400
    with pytest.raises(cn.CnError) as e:
        g.run(20.0, 0.0125)
    assert e.value.code == -5
    # delay below one step
    d = W.config1()
    d["netcons"] = dict(d["netcons"]); d["netcons"]["delay"] = np.full(8, 0.01)
    with pytest.raises(cn.CnError) as e:
        cn.Model(d).run(1.0, DT)
    assert e.value.code == -4
    # spike buffer overflow is reported
    m = cn.Model(W.config1())
    m.set_spike_capacity(3)
    with pytest.raises(cn.CnError) as e:
        m.run(30.0, DT)
    assert e.value.code == -7


def test_scripted_sources_and_delays(cn, strategy):
    from tests.test_oracle_pins import _syn_target
    for ks in (0, 7):
        d = _syn_target([1 * DT, 40 * DT, 400 * DT], ks * DT)
        o, g = run_both(cn, d, (ks + 402) * DT)
        check(o, g)
        assert np.max(np.abs(o.get_state(1, 0) - g.get_state(1, 0))) < 1e-15


def test_node_renumbering_invariance(cn, strategy):
    desc = W.random_tree_cells(4, 30, 60, stream="gpu-r", weight=0.4, amp=4.0)
    ren = W.renumber_nodes(desc)
    a, b = cn.Model(desc), cn.Model(ren)
    a.run(15.0, DT)
    b.run(15.0, DT)
    assert np.max(np.abs(b.get_v()[ren["_new_of_old"]] - a.get_v())) < 1e-9
    assert [list(x) for x in a.get_spikes()] == [list(x) for x in b.get_spikes()]


@pytest.mark.parametrize("which", ["config3", "config5"])
def test_instance_order_invariance(cn, strategy, which):
    """The instances of every mechanism table in a random order (tables not ordered by node take
    the general path of the per-cell instance lists): same voltages, spikes and states, bit for
    bit -- one distributed instance per node, point-process sums are fixed-point."""
    desc = W.config3(n_cell=140, syn_per_cell=60) if which == "config3" else \
        W.config5(n_cell=110, syn_per_cell=40)
    shuf = W.shuffle_instances(desc)
    a, b = cn.Model(desc), cn.Model(shuf)
    a.run(20.0, DT)
    b.run(20.0, DT)
    assert len(a.get_spikes()[0]) > 0
    assert np.array_equal(a.get_v(), b.get_v())
    assert [list(x) for x in a.get_spikes()] == [list(x) for x in b.get_spikes()]
    for t, m in enumerate(desc["mechs"]):
        s = 0
        while True:
            try:
                sa = a.get_state(t, s)
            except cn.CnError:
                break
            assert np.array_equal(sa, b.get_state(t, s)[shuf["_new_of_old_inst"][t]]), (t, s)
            s += 1


@pytest.mark.parametrize("force_g", ["1", "2", "8"])
def test_lanes_per_cell_variants(cn, force_g, opts):
    opts["tape"] = 0       # the warp-cooperative kernel, G cells per warp
    opts["force_g"] = int(force_g)
    desc = W.config4(n_cell=64, n_types=2)
    o, g = run_both(cn, desc, 30.0)
    check(o, g, min_spikes=10)


@pytest.mark.parametrize("which", ["config1", "config4", "config3", "unique"])
def test_window_mode_matches_oracle(cn, which, opts):
    """Without per-step probes a model whose cells all sit on the interleaved kernel runs in
    WINDOW mode: one launch integrates up to min-delay steps, (step, group) work items are handed
    out by a ticket counter, events and point processes of the window are prepared up front.
    Final voltages, states and the whole spike list must still match the oracle."""
    from oracle import OracleModel
    opts["tape"] = 1
    opts["tape_min_group"] = 1
    desc, tstop = {
        "config1": (W.config1(), 60.0),
        "config4": (W.config4(n_cell=256, n_types=8), 50.0),
        "config3": (W.config3(n_cell=140, syn_per_cell=60), 40.0),
        "unique": (W.random_tree_cells(13, 5, 120, stream="gpu-u", weight=0.2, amp=2.0), 40.0),
    }[which]
    o = OracleModel(desc)
    o.run(tstop, DT)
    g = cn.Model(desc)
    for t in (0.3 * tstop, 0.3 * tstop + DT, tstop):      # windows of different lengths
        g.run(t, DT)
    nsteps = int(round(tstop / DT))
    assert g.steps_done == nsteps and g.launch_count < nsteps      # not one launch per step
    err = np.max(np.abs(o.get_v() - g.get_v()))
    assert err <= TOL, err
    og, os_ = o.get_spikes()
    gg, gs = g.get_spikes()
    assert len(og) >= 5 and list(og) == list(gg) and list(os_) == list(gs)
    assert o.min_margin > 1e3 * max(err, 1e-12)
    for t, m in enumerate(desc["mechs"]):
        if m["type"] in ("hh", "expsyn", "exp2syn", "sk"):
            assert np.max(np.abs(o.get_state(t, 0) - g.get_state(t, 0))) < 1e-9, m["type"]


def test_window_mode_one_step_per_call(cn, opts):
    """cn_run called once per dt for 300 steps with delays of up to 200 steps: every window is one
    step long, the events of spikes recorded 200 windows ago must still be found."""
    from oracle import OracleModel
    opts["tape"] = 1
    opts["tape_min_group"] = 1
    desc = W.config3(n_cell=28, syn_per_cell=40)
    assert np.round(desc["netcons"]["delay"].max() / DT) == 200
    o = OracleModel(desc)
    g = cn.Model(desc)
    for k in range(1, 701):
        g.run(k * DT, DT)
    o.run(700 * DT, DT)
    assert g.launch_count <= 3 * 700 + 8
    assert np.max(np.abs(o.get_v() - g.get_v())) <= TOL
    og, os_ = o.get_spikes()
    gg, gs = g.get_spikes()
    assert len(og) >= 20 and list(og) == list(gg) and list(os_) == list(gs)


@pytest.mark.parametrize("per_type", [32, 4])
def test_fig5f_node_ordering_workload(cn, per_type):
    """The paper's node-ordering workload (83-node cells, random branching of 40 dendrites,
    PAPER.md L204) at 2,048 cells... the library picks the interleaved kernel for 32 identical
    cells per type and the warp-cooperative one for 4; both must match the oracle."""
    desc = W.fig5f(n_cell=8192, per_type=per_type)
    o, g = run_both(cn, desc, 8.0, probes=np.asarray(desc["cell_first"][:64], dtype=np.int32))
    info = g.layout_info()
    assert (info["n_tape_group"] > 0) == (per_type == 32)
    check(o, g, min_spikes=300)


# ---------------------------------------------------------------------------------------------
# gap junctions
# ---------------------------------------------------------------------------------------------

def test_gap_junctions_between_ring_cells(cn, strategy):
    """HH ring cells with 60 symmetric gap junctions between neighbours (any node to any node):
    the peer voltages are the ones of the start of the step.  The coupling is strong enough to
    move the spike times (checked on the oracle), so a dropped or mis-addressed junction fails."""
    from oracle import OracleModel
    base = W.config2(n_cell=64, ring_size=32, depth=2, ncomp_branch=10, weight=0.05)
    desc = W.with_gap_junctions(base, 60, g=0.02)
    o, g = run_both(cn, desc, 30.0)
    check(o, g, min_spikes=20)
    ob = OracleModel(base)
    ob.run(30.0, DT)
    assert [list(x) for x in ob.get_spikes()] != [list(x) for x in o.get_spikes()]
    # without probes the model would qualify for window mode but for the junctions (their current
    # depends on the voltages of the step before): one launch sequence per dt, same results
    g2 = cn.Model(desc)
    g2.run(30.0, DT)
    assert g2.launch_count >= 1200
    assert np.max(np.abs(o.get_v() - g2.get_v())) <= TOL
    assert [list(x) for x in g2.get_spikes()] == [list(x) for x in o.get_spikes()]


def test_gap_junctions_across_kernels(cn, opts):
    """Junctions between cells on the interleaved kernel (groups of >= 16 identical cells) and
    cells on the warp-cooperative kernel (unique topologies): the peer position addresses the
    one voltage arena both kernels write."""
    opts["tape"] = 1
    opts["tape_min_group"] = 16
    a = W.random_tree_cells(24, 40, 40, stream="gap-a", identical=True, weight=0.2, amp=2.0)
    b = W.random_tree_cells(9, 20, 90, stream="gap-b", weight=0.2, amp=2.0)
    desc = W.with_gap_junctions(W.concat_models([a, b]), 50, g=0.01, neighbours_only=False)
    o, g = run_both(cn, desc, 30.0)
    info = g.layout_info()
    assert info["n_tape_group"] >= 1 and info["n_group"] > info["n_tape_group"]
    check(o, g, min_spikes=5)


def test_probe_capacity_and_interior_nodes(cn, strategy):
    """Probes on interior nodes of several cells (two of them in the same group), a trace capacity
    shorter than the run, cn_run in uneven pieces: the first `cap` rows must be the oracle's, the
    rest is dropped -- whether a probe kernel follows every step or the interleaved kernel records
    the voltages itself (window mode)."""
    desc = W.config4(n_cell=128, n_types=2)
    cf = desc["cell_first"]
    probes = np.array([cf[0], cf[0] + 17, cf[1] + 290, cf[70] + 5, cf[127] + 100, cf[64]], np.int32)
    cap, nsteps = 150, 400
    from oracle import OracleModel
    o = OracleModel(desc)
    o.set_probes(probes)
    o.run(nsteps * DT, DT)
    g = cn.Model(desc)
    g.set_probes(probes, cap)
    for k in (3, 44, 149, 151, 290, nsteps):
        g.run(k * DT, DT)
    tr = g.get_trace()
    assert tr.shape == (cap, len(probes))
    assert np.max(np.abs(tr - o.get_trace()[:cap])) <= TOL
    assert np.max(np.abs(g.get_v() - o.get_v())) <= TOL
    assert [list(x) for x in g.get_spikes()] == [list(x) for x in o.get_spikes()]


def test_device_memory_returns_after_destroy(cn):
    """Every device allocation of a model (the arena, tables, the compact arrays that a large
    model uploads at cn_model_create, scratch) is released by cn_model_destroy -- run or not run,
    read back or not."""
    import torch
    desc = W.config4(n_cell=320, n_types=8, ring_size=64)     # 93,120 nodes: the early upload path
    def free():
        torch.cuda.synchronize()
        return torch.cuda.mem_get_info()[0]
    cases = (({"tape": 1}, True), ({"tape": 1}, False), ({"tape": 1, "tape_min_group": 32}, True),
             ({"tape": 0}, True), (None, False))

    def cycle(opts, run):
        m = cn.Model(desc, options=opts)
        if run:
            m.run(2.0, DT)
            m.get_v()
            m.get_state(0, 0)
            m.checkpoint()
        m.destroy()

    for opts, run in cases:      # first pass: context, lazy loading of every kernel involved
        cycle(opts, run)
    base = free()
    for rep in range(2):
        for opts, run in cases:
            cycle(opts, run)
            assert free() == base, (rep, opts, run, base - free())
