"""Checkpoint / restore through the C ABI on the GPU.

A run that is saved at T1, loaded into a FRESH model of the same description and continued to T2
must end exactly where the uninterrupted run ends -- including the events that were in flight at
T1, which the checkpoint does not store: they are regenerated from the recorded spikes (L156) --
and both must match the oracle.  A checkpoint holds state only, in the caller's order: it loads
into models with other stimuli ("launch multiple simulations with different stimuli", L156), other
launch modes and the other kernel.
"""
import numpy as np
import pytest

import cn_workloads as W

pytestmark = pytest.mark.gpu
DT = 0.025


@pytest.fixture(autouse=True)
def _gpu(need_gpu):
    pass


TAPE = {"tape": 1, "tape_min_group": 1}
CASES = {
    "config1-onchip": (lambda: W.config1(), {}, 13.7, 40.0),
    "config1-window": (lambda: W.config1(), TAPE, 13.7, 40.0),
    "config1-per-step": (lambda: W.config1(), dict(TAPE, tape_window=0), 13.7, 40.0),
    "config1-coop": (lambda: W.config1(), {"tape": 0, "onchip": 0}, 13.7, 40.0),
    "config4-window": (lambda: W.config4(n_cell=256, n_types=8), TAPE, 20.3, 45.0),
    "config3-window": (lambda: W.config3(n_cell=140, syn_per_cell=60), TAPE, 9.1, 30.0),
    "config3-onchip": (lambda: W.config3(n_cell=140, syn_per_cell=60), {}, 9.1, 30.0),
    "config5-coop": (lambda: W.config5(n_cell=110, syn_per_cell=40), {"onchip": 0}, 6.0, 16.0),
    "config5-onchip": (lambda: W.config5(n_cell=110, syn_per_cell=40), {}, 6.0, 16.0),
}


@pytest.mark.parametrize("case", sorted(CASES))
def test_save_load_continue_equals_straight_run(cn, case, opts):
    from oracle import OracleModel
    make, env, t1, t2 = CASES[case]
    opts.update(env)
    desc = make()
    a = cn.Model(desc)
    a.run(t2, DT)
    b = cn.Model(desc)
    b.run(t1, DT)
    ck = b.checkpoint()
    assert ck.dtype == np.uint8 and ck.size > 64
    b.run(t1 + 2.0, DT)                       # the saved state is a copy: b may go on
    c = cn.Model(desc)                        # a fresh model that never ran
    c.restore(ck)
    assert c.steps_done == int(round(t1 / DT))
    c.run(t2, DT)
    assert c.steps_done == a.steps_done
    exact = True    # (point-process sums are fixed-point: no dependence on the order of the atomics)
    dv = np.max(np.abs(a.get_v() - c.get_v()))
    assert dv == 0.0, dv
    assert [list(x) for x in a.get_spikes()] == [list(x) for x in c.get_spikes()]
    for t, m in enumerate(desc["mechs"]):
        if m["type"] in ("hh", "hhform", "sk", "expsyn", "exp2syn", "ampanmda"):
            ds = np.max(np.abs(a.get_state(t, 0) - c.get_state(t, 0)))
            assert ds == 0.0 if exact else ds < 1e-9, (m["type"], ds)
    o = OracleModel(desc)
    o.run(t2, DT)
    assert np.max(np.abs(o.get_v() - c.get_v())) <= 1e-6
    og, os_ = o.get_spikes()
    cg, cs = c.get_spikes()
    assert len(og) > 0 and list(og) == list(cg) and list(os_) == list(cs)
    # a checkpoint is loadable into a model that already ran, too (rewinds it)
    b.restore(ck)
    b.run(t2, DT)
    assert np.array_equal(b.get_v(), c.get_v()) or not exact


def test_checkpoint_rejects_other_models(cn):
    a = cn.Model(W.config1())
    a.run(1.0, DT)
    ck = a.checkpoint()
    other = cn.Model(W.config4(n_cell=64, n_types=2))
    with pytest.raises(cn.CnError) as e:
        other.restore(ck)
    assert e.value.code == -1
    with pytest.raises(cn.CnError):
        cn.Model(W.config1()).restore(ck[:40])
    fresh = cn.Model(W.config1())
    with pytest.raises(cn.CnError):
        fresh.checkpoint()                    # nothing to save before the first cn_run
    # same sizes, other topology: the structure hash covers parent[]
    d = W.config1()
    d["parent"] = d["parent"].copy()
    d["parent"][20] = 10
    with pytest.raises(cn.CnError) as e:
        cn.Model(d).restore(ck)
    assert e.value.code == -1


def _corrupt(ck, what):
    import struct
    b = ck.copy()
    # header: magic u64, k, n_sp, n_node, n_cell, n_state_doubles, has_cai, total_bytes (i64), dt f64, hash u64
    if what == "truncated":
        return b[:len(b) - 8]
    if what == "dt-nan":
        b[64:72] = np.frombuffer(struct.pack("<d", float("nan")), np.uint8)
    elif what == "dt-negative":
        b[64:72] = np.frombuffer(struct.pack("<d", -0.025), np.uint8)
    elif what == "n_sp-negative":
        b[16:24] = np.frombuffer(struct.pack("<q", -3), np.uint8)
    elif what == "n_sp-huge":
        b[16:24] = np.frombuffer(struct.pack("<q", 1 << 40), np.uint8)
    elif what == "spike-gid":
        b[len(b) - 8 * 5 - 4 * 6:len(b) - 8 * 5 - 4 * 6 + 4] = np.frombuffer(struct.pack("<i", 999), np.uint8)
    elif what == "magic":
        b[0] ^= 1
    return b


@pytest.mark.parametrize("what", ["truncated", "dt-nan", "dt-negative", "n_sp-negative", "n_sp-huge",
                                  "spike-gid", "magic"])
def test_rejected_buffer_leaves_the_model_untouched(cn, what):
    """Every check runs before the first write: a corrupt or truncated buffer is refused and the
    model -- fresh or running -- continues exactly like a model that never saw it."""
    desc = W.config1()
    a = cn.Model(desc)
    a.run(10.0, DT)
    ck = a.checkpoint()
    assert len(a.get_spikes()[0]) >= 5
    bad = _corrupt(ck, what)
    ref = cn.Model(desc)
    ref.run(14.0, DT)
    for fresh in (True, False):
        m = cn.Model(desc)
        if not fresh:
            m.run(3.0, DT)
        with pytest.raises(cn.CnError):
            m.restore(bad)
        assert m.steps_done == (0 if fresh else 120)
        m.run(14.0, DT)                       # (a fresh model must not have been finalized with a bad dt)
        assert np.array_equal(m.get_v(), ref.get_v())
        assert [list(x) for x in m.get_spikes()] == [list(x) for x in ref.get_spikes()]


def _with_late_stimuli(desc, variant, t_on):
    """The description with extra stimuli that start after t_on: IClamp pulses on other cells and a
    scripted source that drives cell 5's synapse (variant-specific)."""
    d = dict(desc)
    d["mechs"] = [dict(m) for m in desc["mechs"]]
    ic = next(j for j, m in enumerate(d["mechs"]) if m["type"] == "iclamp")
    syn = next(j for j, m in enumerate(d["mechs"]) if m["type"] == "expsyn")
    roots = np.asarray(desc["cell_first"][:-1], np.int32)
    old = d["mechs"][ic]
    # four extra IClamp instances on the same nodes in every variant (the structure must match);
    # which of them ever fire, when and how strongly, is the variant's business
    extra = roots[[2, 6, 4, 7]]
    if variant == "A":
        dels, amp = [t_on + 1.0, t_on + 4.0, 1e9, 1e9], 0.6
    else:
        dels, amp = [1e9, 1e9, t_on + 1.5, 1e9], 0.9
    d["mechs"][ic] = {"type": "iclamp", "globals": {},
                      "node": np.concatenate([old["node"], extra]).astype(np.int32),
                      "params": {"del": np.concatenate([old["params"]["del"], dels]),
                                 "dur": np.concatenate([old["params"]["dur"], [1.0] * 4]),
                                 "amp": np.concatenate([old["params"]["amp"], [amp] * 4])}}
    n_cell = len(roots)
    nc = desc["netcons"]
    d["netcons"] = {"src": np.concatenate([nc["src"], [n_cell]]).astype(np.int32),
                    "tgt_mech": np.concatenate([nc["tgt_mech"], [syn]]).astype(np.int32),
                    "tgt_inst": np.concatenate([nc["tgt_inst"], [5]]).astype(np.int64),
                    "weight": np.concatenate([nc["weight"], [0.08]]),
                    "delay": np.concatenate([nc["delay"], [1.0]])}
    d["stim"] = {"gid": np.full(2, n_cell, np.int32),
                 "t": np.array([t_on + 2.0, t_on + (9.0 if variant == "A" else 4.5)])}
    return d


@pytest.mark.parametrize("mode", ["window", "per-step", "coop", "onchip"])
def test_restart_with_different_stimuli(cn, mode, opts):
    """save at T1, restore into models whose stimuli differ after T1 (IClamp tables,
    scripted sources); each continuation must equal ITS OWN uninterrupted oracle run (the variants
    agree up to T1 because their stimuli only start later, so the state at T1 is theirs too)."""
    from oracle import OracleModel
    opts.update({"window": TAPE, "per-step": dict(TAPE, tape_window=0), "coop": {"tape": 0, "onchip": 0},
                 "onchip": {}}[mode])
    t1, t2 = 12.0, 40.0
    base = W.config1()
    a_desc, b_desc = _with_late_stimuli(base, "A", t1), _with_late_stimuli(base, "B", t1)
    src = cn.Model(a_desc)
    src.run(t1, DT)
    ck = src.checkpoint()
    results = {}
    for name, d in (("A", a_desc), ("B", b_desc)):
        g = cn.Model(d)
        g.restore(ck)
        g.run(t2, DT)
        o = OracleModel(d)
        o.run(t2, DT)
        assert np.max(np.abs(o.get_v() - g.get_v())) <= 1e-6, name
        assert [list(x) for x in g.get_spikes()] == [list(x) for x in o.get_spikes()], name
        results[name] = [list(x) for x in g.get_spikes()]
    assert results["A"] != results["B"]       # the stimuli do change the continuation


def test_checkpoint_moves_between_kernels_and_launch_modes(cn):
    """The file holds state in the caller's order and nothing of the layout: saved by the
    interleaved kernel in window mode, continued on the warp-cooperative kernel, and back."""
    from oracle import OracleModel
    desc = W.config3(n_cell=140, syn_per_cell=60)
    t1, t2, t3 = 9.1, 20.0, 30.0
    a = cn.Model(desc, options=TAPE)                    # interleaved, window mode
    a.run(t1, DT)
    assert a.run_info()["mode"] == "window"
    b = cn.Model(desc, options={"tape": 0, "onchip": 0})  # warp-cooperative, per step
    b.restore(a.checkpoint())
    b.run(t2, DT)
    c = cn.Model(desc, options={"tape": 1, "tape_window": 0, "tape_min_group": 1})
    c.restore(b.checkpoint())
    c.run(t3, DT)
    o = OracleModel(desc)
    o.run(t3, DT)
    assert np.max(np.abs(o.get_v() - c.get_v())) <= 1e-6
    assert [list(x) for x in c.get_spikes()] == [list(x) for x in o.get_spikes()]
    for t, m in enumerate(desc["mechs"]):
        if m["type"] in ("hh", "hhform", "sk", "exp2syn"):
            assert np.max(np.abs(o.get_state(t, 0) - c.get_state(t, 0))) < 1e-9, m["type"]
    # state-sized: 8 B per node and state, not a dump of the tapes
    n_state = sum(len(m["node"]) * {"hh": 3, "hhform": 2, "sk": 1, "exp2syn": 2}.get(m["type"], 0)
                  for m in desc["mechs"])
    assert a.checkpoint().size < 8 * (2 * len(desc["parent"]) + n_state) + 64 * 1024
