"""Checkpoint / restore through the C ABI on the GPU.

A run that is saved at T1, loaded into a FRESH model of the same description and continued to T2
must end exactly where the uninterrupted run ends -- including the events that were in flight at
T1, which the checkpoint does not store: they are regenerated from the recorded spikes (L156) --
and both must match the oracle.
"""
import numpy as np
import pytest

import cn_workloads as W

pytestmark = pytest.mark.gpu
DT = 0.025


@pytest.fixture(scope="module")
def cn():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1901_10975_b200.build import build
    build()
    import paper_1901_10975_b200 as cn
    return cn


CASES = {
    "config1-window": (lambda: W.config1(), {}, 13.7, 40.0),
    "config1-per-step": (lambda: W.config1(), {"CN_TAPE_WINDOW": "0"}, 13.7, 40.0),
    "config1-coop": (lambda: W.config1(), {"CN_TAPE": "0"}, 13.7, 40.0),
    "config4-window": (lambda: W.config4(n_cell=256, n_types=8), {}, 20.3, 45.0),
    "config3-window": (lambda: W.config3(n_cell=140, syn_per_cell=60), {}, 9.1, 30.0),
    "config5-coop": (lambda: W.config5(n_cell=110, syn_per_cell=40), {}, 6.0, 16.0),
}


@pytest.mark.parametrize("case", sorted(CASES))
def test_save_load_continue_equals_straight_run(cn, case, monkeypatch):
    from oracle import OracleModel
    make, env, t1, t2 = CASES[case]
    for k, v in env.items():
        monkeypatch.setenv(k, v)
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
    exact = not case.startswith("config3") and not case.startswith("config5")
    dv = np.max(np.abs(a.get_v() - c.get_v()))
    assert dv == 0.0 if exact else dv < 1e-9, dv    # (several events per synapse and step: summation order)
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
