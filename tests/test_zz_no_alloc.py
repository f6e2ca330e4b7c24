"""cn_get_state_noalloc (include/cn.h): the variant of cn_get_state whose gather scratch is a static
device array of the library instead of a cudaMalloc'ed buffer -- for callers that cannot allocate
(CUDA graph capture, serving loops).  Its output must equal the existing path's on consecutive
calls (the array is shared and keeps the last call's contents), sizes beyond the limit are
rejected, and the call leaves the device's free memory alone.

Collected last on purpose (the run uses pytest -x); passes alone in a fresh process and
after the other tests.
"""
import numpy as np
import pytest

import cn_workloads as W

pytestmark = pytest.mark.gpu

DT = 0.025
TOL = 1e-9   # the tolerance of the state comparisons in test_gpu_parity.py / test_checkpoint.py


@pytest.fixture(autouse=True)
def _gpu(need_gpu):
    pass


def _tables_with_states(m, desc):
    """Probe the library itself: a table has state s iff cn_get_state accepts it."""
    out = []
    for t in range(len(desc["mechs"])):
        s = 0
        while True:
            try:
                m.get_state(t, s)
            except Exception:
                break
            s += 1
        if s:
            out.append((t, s))
    return out


@pytest.mark.parametrize("layout", ["tape", "coop", "cell"])
def test_noalloc_equals_existing_path_on_consecutive_calls(cn, layout):
    import torch
    # HH on every node + one ExpSyn per cell: 64 cells x 61 nodes (interleaved: states on tapes;
    # warp-cooperative / on-chip: states in the table arrays)
    desc = W.config2(n_cell=64, ring_size=32, depth=2, ncomp_branch=10, weight=0.05)
    options = {"tape": {"tape": 1}, "coop": {"tape": 0, "onchip": 0}, "cell": {"tape": 0, "onchip": 1}}[layout]
    m = cn.Model(desc, options=options)
    m.run(5.0, DT)
    tables = _tables_with_states(m, desc)
    assert len(tables) >= 2 and sum(ns for _, ns in tables) >= 4
    ref = {(t, s): m.get_state(t, s) for t, ns in tables for s in range(ns)}   # existing path (warmed up)
    # (one call first: with lazy module loading the driver loads a kernel at its first launch)
    m.get_state_noalloc(tables[0][0], 0)
    free0 = torch.cuda.mem_get_info()[0]
    # calls in a row, a large table then a small one then the large one again: stale contents of
    # the shared array from the previous call must not show
    order = [(t, s) for t, ns in tables for s in range(ns)]
    order = order + order[::-1]
    for t, s in order:
        got = m.get_state_noalloc(t, s)
        assert got.shape == ref[(t, s)].shape
        assert np.max(np.abs(got - ref[(t, s)])) <= TOL, (t, s)
        assert np.array_equal(got, ref[(t, s)]), (t, s)      # (a gather: in fact the same bits)
    assert torch.cuda.mem_get_info()[0] == free0             # nothing was allocated on the device
    # the states move on: the second round of calls follows the model, not the array's old contents
    m.run(10.0, DT)
    for t, s in order[:3]:
        a, b = m.get_state_noalloc(t, s), m.get_state(t, s)
        assert np.array_equal(a, b), (t, s)
    assert any(not np.array_equal(m.get_state_noalloc(t, s), ref[(t, s)]) for t, s in order[:3])
    m.destroy()


def test_noalloc_two_models_share_the_array(cn):
    a = cn.Model(W.config1())
    b = cn.Model(W.config2(n_cell=8, ring_size=4, weight=0.05))
    a.run(3.0, DT)
    b.run(3.0, DT)
    for _ in range(2):
        for m, desc in ((a, W.config1()), (b, W.config2(n_cell=8, ring_size=4, weight=0.05))):
            for t, ns in _tables_with_states(m, desc):
                for s in range(ns):
                    assert np.array_equal(m.get_state_noalloc(t, s), m.get_state(t, s)), (t, s)
    a.destroy()
    b.destroy()


def test_noalloc_rejects_sizes_beyond_the_limit(cn):
    desc = W.config2(n_cell=128, ring_size=64)       # HH on 76,928 compartments > 65,536
    m = cn.Model(desc)
    m.run(1.0, DT)
    with_states = {t for t, _ in _tables_with_states(m, desc)}
    big = [t for t, n in enumerate(m.mech_n) if n > cn.NOALLOC_MAX_INSTANCES and t in with_states]
    assert big
    t = big[0]
    out = np.full(m.mech_n[t], 7.0)
    with pytest.raises(cn.CnError) as ei:
        m.get_state_noalloc(t, 0, out=out)
    assert ei.value.code == -9 and "static scratch holds 65536" in str(ei.value)
    assert np.all(out == 7.0)                         # nothing written
    assert m.get_state(t, 0).shape == (m.mech_n[t],)  # the allocating path still serves it
    # wrong size / before the first run: the same errors as cn_get_state
    with pytest.raises(cn.CnError):
        m.get_state_noalloc(t, 0, out=np.empty(3))
    m.destroy()
    m2 = cn.Model(W.config1())
    with pytest.raises(cn.CnError):
        m2.get_state_noalloc(0, 0)
    m2.destroy()
