"""Host-side checks of the C ABI (no GPU): the library loads, exports every symbol include/cn.h
declares, validates descriptions at create time, and refuses to compute without a device."""
import re
from pathlib import Path

import numpy as np
import pytest

import cn_workloads as W
import paper_1901_10975_b200 as cn

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module", autouse=True)
def built():
    from paper_1901_10975_b200.build import build
    build()


def test_exports_every_declared_symbol():
    hdr = (ROOT / "include" / "cn.h").read_text()
    declared = set(re.findall(r"\b(cn_[a-z_0-9]+)\s*\(", hdr))
    assert {"cn_model_create", "cn_run", "cn_get_v", "cn_get_spikes"} <= declared
    L = cn.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(cn.EXPORTS)
    # ... and nothing else: every cn_* symbol the shared library exports is declared in the header
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", str(ROOT / "paper_1901_10975_b200" / "libcn.so")],
                         capture_output=True, text=True, check=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if ln.split() and ln.split()[-2] in "TW"}
    exported = {x for x in exported if re.fullmatch(r"cn_[a-z_0-9]+", x)}
    assert exported == declared, exported ^ declared


def test_options_are_per_model_and_validated(monkeypatch):
    """cn_model_create_opts: the only knobs; unknown keys and malformed pairs are rejected, the
    environment is not consulted."""
    d = W.config4(n_cell=64, n_types=2)
    assert cn.Model(d, options={"tape": 1}).layout_info()["n_tape_group"] == 2
    assert cn.Model(d, options="tape=0; force_g=4").layout_info()["n_tape_group"] == 0
    assert cn.Model(d, options="tape=1,tape_w=4").layout_info()["tape_warps"] == 4
    before = cn.Model(d).layout_info()
    monkeypatch.setenv("CN_TAPE", "0")          # ambient state steers nothing
    monkeypatch.setenv("CN_TAPE_W", "4")
    info = cn.Model(d).layout_info()
    assert info == before and info["tape_warps"] == 12    # (small model: 12 warps per group)
    for bad in ("bogus=1", "tape", "tape=", "tape=yes", "=1"):
        with pytest.raises(cn.CnError) as e:
            cn.Model(d, options=bad)
        assert e.value.code == -1, bad
    src = "".join(f.read_text() for f in (ROOT / "paper_1901_10975_b200" / "csrc").iterdir())
    assert "getenv" not in src


def test_null_arrays_with_nonzero_counts_are_rejected():
    """A description whose counts promise arrays that are NULL returns an error, never a crash."""
    import ctypes as C
    d, keep, _ = cn.marshal(W.config1())
    L = cn.lib()
    h = C.c_void_p()
    for field, code in (("nc_weight", -4), ("nc_src", -4), ("mech", -3), ("parent", -1)):
        saved = getattr(d, field)
        setattr(d, field, None)
        assert L.cn_model_create(C.byref(d), C.byref(h)) == code, field
        assert not h.value
        setattr(d, field, saved)
    d.n_stim = 3
    d.stim_gid = None
    assert L.cn_model_create(C.byref(d), C.byref(h)) == -4


def test_create_and_initial_v_without_device():
    m = cn.Model(W.config1())
    assert m.n_node == 488 and m.n_cell == 8
    assert np.all(m.get_v() == -65.0)
    g, s = m.get_spikes()
    assert len(g) == 0
    info = m.layout_info()
    assert info["n_class"] == 1 and info["n_group"] >= 1


def test_shape_classes_found_in_shuffled_cells():
    d = W.config4(n_cell=256, n_types=8)
    m = cn.Model(d)
    assert m.layout_info()["n_class"] == 8
    d = W.random_tree_cells(9, 10, 40, stream="abi")
    assert cn.Model(d).layout_info()["n_class"] == 9


def _expect(desc, code):
    with pytest.raises(cn.CnError) as e:
        cn.Model(desc)
    assert e.value.code == code


def test_validation_errors():
    base = W.config1()
    d = dict(base); d["parent"] = base["parent"].copy(); d["parent"][5] = 9
    _expect(d, -2)
    d = dict(base); d["parent"] = base["parent"].copy(); d["parent"][62] = 3
    _expect(d, -2)
    d = dict(base); d["parent"] = base["parent"].copy(); d["parent"][61] = 60
    _expect(d, -2)
    d = dict(base); d["area"] = base["area"].copy(); d["area"][7] = 0.0
    _expect(d, -1)
    d = dict(base); d["cm"] = base["cm"].copy(); d["cm"][7] = np.nan
    _expect(d, -1)
    d = dict(base); d["ri"] = base["ri"].copy(); d["ri"][7] = -1.0
    _expect(d, -1)
    d = dict(base); d["mechs"] = [dict(m) for m in base["mechs"]]
    d["mechs"][0] = dict(d["mechs"][0]); d["mechs"][0]["node"] = np.array([10 ** 6] * 8, np.int32)
    _expect(d, -3)
    d = dict(base); d["netcons"] = dict(base["netcons"])
    d["netcons"]["tgt_inst"] = base["netcons"]["tgt_inst"].copy(); d["netcons"]["tgt_inst"][0] = 99
    _expect(d, -4)
    d = dict(base); d["netcons"] = dict(base["netcons"])
    d["netcons"]["tgt_mech"] = base["netcons"]["tgt_mech"].copy(); d["netcons"]["tgt_mech"][0] = 1
    _expect(d, -4)          # pas receives no events
    d = dict(base); d["netcons"] = dict(base["netcons"])
    d["netcons"]["delay"] = base["netcons"]["delay"].copy(); d["netcons"]["delay"][0] = -1.0
    _expect(d, -4)
    # two instances of one distributed table on one node
    d = dict(base); d["mechs"] = list(base["mechs"])
    pas = dict(d["mechs"][1]); pas["node"] = pas["node"].copy(); pas["node"][1] = pas["node"][0]
    d["mechs"][1] = pas
    _expect(d, -3)
    # an HH-form gate with a zero slope constant (its rate functions divide by it)
    import cn_workloads.networks as NW
    for key in ("m_k", "h_s"):
        g = NW.hhform_globals("CaHVA"); g[key] = 0.0
        d = dict(base)
        d["mechs"] = list(base["mechs"]) + [
            {"type": "hhform", "node": np.array([3], np.int32), "params": {"gbar": np.array([1e-4])},
             "globals": g}]
        _expect(d, -3)
    # gap junction without a peer node
    for bad in (488.0, -1.0, 2.5):
        d = dict(base)
        d["mechs"] = list(base["mechs"]) + [
            {"type": "gap", "node": np.array([3], np.int32),
             "params": {"g": np.array([0.01]), "peer": np.array([bad])}, "globals": {}}]
        _expect(d, -3)


def test_validation_on_all_cores_reports_the_first_failure():
    """The validation passes run on all host cores over a model large enough to be split; the
    failure with the smallest index is the one reported, whatever thread found it."""
    base = W.config4(n_cell=2048, n_types=8)
    n = len(base["parent"])
    assert n > 8 * 65536                       # several ranges per pass
    d = dict(base); d["area"] = base["area"].copy()
    for i in (n - 5, n // 2, 70001):
        d["area"][i] = -1.0
    with pytest.raises(cn.CnError) as e:
        cn.Model(d)
    assert e.value.code == -1 and "node 70001)" in str(e.value)
    d = dict(base); d["parent"] = base["parent"].copy()
    cf = base["cell_first"]
    for c in (1900, 700):
        d["parent"][cf[c] + 4] = cf[c] + 9
    with pytest.raises(cn.CnError) as e:
        cn.Model(d)
    assert e.value.code == -2 and "cell 700" in str(e.value)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    m = cn.Model(W.config1())
    with pytest.raises(cn.CnError) as e:
        m.run(1.0, 0.025)
    assert e.value.code == -6
    with pytest.raises(cn.CnError) as e:
        m.run(1.0, -0.025)
    assert e.value.code == -5


def test_binding_never_imports_the_oracle():
    src = (ROOT / "paper_1901_10975_b200" / "__init__.py").read_text()
    assert "import oracle" not in src and "from oracle" not in src
    for f in (ROOT / "paper_1901_10975_b200" / "csrc").iterdir():
        assert "oracle" not in f.read_text().lower().replace("no cpu", "")
