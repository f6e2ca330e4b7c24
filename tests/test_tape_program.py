"""The host-side compiler of the interleaved kernel (cn_model_create needs no GPU).

`build_tape_program` cuts every cell shape into W record lists and then dry-runs them with the
kernel's wait / signal / hand-over rules (every node eliminated after its children, every
contribution stored or added exactly once and in order, back-substitution parents first, no
deadlock); cn_model_create fails with CN_ERR_TOPOLOGY if that check trips.  Here the compiler is
driven over many tree shapes, warp counts and ring geometries on the CPU.
"""
import numpy as np
import pytest

import cn_workloads as W


def _model(cn, desc, **options):
    m = cn.Model(desc, options=dict({"tape": 1, "tape_min_group": 1}, **options))
    info = m.layout_info()
    m.destroy()
    return info


@pytest.mark.parametrize("warps", [1, 2, 3, 5, 8, 16])
def test_compiles_for_every_warp_count(cn, warps):
    desc = W.config4(n_cell=128, n_types=4)
    info = _model(cn, desc, tape_w=warps, tape_ch=10 if warps > 8 else 15)
    assert info["n_class"] == 4 and info["n_tape_group"] == 4 and info["tape_warps"] == warps


@pytest.mark.parametrize("s,ch", [(2, 9), (2, 15), (3, 10), (4, 9), (2, 40)])
def test_ring_geometries(cn, s, ch):
    desc = W.config4(n_cell=64, n_types=2)
    info = _model(cn, desc, tape_s=s, tape_ch=ch, tape_w=8)
    assert info["n_tape_group"] == 2


def test_random_trees_of_every_size(cn):
    # 40 unique topologies from single nodes to 300 nodes, up to 3 children per node
    desc = W.random_tree_cells(40, 1, 300, stream="prog-a", weight=0.2, amp=2.0)
    info = _model(cn, desc)
    assert info["n_class"] == 40 and info["n_tape_group"] == 40


def test_mechanism_heavy_shapes(cn):
    # every node with HH (all system rows in shared memory), and config 3's four tables per node
    info = _model(cn, W.config2(n_cell=32, ring_size=32, depth=2, ncomp_branch=10))
    assert info["n_tape_group"] == 1 and info["tape_sys_rows"] == 61      # no private rows at all
    info = _model(cn, W.config3(n_cell=28, syn_per_cell=20))
    assert info["n_class"] == 14 and info["n_tape_group"] == 14


def test_shapes_that_do_not_fit_fall_back(cn):
    # config 2's 601-node cells with a mechanism on every node: 601 shared-memory rows > 227 KB
    info = _model(cn, W.config2(n_cell=8, ring_size=4))
    assert info["n_tape_group"] == 0 and info["n_group"] > 0
    # config 5's 30-row mechanism records and 330..580-node cells
    info = _model(cn, W.config5(n_cell=55, syn_per_cell=8))
    assert info["n_tape_group"] == 0


def test_auto_strategy_for_small_models(cn):
    """Default strategy below 8,192 cells: a model whose cells are all resident on chip at once goes
    to the on-chip window kernel (warp-cooperative layout, one cell per CTA); a larger one to the
    interleaved kernel if all of it fits there; else the warp-cooperative kernel."""
    for desc, on_tape in ((W.config1(), False), (W.config3(n_cell=140, syn_per_cell=20), False),
                          (W.config2(n_cell=8, ring_size=4), False),
                          (W.random_tree_cells(13, 5, 120, stream="gpu-u"), False),
                          (W.config3(syn_per_cell=2), True),
                          (W.config5(n_cell=3000, syn_per_cell=2), False)):
        m = cn.Model(desc)
        info = m.layout_info()
        m.destroy()
        assert (info["n_tape_group"] == info["n_group"]) == on_tape, info
        assert on_tape or info["n_tape_group"] == 0
    # the explicit options still decide
    m = cn.Model(W.config1(), options={"onchip": 0})
    assert m.layout_info()["n_tape_group"] == m.layout_info()["n_group"] == 1
