#!/usr/bin/env python
"""Writes tests/golden/config3_100ms.npz: the ORACLE's results for config 3 at its full size
(3,560 cells, 465,740 compartments, 1,100,040 Exp2Syn) and full length (100 ms = 4,000 dt).

The oracle needs several minutes for this run (4.4e9 synapse-steps with two libm exp each), more
than the GPU suite may spend, so its results are stored.  This script calls only oracle/ and the
seeded input generators (cn_workloads); nothing here comes from the CUDA path.  The file carries
the SHA-256 of the generated description and of the oracle's source: the test that uses it
(tests/test_gpu_full_size.py) refuses a file that does not match the current generator / oracle,
and re-runs the oracle for the first 10 ms to tie the stored spike list to the live oracle.

    python tests/golden/make_config3_golden.py
"""
import hashlib
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent.parent
sys.path.insert(0, str(ROOT))
OUT = Path(__file__).resolve().parent / "config3_100ms.npz"
DT, TSTOP = 0.025, 100.0
N_TRACE_CELLS = 64          # soma voltage of these cells at every step
TRACE_EVERY = 100           # soma voltage of every cell at every 100th step


def oracle_sha():
    h = hashlib.sha256()
    for f in ("cn_oracle.c", "cn_oracle.h"):
        h.update((ROOT / "oracle" / f).read_bytes())
    return h.hexdigest()


def trace_cells(n_cell):
    return np.linspace(0, n_cell - 1, N_TRACE_CELLS).astype(np.int64)


def main():
    import cn_workloads as W
    from oracle import OracleModel
    desc = W.config3()
    roots = np.asarray(desc["cell_first"][:-1], np.int32)
    o = OracleModel(desc)
    o.set_probes(roots)
    t0 = time.time()
    o.run(TSTOP, DT)
    print("oracle: %.0f s" % (time.time() - t0))
    tr = o.get_trace()
    gid, step = o.get_spikes()
    states = {}
    for t, m in enumerate(desc["mechs"]):
        ns = {"hh": 3, "hhform": 2, "sk": 1}.get(m["type"], 0)
        for s in range(ns):
            states["state_%d_%d" % (t, s)] = o.get_state(t, s)
    syn = o.get_state(5, 1)
    np.savez_compressed(
        OUT, desc_sha256=W.desc_hash(desc), oracle_sha256=oracle_sha(), dt=DT, tstop=TSTOP,
        spike_gid=gid, spike_step=step, min_margin=o.min_margin, v_final=o.get_v(),
        trace_cells=trace_cells(len(roots)), trace_dense=tr[:, trace_cells(len(roots))],
        trace_sparse=tr[TRACE_EVERY - 1::TRACE_EVERY], cai_final=o.get_cai(),
        exp2syn_B_sum=float(np.sum(syn)), exp2syn_B_sample=syn[::97], **states)
    print("wrote", OUT, OUT.stat().st_size, "bytes;", len(gid), "spikes")


if __name__ == "__main__":
    main()
