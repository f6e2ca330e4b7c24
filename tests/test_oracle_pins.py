"""Pins P1..P16: the CPU oracle against what the paper and the mathematics fix.

Nothing here touches the CUDA path.  Every expected value is a closed form, an independent
library routine (scipy banded / numpy dense LU), an independent integrator (RK4) written in this
file, an invariant, or the paper's printed workload size (tests/golden/).
"""
import math
from pathlib import Path

import numpy as np
import pytest
import scipy.linalg

import cn_workloads as W
import oracle
from oracle import OracleModel

DT = 0.025


# ---------------------------------------------------------------------------------------------
# P1: single passive compartment, closed-form backward-Euler decay (Eq. 1 with d2v/dx2 = 0)
# ---------------------------------------------------------------------------------------------

def _passive(v0, e=-65.0, g=0.001, cm=1.0):
    return W.single_compartment([("pas", {"g": g, "e": e}, {})], v_init=v0, cm=cm)


def test_p1_passive_decay_closed_form():
    v0, e, g, cm = -50.0, -65.0, 0.001, 1.0
    tau = 1e-3 * cm / g  # ms (= 1 ms)
    m = OracleModel(_passive(v0, e, g, cm))
    m.set_probes([0])
    m.run(5.0, DT)
    tr = m.get_trace()[:, 0]
    n = np.arange(1, len(tr) + 1)
    exact_be = e + (v0 - e) * (1.0 + DT / tau) ** (-n)
    assert np.max(np.abs(tr - exact_be)) < 1e-12
    # first-order bound against the continuous exponential, error halves with dt
    cont = e + (v0 - e) * np.exp(-n * DT / tau)
    err = np.max(np.abs(tr - cont))
    assert err < 1.05 * (DT / (2 * tau)) * math.exp(-1) * abs(v0 - e)
    m2 = OracleModel(_passive(v0, e, g, cm))
    m2.set_probes([0])
    m2.run(5.0, DT / 2)
    tr2 = m2.get_trace()[1::2, 0]
    err2 = np.max(np.abs(tr2 - cont))
    assert 1.8 < err / err2 < 2.2


# ---------------------------------------------------------------------------------------------
# P2: chain == Thomas / banded solve (library routine)
# ---------------------------------------------------------------------------------------------

def test_p2_chain_equals_banded_solve():
    n = 257
    u = W.rng.uniform("p2", 4 * n)
    a = -(0.05 + u[:n])
    b = -(0.05 + u[n:2 * n])
    a[0] = b[0] = 0.0
    d = 2.5 + u[2 * n:3 * n]
    rhs = u[3 * n:] - 0.5
    parent = np.arange(-1, n - 1)
    x = oracle.hines(parent, a, b, d, rhs)
    ab = np.zeros((3, n))
    ab[0, 1:] = a[1:]      # super-diagonal M[i-1, i] = a[i]
    ab[1, :] = d
    ab[2, :-1] = b[1:]     # sub-diagonal   M[i, i-1] = b[i]
    ref = scipy.linalg.solve_banded((1, 1), ab, rhs)
    assert np.max(np.abs(x - ref) / np.maximum(np.abs(ref), 1e-300)) < 1e-12


# ---------------------------------------------------------------------------------------------
# P3: random trees == dense LU; assembled model system == independent absolute-unit formulation
# ---------------------------------------------------------------------------------------------

def _dense(parent, a, b, d):
    n = len(parent)
    M = np.diag(np.asarray(d, dtype=float))
    for i in range(n):
        p = parent[i]
        if p >= 0:
            M[i, p] = b[i]
            M[p, i] = a[i]
    return M


@pytest.mark.parametrize("seed", range(12))
def test_p3_random_tree_equals_dense_lu(seed):
    n = 2 + seed * 18 // 11  # 2 .. 20
    parent = W.random_tree_parent(n, ("p3", seed))
    u = W.rng.uniform(("p3u", seed), 4 * n)
    a = -(0.1 + u[:n])
    b = -(0.1 + u[n:2 * n])
    d = 4.0 + 3 * u[2 * n:3 * n]
    rhs = u[3 * n:] - 0.5
    x = oracle.hines(parent, a, b, d, rhs)
    ref = np.linalg.solve(_dense(parent, a, b, d), rhs)
    assert np.max(np.abs(x - ref)) < 1e-12 * max(1.0, np.max(np.abs(ref)))


def test_p3_hines_is_not_symmetric_in_a_b():
    # a transposed operand (a <-> b) must be caught: area-asymmetric off-diagonals
    parent = np.array([-1, 0, 0, 1])
    a = np.array([0.0, -0.3, -0.9, -0.2])
    b = np.array([0.0, -1.1, -0.4, -0.7])
    d = np.array([3.0, 4.0, 5.0, 6.0])
    rhs = np.array([1.0, -2.0, 0.5, 0.25])
    x = oracle.hines(parent, a, b, d, rhs)
    ref = np.linalg.solve(_dense(parent, a, b, d), rhs)
    wrong = np.linalg.solve(_dense(parent, b, a, d), rhs)
    assert np.max(np.abs(x - ref)) < 1e-13
    assert np.max(np.abs(x - wrong)) > 1e-3


def test_p3_model_step_equals_absolute_unit_dense_solve():
    """One full step of a branched passive+stimulated cell against an independent formulation in
    absolute units (nA, uS, nF): (C/dt + G_m) dv_i + sum_j G_ij (dv_i - dv_j) = -I_i + sum_j
    G_ij (v_j - v_i).  Pins the unit factors of R1 (1e-3 cm/dt, 100/area) and the axial terms."""
    desc = W.random_tree_cells(1, 17, 17, stream="p3m", with_ring=False)
    # passive membrane everywhere incl. the soma, plus a current clamp; drop the HH table
    N = len(desc["parent"])
    g = W.rng.uniform("p3g", N, 5e-4, 2e-3)
    e = W.rng.uniform("p3e", N, -80.0, -50.0)
    desc["mechs"] = [
        {"type": "pas", "node": np.arange(N, dtype=np.int32), "params": {"g": g, "e": e},
         "globals": {}},
        {"type": "iclamp", "node": np.array([3], np.int32),
         "params": {"del": np.array([0.0]), "dur": np.array([1.0]), "amp": np.array([0.2])},
         "globals": {}},
    ]
    desc["netcons"] = {k: v[:0] for k, v in desc["netcons"].items()}
    m = OracleModel(desc)
    v0 = m.get_v()
    m.run(DT, DT)
    v1 = m.get_v()
    area, ri, cm, parent = desc["area"], desc["ri"], desc["cm"], desc["parent"]
    C = cm * area * 1e-5               # nF
    Gm = g * area * 1e-2               # uS
    A = np.diag(C / DT + Gm)
    r = -Gm * (v0 - e)                 # nA (v0 is uniform, so axial rhs terms vanish here)
    r[3] += 0.2
    for i in range(N):
        p = parent[i]
        if p >= 0:
            G = 1.0 / ri[i]
            A[i, i] += G
            A[p, p] += G
            A[i, p] -= G
            A[p, i] -= G
    dv = np.linalg.solve(A, r)
    assert np.max(np.abs((v1 - v0) - dv)) < 1e-12
    # second step: non-uniform v exercises the axial rhs terms (O4)
    m.run(2 * DT, DT)
    v2 = m.get_v()
    r = -Gm * (v1 - e)
    r[3] += 0.2
    for i in range(N):
        p = parent[i]
        if p >= 0:
            G = 1.0 / ri[i]
            r[i] += G * (v1[p] - v1[i])
            r[p] += G * (v1[i] - v1[p])
    dv = np.linalg.solve(A, r)
    assert np.max(np.abs((v2 - v1) - dv)) < 1e-11
    # residual of the oracle's own assembled system
    d, rhs, sol = m.get_last_system()
    a, b = m.get_ab()
    res = _dense(parent, a, b, d) @ sol - rhs
    assert np.max(np.abs(res)) <= 1e-12 * np.max(np.abs(rhs))


def test_p3_residual_large_tree():
    desc = W.config1()
    m = OracleModel(desc)
    m.run(3.0, DT)  # during the stimulus aftermath: v is non-uniform
    d, rhs, sol = m.get_last_system()
    a, b = m.get_ab()
    parent = desc["parent"]
    res = d * sol - rhs
    for i in range(len(parent)):
        p = parent[i]
        if p >= 0:
            res[i] += b[i] * sol[p]
            res[p] += a[i] * sol[i]
    assert np.max(np.abs(res)) <= 1e-12 * np.max(np.abs(rhs))


# ---------------------------------------------------------------------------------------------
# P4: unit factors and axial terms
# ---------------------------------------------------------------------------------------------

def test_p4_eq1_identity_and_area_symmetry():
    desc = W.config1()
    m = OracleModel(desc)
    a, b = m.get_ab()
    # Eq. 1: d/(4 Ra dx^2) with d = 1 um, Ra = 100 Ohm cm, dx = 20 um -> 0.0625 S/cm2
    expect = 1e-4 / (4 * 100.0 * (20e-4) ** 2)
    assert abs(expect - 0.0625) < 1e-15
    assert abs(-b[5] - 0.0625) < 1e-14 and abs(-a[5] - 0.0625) < 1e-14
    # soma-dendrite link
    assert abs(-b[1] - 0.124688279301745) < 1e-12
    assert abs(-a[1] - 0.00623441396508728) < 1e-13
    parent, area = desc["parent"], desc["area"]
    nz = parent >= 0
    assert np.allclose(a[nz] * area[parent[nz]], b[nz] * area[nz], rtol=1e-14, atol=0)


def test_p4_charge_conservation():
    desc = W.random_tree_cells(1, 40, 40, stream="p4c", with_ring=False)
    desc["mechs"] = [{"type": "iclamp", "node": np.array([7], np.int32),
                      "params": {"del": np.array([0.5]), "dur": np.array([1.0]),
                                 "amp": np.array([0.05])}, "globals": {}}]
    desc["netcons"] = {k: v[:0] for k, v in desc["netcons"].items()}
    C = desc["cm"] * desc["area"] * 1e-5  # nF
    m = OracleModel(desc)
    m.run(0.5, DT)
    assert np.all(m.get_v() == -65.0)
    m.run(2.0, DT)
    q = np.sum(C * (m.get_v() + 65.0))       # pC
    assert abs(q - 0.05 * 1.0) < 1e-12       # nA * ms
    m.run(4.0, DT)
    assert abs(np.sum(C * (m.get_v() + 65.0)) - 0.05) < 1e-12
    m.run(2000.0, 0.025)
    v = m.get_v()
    assert np.max(v) - np.min(v) < 1e-9      # relaxes to the capacitance-weighted mean
    assert abs(v[0] - (-65.0 + 0.05 / np.sum(C))) < 1e-9


def test_p4_cable_steady_state_cosh():
    n, diam, L, Ra, g, e, amp = 40, 1.0, 400.0, 100.0, 0.001, -65.0, 0.01
    desc = W.cable(n, diam=diam, L=L, Ra=Ra, g_pas=g, e_pas=e)
    desc["mechs"].append({"type": "iclamp", "node": np.array([0], np.int32),
                          "params": {"del": np.array([0.0]), "dur": np.array([1e9]),
                                     "amp": np.array([amp])}, "globals": {}})
    m = OracleModel(desc)
    m.run(60.0, DT)
    v = m.get_v()
    dx = L / n
    Gax = 1.0 / (1e-2 * Ra * dx / (math.pi * diam * diam / 4))   # uS between neighbours
    gm = g * math.pi * diam * dx * 1e-2                          # uS per compartment
    kappa = math.acosh(1.0 + gm / (2 * Gax))
    i = np.arange(n)
    shape = np.cosh(kappa * (n - 0.5 - i))
    A = amp / (gm * shape[0] - Gax * (shape[1] - shape[0]))
    assert np.max(np.abs(v - (e + A * shape))) < 1e-10


# ---------------------------------------------------------------------------------------------
# P5 / P6: Hodgkin-Huxley rest and spike, against independent code in this file
# ---------------------------------------------------------------------------------------------

def _hh_ab(v):
    def vtrap(x, y):
        return y * (1 - x / y / 2) if abs(x / y) < 1e-6 else x / math.expm1(x / y)
    am = 0.1 * vtrap(-(v + 40), 10)
    bm = 4 * math.exp(-(v + 65) / 18)
    ah = 0.07 * math.exp(-(v + 65) / 20)
    bh = 1 / (1 + math.exp(-(v + 35) / 10))
    an = 0.01 * vtrap(-(v + 55), 10)
    bn = 0.125 * math.exp(-(v + 65) / 80)
    return am, bm, ah, bh, an, bn


def _hh_iss(v, p=W.HH_SQUID):
    am, bm, ah, bh, an, bn = _hh_ab(v)
    mi, hi, ni = am / (am + bm), ah / (ah + bh), an / (an + bn)
    return (p["gnabar"] * mi ** 3 * hi * (v - 50) + p["gkbar"] * ni ** 4 * (v + 77)
            + p["gl"] * (v - p["el"]))


def _hh_cell(amp=None, dur=1.0, delay=1.0):
    mechs = [("hh", dict(W.HH_SQUID), dict(W.HH_GLOBALS))]
    if amp is not None:
        mechs.append(("iclamp", {"del": delay, "dur": dur, "amp": amp}, {}))
    return W.single_compartment(mechs)


def test_p5_hh_rest_is_root_of_steady_state_current():
    lo, hi = -80.0, -50.0
    assert _hh_iss(lo) < 0 < _hh_iss(hi)
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if _hh_iss(mid) > 0:
            hi = mid
        else:
            lo = mid
    vrest = 0.5 * (lo + hi)
    assert abs(vrest + 65.0) < 0.1
    m = OracleModel(_hh_cell())
    m.run(400.0, DT)
    assert abs(m.get_v()[0] - vrest) < 1e-8
    assert len(m.get_spikes()[0]) == 0


def _rk4_hh(tstop, h, amp, area, t_on=1.0, t_off=2.0):
    p = W.HH_SQUID
    def f(y, i_inj):
        v, m_, h_, n_ = y
        am, bm, ah, bh, an, bn = _hh_ab(v)
        iion = (p["gnabar"] * m_ ** 3 * h_ * (v - 50) + p["gkbar"] * n_ ** 4 * (v + 77)
                + p["gl"] * (v - p["el"]))
        dv = (-iion + 100.0 * i_inj / area) / 1e-3   # cm = 1 uF/cm2 -> 1e-3 mA ms / (mV cm2)
        return np.array([dv, am * (1 - m_) - bm * m_, ah * (1 - h_) - bh * h_,
                         an * (1 - n_) - bn * n_])
    am, bm, ah, bh, an, bn = _hh_ab(-65.0)
    y = np.array([-65.0, am / (am + bm), ah / (ah + bh), an / (an + bn)])
    nst = int(round(tstop / h))
    out = np.empty(nst + 1)
    out[0] = y[0]
    for k in range(nst):
        t = k * h
        ii = amp if (t_on - 1e-12 <= t < t_off - 1e-12) else 0.0
        k1 = f(y, ii)
        k2 = f(y + 0.5 * h * k1, ii)
        k3 = f(y + 0.5 * h * k2, ii)
        k4 = f(y + h * k3, ii)
        y = y + (h / 6) * (k1 + 2 * k2 + 2 * k3 + k4)
        out[k + 1] = y[0]
    return out


def test_p6_hh_spike_first_order_against_rk4():
    amp, tstop, hrk = 0.5, 8.0, 1e-3
    desc = _hh_cell(amp)
    area = desc["area"][0]
    ref = _rk4_hh(tstop, hrk, amp, area)
    errs = []
    for dt in (0.025, 0.0125, 0.00625):
        m = OracleModel(_hh_cell(amp))
        m.set_probes([0])
        m.run(tstop, dt)
        tr = m.get_trace()[:, 0]
        stride = int(round(dt / hrk * 1000)) / 1000.0
        idx = np.rint(np.arange(1, len(tr) + 1) * dt / hrk).astype(int)
        errs.append(np.max(np.abs(tr - ref[idx])))
        if dt == 0.025:
            assert 30.0 < tr.max() < 50.0 and tr.min() < -70.0
            g, s = m.get_spikes()
            assert len(g) == 1
    assert 1.6 < errs[0] / errs[1] < 2.4
    assert 1.6 < errs[1] / errs[2] < 2.4
    assert np.max(ref) > 30.0


# ---------------------------------------------------------------------------------------------
# P7: cnexp gates under voltage clamp
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("v", [-90.0, -65.0, -40.0, -20.0, 10.0])
def test_p7_hh_gates_exact_exponential(v):
    am, bm, ah, bh, an, bn = _hh_ab(v)
    inf = [am / (am + bm), ah / (ah + bh), an / (an + bn)]
    tau = [1 / (am + bm), 1 / (ah + bh), 1 / (an + bn)]
    S = [0.3, 0.2, 0.9]
    S0 = list(S)
    for k in range(1, 60):
        S, _ = oracle.mech_state("hh", W.HH_SQUID, W.HH_GLOBALS, S, v, DT)
        for j in range(3):
            ex = inf[j] + (S0[j] - inf[j]) * math.exp(-k * DT / tau[j])
            assert abs(S[j] - ex) < 1e-13
    r = oracle.hh_rates(v)
    assert np.allclose(r, [inf[0], tau[0], inf[1], tau[1], inf[2], tau[2]], rtol=1e-13)


def test_p7_hh_vtrap_singularity_and_q10():
    # alpha_m at v = -40 and alpha_n at v = -55 are removable singularities with limits 1 and 0.1
    for v0, lim_idx in ((-40.0, 0), (-55.0, 4)):
        r0 = oracle.hh_rates(v0)
        rp = oracle.hh_rates(v0 + 1e-4)
        rm = oracle.hh_rates(v0 - 1e-4)
        assert abs(r0[lim_idx] - 0.5 * (rp[lim_idx] + rm[lim_idx])) < 1e-8
    r63 = oracle.hh_rates(-50.0, 6.3)
    r163 = oracle.hh_rates(-50.0, 16.3)
    assert abs(r63[1] / r163[1] - 3.0) < 1e-12 and abs(r63[0] - r163[0]) < 1e-15


HHFORM_TABLE = {  # SURVEY 8(c) synthetic constants: p,q,E, m(vh,k,t0,t1,vt,s), h(...)
    "NaT": (3, 1, 50.0, (-38, 6, 0.02, 0.4, -38, 12), (-66, -6, 0.3, 10, -60, 12)),
    "NaP": (3, 1, 50.0, (-52, 5, 0.5, 5, -52, 15), (-49, -10, 100, 4000, -49, 15)),
    "Kv31": (1, 0, -85.0, (18.7, 9.7, 0.2, 8, -46, 44), (0, 1, 1, 0, 0, 1)),
    "Kv1": (2, 1, -85.0, (-11, 12, 1, 10, -11, 30), (-64, -11, 300, 1000, -64, 25)),
    "Ih": (1, 0, -45.0, (-90, -9, 20, 1000, -90, 20), (0, 1, 1, 0, 0, 1)),
    "CaHVA": (2, 1, 132.4579, (-27, 5, 0.5, 3, -27, 15), (-40, -8, 200, 500, -40, 20)),
    "CaLVA": (2, 1, 132.4579, (-40, 6, 5, 25, -40, 15), (-90, -6.4, 20, 70, -75, 15)),
}


def _hhform_globals(name):
    p, q, E, mg, hg = HHFORM_TABLE[name]
    G = {"p": p, "q": q, "E": E, "to_ica": 1.0 if name.startswith("Ca") else 0.0}
    for pre, gate in (("m", mg), ("h", hg)):
        for key, val in zip(("vh", "k", "t0", "t1", "vt", "s"), gate):
            G[f"{pre}_{key}"] = float(val)
    return G


@pytest.mark.parametrize("name", sorted(HHFORM_TABLE))
def test_p7_hhform_gates_and_current(name):
    p, q, E, mg, hg = HHFORM_TABLE[name]
    G = _hhform_globals(name)
    for v in (-80.0, -50.0, -10.0):
        def gate(g6):
            vh, k, t0, t1, vt, s = g6
            return (1 / (1 + math.exp((vh - v) / k)),
                    t0 + t1 / (2 * math.cosh((v - vt) / s)))
        minf, mtau = gate(mg)
        hinf, htau = gate(hg)
        S0 = [0.11, 0.77]
        S = list(S0)
        for k in range(1, 40):
            S, _ = oracle.mech_state("hhform", {"gbar": 0.01}, G, S, v, DT)
            assert abs(S[0] - (minf + (S0[0] - minf) * math.exp(-k * DT / mtau))) < 1e-13
            if q > 0:
                assert abs(S[1] - (hinf + (S0[1] - hinf) * math.exp(-k * DT / htau))) < 1e-13
            else:
                assert S[1] == S0[1]
        i, g, ica = oracle.mech_cur("hhform", {"gbar": 0.01}, G, [0.4, 0.6], v)
        gexp = 0.01 * 0.4 ** p * 0.6 ** q
        assert abs(g - gexp) < 1e-16 and abs(i - gexp * (v - E)) < 1e-14
        assert ica == (i if name.startswith("Ca") else 0.0)
        init = oracle.mech_init("hhform", {"gbar": 0.01}, G, v)
        assert abs(init[0] - minf) < 1e-15 and abs(init[1] - hinf) < 1e-15


def test_p7_sk_gate():
    G = {"E": -85.0, "Kd": 4.3e-4, "n": 4.8, "tau_z": 1.0}
    for cai in (1e-4, 4.3e-4, 2e-3):
        zinf = 1 / (1 + (4.3e-4 / cai) ** 4.8)
        S = [0.5]
        for k in range(1, 30):
            S, _ = oracle.mech_state("sk", {"gbar": 1e-3}, G, S, -60.0, DT, cai=cai)
            assert abs(S[0] - (zinf + (0.5 - zinf) * math.exp(-k * DT / 1.0))) < 1e-13
    assert abs(1 / (1 + 1.0) - 0.5) == 0  # at cai = Kd, z_inf = 1/2
    S, _ = oracle.mech_state("sk", {"gbar": 1e-3}, G, [0.5], -60.0, 1e9, cai=4.3e-4)
    assert abs(S[0] - 0.5) < 1e-15
    i, g, _ = oracle.mech_cur("sk", {"gbar": 1e-3}, G, [0.25], -60.0)
    assert abs(g - 2.5e-4) < 1e-18 and abs(i - 2.5e-4 * 25.0) < 1e-15


# ---------------------------------------------------------------------------------------------
# P8: synapse states after one event
# ---------------------------------------------------------------------------------------------

def test_p8_expsyn_exp2syn_ampanmda():
    w = 0.013
    S = oracle.mech_receive("expsyn", {"tau": 2.0, "e": 0.0}, {}, [0.0], w)
    assert S == [w]
    for k in range(1, 50):
        S, _ = oracle.mech_state("expsyn", {"tau": 2.0, "e": 0.0}, {}, S, -30.0, DT)
        assert abs(S[0] - w * math.exp(-k * DT / 2.0)) < 1e-16
    t1, t2 = 0.5, 5.0
    tp = t1 * t2 / (t2 - t1) * math.log(t2 / t1)
    f = oracle.exp2syn_factor(t1, t2)
    assert abs(f * (math.exp(-tp / t2) - math.exp(-tp / t1)) - 1.0) < 1e-14
    # t_p maximises B - A
    g = lambda t: f * (math.exp(-t / t2) - math.exp(-t / t1))
    assert g(tp) > g(tp * 1.001) and g(tp) > g(tp * 0.999)
    P = {"tau1": t1, "tau2": t2, "e": 0.0}
    S = oracle.mech_receive("exp2syn", P, {}, [0.0, 0.0], w)
    assert abs(S[0] - w * f) < 1e-17 and abs(S[1] - w * f) < 1e-17
    for k in range(1, 80):
        S, _ = oracle.mech_state("exp2syn", P, {}, S, -30.0, DT)
        assert abs(S[0] - w * f * math.exp(-k * DT / t1)) < 1e-15
        assert abs(S[1] - w * f * math.exp(-k * DT / t2)) < 1e-15
    i, gg, _ = oracle.mech_cur("exp2syn", P, {}, S, -30.0)
    assert abs(gg - (S[1] - S[0])) == 0 and abs(i - gg * (-30.0)) < 1e-18
    G = {"tau_r_A": 0.2, "tau_d_A": 1.7, "tau_r_N": 0.29, "tau_d_N": 43.0, "r_nmda": 0.71,
         "mg": 1.0, "e": 0.0}
    S = oracle.mech_receive("ampanmda", {}, G, [0.0] * 4, w)
    fA, fN = oracle.exp2syn_factor(0.2, 1.7), oracle.exp2syn_factor(0.29, 43.0)
    assert np.allclose(S, [w * fA, w * fA, w * fN, w * fN], rtol=1e-15)
    S = [0.0, 0.3, 0.0, 0.5]
    _, g0, _ = oracle.mech_cur("ampanmda", {}, G, S, 0.0)
    assert abs(g0 - (0.3 + 0.71 * 0.5 / (1 + 1.0 / 3.57))) < 1e-15
    iv, gv, _ = oracle.mech_cur("ampanmda", {}, G, S, -70.0)
    mgb = 1 / (1 + math.exp(0.062 * 70.0) / 3.57)
    assert abs(gv - (0.3 + 0.71 * 0.5 * mgb)) < 1e-15 and abs(iv - gv * -70.0) < 1e-13


# ---------------------------------------------------------------------------------------------
# P9: derivimplicit cai
# ---------------------------------------------------------------------------------------------

def test_p9_cadyn_newton_equals_closed_form():
    G = {"gamma": 0.05, "depth": 0.1, "tau_d": 80.0, "cai_min": 1e-4}
    kappa = 1e4 * 0.05 / (2 * 96485.33212 * 0.1)
    ica = -2.5e-3
    cai = 1e-4
    ref = cai
    for _ in range(400):
        _, cai = oracle.mech_state("cadyn", {}, G, [], -65.0, DT, cai=cai, ica=ica)
        ref = (ref + DT * (-kappa * ica + 1e-4 / 80.0)) / (1 + DT / 80.0)
        assert abs(cai - ref) < 1e-14 * max(1.0, abs(ref) / 1e-4) * 1e-4 + 1e-18
    star = 1e-4 - kappa * ica * 80.0
    for _ in range(200000):
        ref = (ref + DT * (-kappa * ica + 1e-4 / 80.0)) / (1 + DT / 80.0)
    assert abs(ref - star) < 1e-12
    _, c2 = oracle.mech_state("cadyn", {}, G, [], -65.0, DT, cai=star, ica=ica)
    assert abs(c2 - star) < 1e-16


# ---------------------------------------------------------------------------------------------
# P9b: model-level plumbing ica -> cai -> SK inside one_step (O2/O3/O9)
# ---------------------------------------------------------------------------------------------

def _ca_cell(order=("cadyn", "sk"), v_init=-30.0, second_source=True):
    """One compartment: pas + Ca_HVA (+ Ca_LVA) as Ca sources, cai dynamics and SK in the given
    table order, and an IClamp so that v (and with it the Ca current) changes from step to step."""
    ms = [("pas", {"g": 3e-5, "e": -75.0}, {}),
          ("hhform", {"gbar": 1e-3}, _hhform_globals("CaHVA"))]
    if second_source:
        ms.append(("hhform", {"gbar": 4e-4}, _hhform_globals("CaLVA")))
    tail = {"cadyn": ("cadyn", {}, dict(gamma=0.05, depth=0.1, tau_d=80.0, cai_min=1e-4)),
            "sk": ("sk", {"gbar": 2e-4}, dict(E=-85.0, Kd=4.3e-4, n=4.8, tau_z=1.0))}
    ms += [tail[o] for o in order]
    ms.append(("iclamp", {"del": 0.0, "dur": 10.0, "amp": 0.3}, {}))
    return W.single_compartment(ms, v_init=v_init)


def _gate_inf_tau(g6, v):
    vh, k, t0, t1, vt, s = g6
    return 1 / (1 + math.exp((vh - v) / k)), t0 + t1 / (2 * math.cosh((v - vt) / s))


def _ca_current(name, gbar, S, v):
    p, q, E, _, _ = HHFORM_TABLE[name]
    return gbar * S[0] ** p * S[1] ** q * (v - E)


def _be_cai(cai, ica, dt=DT, gamma=0.05, depth=0.1, tau_d=80.0, cai_min=1e-4):
    kappa = 1e4 * gamma / (2 * 96485.33212 * depth)
    return (cai + dt * (-kappa * ica + cai_min / tau_d)) / (1 + dt / tau_d)


def test_p9b_ica_feeds_cai_per_step_and_is_zeroed():
    """cai after step 1 is the closed-form backward-Euler update with the Ca current of step 1
    (sum over BOTH Ca channels, evaluated at the OLD v with the OLD gates, mA/cm2 -> mM through
    kappa = 1e4 gamma / (2 F depth)); after step 2 with the current of step 2 ONLY (the per-step
    zeroing of ica), evaluated with the gates advanced at the end of step 1 and v after step 1.
    The gate values used here come from the gate formulas, not from the oracle."""
    v0 = -30.0
    desc = _ca_cell(v_init=v0)
    m = OracleModel(desc)
    m.set_probes([0])
    # step 1: gates at steady state of v_init
    S = {}
    for name in ("CaHVA", "CaLVA"):
        _, _, _, mg, hg = HHFORM_TABLE[name]
        S[name] = [_gate_inf_tau(mg, v0)[0], _gate_inf_tau(hg, v0)[0]]
    ica0 = _ca_current("CaHVA", 1e-3, S["CaHVA"], v0) + _ca_current("CaLVA", 4e-4, S["CaLVA"], v0)
    assert ica0 < -1e-3                       # an inward current large enough to move cai by %
    m.run(DT, DT)
    cai1 = _be_cai(1e-4, ica0)
    assert abs(cai1 - 1e-4) > 1e-6
    assert abs(m.get_cai()[0] - cai1) < 1e-16
    # a single-source reading (accumulation "=" instead of "+=") is visibly different
    assert abs(_be_cai(1e-4, _ca_current("CaLVA", 4e-4, S["CaLVA"], v0)) - cai1) > 1e-8
    # step 2: gates were advanced by cnexp at v1 (the new v of step 1)
    v1 = m.get_trace()[0, 0]
    assert abs(v1 - v0) > 1e-3
    for name in ("CaHVA", "CaLVA"):
        _, _, _, mg, hg = HHFORM_TABLE[name]
        for j, g6 in enumerate((mg, hg)):
            inf, tau = _gate_inf_tau(g6, v1)
            S[name][j] = S[name][j] + (1 - math.exp(-DT / tau)) * (inf - S[name][j])
    ica1 = _ca_current("CaHVA", 1e-3, S["CaHVA"], v1) + _ca_current("CaLVA", 4e-4, S["CaLVA"], v1)
    m.run(2 * DT, DT)
    cai2 = _be_cai(cai1, ica1)
    assert abs(m.get_cai()[0] - cai2) < 1e-16
    # without the per-step zeroing step 2 would see ica0 + ica1
    assert abs(_be_cai(cai1, ica0 + ica1) - cai2) > 1e-7
    # the oracle's own gates agree with the formulas used above
    assert abs(m.get_state(1, 0)[0] - _advance(S["CaHVA"][0], HHFORM_TABLE["CaHVA"][3],
                                               m.get_trace()[1, 0])) < 1e-15


def _advance(x, g6, v):
    inf, tau = _gate_inf_tau(g6, v)
    return x + (1 - math.exp(-DT / tau)) * (inf - x)


def test_p9b_state_order_cadyn_before_or_after_sk():
    """O9 runs the tables in description order: with cai dynamics BEFORE SK the gate relaxes
    towards z_inf(cai after this step), with SK first towards z_inf(cai before it).  Initial
    z = z_inf(cai_min), so in the second case step 1 leaves z exactly where it was."""
    Kd, n, tau_z = 4.3e-4, 4.8, 1.0
    zinf = lambda c: 1 / (1 + (Kd / c) ** n)
    z0 = zinf(1e-4)
    a = OracleModel(_ca_cell(("cadyn", "sk")))
    b = OracleModel(_ca_cell(("sk", "cadyn")))
    a.run(DT, DT)
    b.run(DT, DT)
    cai1 = a.get_cai()[0]
    assert cai1 == b.get_cai()[0]             # cai itself does not depend on the order
    za = a.get_state(4, 0)[0]                 # tables: pas, CaHVA, CaLVA, cadyn, sk
    zb = b.get_state(3, 0)[0]                 # tables: pas, CaHVA, CaLVA, sk, cadyn
    assert abs(za - (z0 + (1 - math.exp(-DT / tau_z)) * (zinf(cai1) - z0))) < 1e-18
    assert zb == z0
    assert abs(za - zb) > 1e-3 * z0
    # SK's current reaches the voltage: a model without SK conductance ends elsewhere
    a.run(40 * DT, DT)
    c = _ca_cell(("cadyn", "sk"))
    c["mechs"][4]["params"]["gbar"] = np.zeros(1)
    cm_ = OracleModel(c)
    cm_.run(40 * DT, DT)
    assert abs(a.get_v()[0] - cm_.get_v()[0]) > 1e-9


def test_p9b_cai_fixed_point_with_a_real_channel_current():
    """Voltage-clamp-like check of the units of kappa with a real channel current: a huge membrane
    capacitance pins v, the Ca gates sit at their steady state for that v, and cai must converge to
    cai_min - kappa * ica * tau_d with ica = gbar m_inf^2 h_inf (v - E_Ca) from the formulas."""
    v0 = -25.0
    desc = _ca_cell(v_init=v0, second_source=False)
    desc["cm"] = np.array([1e12])
    desc["mechs"] = [x for x in desc["mechs"] if x["type"] not in ("iclamp", "sk")]
    m = OracleModel(desc)
    m.run(3000.0, 0.5)
    _, _, _, mg, hg = HHFORM_TABLE["CaHVA"]
    S = [_gate_inf_tau(mg, v0)[0], _gate_inf_tau(hg, v0)[0]]
    ica = _ca_current("CaHVA", 1e-3, S, v0)
    kappa = 1e4 * 0.05 / (2 * 96485.33212 * 0.1)
    star = 1e-4 - kappa * ica * 80.0
    assert abs(m.get_v()[0] - v0) < 1e-7
    assert star > 5e-3 and abs(m.get_cai()[0] - star) < 1e-8 * star


def test_p9b_sk_cai_floor():
    """z_inf floors cai at 1e-9 mM: cai = 0, 1e-12 and negative values give the
    1e-9 value, which is 1 / (1 + (Kd/1e-9)^n); just above the floor the value moves again.
    (z starts at 0 so that the tiny z_inf is not absorbed by rounding.)"""
    G = {"E": -85.0, "Kd": 4.3e-4, "n": 4.8, "tau_z": 1.0}
    ref, _ = oracle.mech_state("sk", {"gbar": 1e-3}, G, [0.0], -60.0, DT, cai=1e-9)
    for cai in (0.0, 1e-12, -1e-5):
        S, _ = oracle.mech_state("sk", {"gbar": 1e-3}, G, [0.0], -60.0, DT, cai=cai)
        assert S[0] == ref[0]
    zinf = 1 / (1 + (4.3e-4 / 1e-9) ** 4.8)
    assert ref[0] > 0 and abs(ref[0] / ((1 - math.exp(-DT)) * zinf) - 1) < 1e-13
    above, _ = oracle.mech_state("sk", {"gbar": 1e-3}, G, [0.0], -60.0, DT, cai=2e-9)
    assert abs(above[0] / ref[0] - 2 ** 4.8) < 1e-9 * 2 ** 4.8


# ---------------------------------------------------------------------------------------------
# P10: event and clamp timing on the integer step grid (R4, R10)
# ---------------------------------------------------------------------------------------------

def _syn_target(delays, ks_time):
    n = len(delays)
    desc = W.single_compartment([("pas", {"g": 0.001, "e": -65.0}, {})])
    desc["mechs"].append({"type": "expsyn", "node": np.zeros(n, np.int32),
                          "params": {"tau": np.full(n, 2.0), "e": np.zeros(n)}, "globals": {}})
    desc["netcons"] = {"src": np.full(n, 1, np.int32), "tgt_mech": np.full(n, 1, np.int32),
                       "tgt_inst": np.arange(n, dtype=np.int64),
                       "weight": np.full(n, 0.01), "delay": np.asarray(delays, float)}
    desc["stim"] = {"gid": np.array([1], np.int32), "t": np.array([ks_time])}
    return desc


@pytest.mark.parametrize("ks", [0, 7])
def test_p10_delivery_step_exact(ks):
    dsteps = [1, 40, 400]
    m = OracleModel(_syn_target([d * DT for d in dsteps], ks * DT))
    for j, d in enumerate(dsteps):
        kd = ks + d
        m.run(kd * DT, DT)           # steps 0 .. kd-1 done: not yet delivered
        assert m.steps_done == kd
        assert m.get_state(1, 0)[j] == 0.0
        m.run((kd + 1) * DT, DT)     # step kd: delivered in O1, decayed once in O9
        assert abs(m.get_state(1, 0)[j] - 0.01 * math.exp(-DT / 2.0)) < 1e-17


def test_p10_delay_below_one_step_rejected():
    m = OracleModel(_syn_target([0.4 * DT], 0.0))
    with pytest.raises(ValueError):
        m.run(1.0, DT)


def test_p10_iclamp_active_steps_40_to_79():
    desc = W.single_compartment([("iclamp", {"del": 1.0, "dur": 1.0, "amp": 0.5}, {})])
    m = OracleModel(desc)
    m.set_probes([0])
    m.run(3.0, DT)
    tr = np.concatenate([[-65.0], m.get_trace()[:, 0]])
    dv = np.diff(tr)                       # dv[k] = change made by step k
    active = np.nonzero(dv != 0.0)[0]
    assert active[0] == 40 and active[-1] == 79 and len(active) == 40
    inc = 100.0 * 0.5 / desc["area"][0] / (1e-3 * 1.0 / DT)
    assert np.allclose(dv[40:80], inc, rtol=1e-12)


# ---------------------------------------------------------------------------------------------
# P10b: gap junctions (L160, L228): explicit peer voltage, exchanged once per step
# ---------------------------------------------------------------------------------------------

def _gap_cells(g, pairs, n_cell=3, amp=0.5, cm=1.0, decoy_e=0.0):
    """n_cell one-compartment cells without membrane conductance (pure capacitors), cell 1 a
    decoy with a leak to decoy_e; `pairs` = (node, peer) list of gap junctions; cell 0 gets a
    current pulse on steps 40..79."""
    area = math.pi * 20.0 * 20.0
    N = n_cell
    nd = np.array([p[0] for p in pairs], np.int32)
    pr = np.array([p[1] for p in pairs], np.float64)
    return {
        "cell_first": np.arange(N + 1, dtype=np.int64), "parent": np.full(N, -1, np.int32),
        "area": np.full(N, area), "ri": np.ones(N), "cm": np.full(N, cm), "v_init": -65.0,
        "celsius": 6.3,
        "mechs": [
            {"type": "pas", "node": np.array([1], np.int32),
             "params": {"g": np.array([0.001]), "e": np.array([decoy_e])}, "globals": {}},
            {"type": "iclamp", "node": np.array([0], np.int32),
             "params": {"del": np.array([1.0]), "dur": np.array([1.0]), "amp": np.array([amp])},
             "globals": {}},
            {"type": "gap", "node": nd, "params": {"g": np.full(len(pairs), g), "peer": pr},
             "globals": {}}],
        "netcons": {"src": np.zeros(0, np.int32), "tgt_mech": np.zeros(0, np.int32),
                    "tgt_inst": np.zeros(0, np.int64), "weight": np.zeros(0),
                    "delay": np.zeros(0)},
        "thr": np.full(N, 1e9), "stim": {"gid": np.zeros(0, np.int32), "t": np.zeros(0)}}, area


def test_p10b_gap_pair_closed_form():
    g, amp = 0.004, 0.5
    desc, area = _gap_cells(g, [(0, 2), (2, 0)])
    m = OracleModel(desc)
    m.set_probes([0, 1, 2])
    m.run(6.0, DT)
    tr = np.vstack([[-65.0] * 3, m.get_trace()])
    c = 1e-3 / DT
    gs = 100.0 * g / area
    v0, v2 = tr[:, 0], tr[:, 2]
    ssum, d = v0 + v2, v0 - v2
    # the pair exchanges charge only: the sum moves only while the electrode is on (steps 40..79),
    # by Is / (c + gs) per step (the junction conductance sits on the diagonal of both rows)
    inc = np.diff(ssum)
    assert np.max(np.abs(inc[:40])) == 0.0 and np.max(np.abs(inc[80:])) < 1e-12
    assert np.allclose(inc[40:80], (100.0 * amp / area) / (c + gs), rtol=1e-11)
    # after the pulse the difference decays by (c - gs)/(c + gs) per step: the peer voltage is the
    # one of the START of the step (an implicit peer would give c/(c + 2 gs))
    r = d[81:] / d[80:-1]
    assert abs(d[80]) > 1.0
    assert np.allclose(r, (c - gs) / (c + gs), rtol=1e-10)
    assert not np.allclose(r, c / (c + 2 * gs), rtol=1e-4)
    # the decoy (same start voltage, leak to 0 mV) is neither read nor written by the junctions
    alone, _ = _gap_cells(g, [])
    ma = OracleModel(alone)
    ma.set_probes([1])
    ma.run(6.0, DT)
    assert np.array_equal(ma.get_trace()[:, 0], tr[1:, 1])
    assert abs(tr[-1, 1] - tr[-1, 2]) > 5.0


def test_p10b_gap_difference_mode_converges_to_continuous_decay():
    g = 0.002
    errs = []
    for dt in (DT, DT / 2):
        desc, area = _gap_cells(g, [(0, 2), (2, 0)])
        m = OracleModel(desc)
        m.set_probes([0, 2])
        m.run(8.0, dt)
        tr = m.get_trace()
        k0 = int(round(2.0 / dt)) + 1            # first row after the pulse
        d = tr[k0:, 0] - tr[k0:, 1]
        t = np.arange(len(d)) * dt
        cont = d[0] * np.exp(-2.0 * (100.0 * g / area) * t / 1e-3)   # C dv/dt = -g (v - v_peer)
        errs.append(np.max(np.abs(d - cont)))
    # (1 - x)/(1 + x), x = gs dt / C, is the (1,1) Pade approximant of exp(-2x): for this mode
    # "own voltage implicit, peer explicit" is the trapezoidal rule, hence SECOND order
    assert errs[0] < 1e-4 * abs(d[0]) and 3.6 < errs[0] / errs[1] < 4.4


def test_p10b_gap_one_way_and_sign():
    # a junction on cell 0 only, towards the decoy: cell 0 is pulled TOWARDS the decoy's voltage,
    # the decoy does not feel it (one half of a junction is one point process)
    desc, area = _gap_cells(0.01, [(0, 1)], amp=0.0)
    m = OracleModel(desc)
    m.set_probes([0, 1, 2])
    m.run(10.0, DT)
    tr = m.get_trace()
    assert np.all(np.diff(tr[:, 0]) > 0) and tr[-1, 0] > -60.0      # decoy rises towards 0 mV
    assert np.all(tr[:, 0] < tr[:, 1])
    assert np.all(tr[:, 2] == -65.0)
    alone, _ = _gap_cells(0.01, [], amp=0.0)
    ma = OracleModel(alone)
    ma.set_probes([1])
    ma.run(10.0, DT)
    assert np.array_equal(ma.get_trace()[:, 0], tr[:, 1])
    # one step by hand: v0' = v0 - gs (v0 - v1) / (c + gs) with v1 of the start of the step
    c, gs = 1e-3 / DT, 100.0 * 0.01 / area
    k = 100
    assert abs(tr[k + 1, 0] - (tr[k, 0] - gs * (tr[k, 0] - tr[k, 1]) / (c + gs))) < 1e-13


def test_p10b_gap_peer_validated():
    for bad in (3.0, -1.0, 0.5):
        desc, _ = _gap_cells(0.01, [(0, bad)])
        with pytest.raises(Exception):
            OracleModel(desc)


# ---------------------------------------------------------------------------------------------
# P11: threshold semantics (R5)
# ---------------------------------------------------------------------------------------------

def _two_pulse(thr):
    desc = W.single_compartment([("pas", {"g": 0.001, "e": -65.0}, {})], thr=thr)
    desc["mechs"].append({"type": "iclamp", "node": np.zeros(2, np.int32),
                          "params": {"del": np.array([1.0, 8.0]), "dur": np.array([1.0, 1.0]),
                                     "amp": np.array([0.4, 0.4])}, "globals": {}})
    return desc


def test_p11_one_spike_per_excursion_and_rearm():
    m = OracleModel(_two_pulse(-50.0))
    m.set_probes([0])
    m.run(15.0, DT)
    tr = m.get_trace()[:, 0]
    g, s = m.get_spikes()
    above = tr > -50.0
    rising = np.nonzero(above[1:] & ~above[:-1])[0] + 2   # trace row j holds v after step j (t_{j+1})
    assert len(g) == 2 and list(s) == list(rising)
    assert np.all(tr[s - 1] > -50.0) and np.all(tr[s - 2] <= -50.0)


def test_p11_equal_to_threshold_is_not_a_crossing():
    m = OracleModel(_two_pulse(-50.0))
    m.set_probes([0])
    m.run(3.0, DT)
    tr = m.get_trace()[:, 0]
    s0 = int(m.get_spikes()[1][0])
    v_at = tr[s0 - 1]                       # first value above -50
    m2 = OracleModel(_two_pulse(float(v_at)))   # threshold exactly equal to that value
    m2.run(3.0, DT)
    s2 = int(m2.get_spikes()[1][0])
    assert s2 == s0 + 1                     # strict '>' : crossing registered one step later


def test_p11_initially_above_threshold_needs_rearm():
    desc = W.single_compartment([("pas", {"g": 0.001, "e": -65.0}, {})], v_init=-10.0, thr=-20.0)
    m = OracleModel(desc)
    m.run(20.0, DT)
    assert len(m.get_spikes()[0]) == 0


# ---------------------------------------------------------------------------------------------
# P12: exact ring timing
# ---------------------------------------------------------------------------------------------

def _passive_ring(n_cell, d_steps, w=0.02, thr=-64.0):
    area = math.pi * 20.0 * 20.0
    N = n_cell
    desc = {
        "cell_first": np.arange(N + 1, dtype=np.int64), "parent": np.full(N, -1, np.int32),
        "area": np.full(N, area), "ri": np.ones(N), "cm": np.ones(N), "v_init": -65.0,
        "celsius": 6.3,
        "mechs": [
            {"type": "pas", "node": np.arange(N, dtype=np.int32),
             "params": {"g": np.full(N, 0.001), "e": np.full(N, -65.0)}, "globals": {}},
            {"type": "expsyn", "node": np.arange(N, dtype=np.int32),
             "params": {"tau": np.full(N, 2.0), "e": np.zeros(N)}, "globals": {}}],
        "netcons": {"src": np.concatenate([np.arange(N), [N]]).astype(np.int32),
                    "tgt_mech": np.ones(N + 1, np.int32),
                    "tgt_inst": np.concatenate([(np.arange(N) + 1) % N, [0]]).astype(np.int64),
                    "weight": np.full(N + 1, w), "delay": np.full(N + 1, d_steps * DT)},
        "thr": np.full(N, thr), "stim": {"gid": np.array([N], np.int32), "t": np.array([0.0])}}
    return desc, area


def test_p12_ring_first_lap_exact():
    n_cell, d_steps, w, thr = 6, 40, 0.001, -64.0
    desc, area = _passive_ring(n_cell, d_steps, w, thr)
    # latency L of one cell from the closed one-compartment recurrence (independent restatement)
    v, g, L = -65.0, w, None
    c = 1e-3 / DT
    for j in range(1, 1000):
        gs = 100.0 * g / area
        v = v + (-0.001 * (v + 65.0) - gs * (v - 0.0)) / (c + 0.001 + gs)
        g = g * math.exp(-DT / 2.0)
        if v > thr:
            L = j            # spike step = delivery step + L
            break
    assert L is not None and 1 < L < 200
    m = OracleModel(desc)
    m.run((n_cell * (d_steps + L) + 5) * DT, DT)
    gid, step = m.get_spikes()
    first = {int(a): int(b) for a, b in zip(gid[::-1], step[::-1])}
    for i in range(n_cell):
        assert first[i] == d_steps + L + i * (d_steps + L)


# ---------------------------------------------------------------------------------------------
# P13: ring invariances (exact)
# ---------------------------------------------------------------------------------------------

def test_p13_rotating_the_stimulus_rotates_the_spikes():
    m0 = OracleModel(W.config1())
    m0.run(30.0, DT)
    g0, s0 = m0.get_spikes()
    assert len(g0) > 10
    for j in (3, 7):
        mj = OracleModel(W.config1(stim_cell=j))
        mj.run(30.0, DT)
        gj, sj = mj.get_spikes()
        assert list(sj) == list(s0) and list(gj) == list((g0 + j) % 8)


def test_p13_rings_alone_equal_rings_together():
    kw = dict(n_cell=12, ring_size=4, depth=2, ncomp_branch=4, weight=0.05)
    full = OracleModel(W.config2(**kw))
    full.run(25.0, DT)
    gf, sf = full.get_spikes()
    vf = full.get_v()
    assert len(gf) > 6
    n = len(vf) // 12
    for r in range(3):
        sub = OracleModel(W.config2(rings=[r], **kw))
        sub.run(25.0, DT)
        gs, ss = sub.get_spikes()
        sel = (gf // 4) == r
        assert list(gs + 4 * r) == list(gf[sel]) and list(ss) == list(sf[sel])
        assert np.array_equal(sub.get_v(), vf[r * 4 * n:(r + 1) * 4 * n])


def test_p13_permuting_cells_permutes_results_bitwise():
    desc = W.random_tree_cells(7, 20, 45, stream="p13", weight=0.08)
    perm = np.array([4, 0, 6, 2, 5, 1, 3])
    m = OracleModel(desc)
    m.run(20.0, DT)
    mp = OracleModel(W.extract_cells(desc, perm))
    mp.run(20.0, DT)
    g, s = m.get_spikes()
    gp, sp = mp.get_spikes()
    assert len(g) > 3
    back = sorted(zip(sp, perm[gp]))
    assert back == sorted(zip(s, g))
    cf = desc["cell_first"]
    v, vp = m.get_v(), mp.get_v()
    cfp = np.concatenate([[0], np.cumsum((cf[1:] - cf[:-1])[perm])])
    for j, c in enumerate(perm):
        assert np.array_equal(vp[cfp[j]:cfp[j + 1]], v[cf[c]:cf[c + 1]])


# ---------------------------------------------------------------------------------------------
# P14: node-order invariance
# ---------------------------------------------------------------------------------------------

def test_p14_node_renumbering():
    # (weight 0.4 / amp 4.0: with the generator's defaults -- 0.08 uS, 0.5 nA -- these small cells
    # never reach threshold, so the pin would compare sub-threshold voltages only; with the stronger
    # drive 12 spikes travel round the ring and the spike list is part of the comparison)
    desc = W.random_tree_cells(3, 30, 60, stream="p14", weight=0.4, amp=4.0)
    ren = W.renumber_nodes(desc)
    m, mr = OracleModel(desc), OracleModel(ren)
    m.run(15.0, DT)
    mr.run(15.0, DT)
    v, vr = m.get_v(), mr.get_v()
    assert not np.array_equal(ren["parent"], desc["parent"])
    assert np.max(np.abs(vr[ren["_new_of_old"]] - v)) < 1e-10
    assert len(m.get_spikes()[0]) >= 10
    assert [list(x) for x in m.get_spikes()] == [list(x) for x in mr.get_spikes()]


# ---------------------------------------------------------------------------------------------
# P15: causality
# ---------------------------------------------------------------------------------------------

def test_p15_causality():
    desc = W.config1()
    m = OracleModel(desc)
    m.run(100.0, DT)
    g, s = m.get_spikes()
    first = {}
    for a, b in zip(g, s):
        first.setdefault(int(a), int(b))
    assert len(first) == 8
    for c in range(1, 8):
        assert first[c] >= first[c - 1] + 40 + 1


# ---------------------------------------------------------------------------------------------
# P16: whole-model first-order convergence
# ---------------------------------------------------------------------------------------------

def test_p16_config1_first_order_in_dt():
    traces = []
    for dt in (0.025, 0.0125, 0.00625):
        m = OracleModel(W.config1())
        m.set_probes([0, 30, 60])   # cell 0 only: later cells see grid-quantised spike times
        m.run(6.0, dt)
        tr = m.get_trace()
        k = int(round(0.025 / dt))
        traces.append(tr[k - 1::k])
    e1 = np.max(np.abs(traces[0] - traces[1]))
    e2 = np.max(np.abs(traces[1] - traces[2]))
    assert 1.8 < e1 / e2 < 2.2


# ---------------------------------------------------------------------------------------------
# workload shapes against the paper's printed sizes
# ---------------------------------------------------------------------------------------------

def test_table1_ring_sizes():
    vals = {}
    for line in (Path(__file__).parent / "golden" / "table1_ring.txt").read_text().splitlines():
        if line and not line.startswith("#"):
            k, v = line.split()
            vals[k] = int(v)
    small = W.config4(n_cell=128, n_types=4)
    n_per = len(small["parent"]) // 128
    assert n_per == 291 and vals["neurons"] * n_per == vals["compartments"]
    n_ring = vals["neurons"] // 64
    assert vals["neurons"] + n_ring == vals["synapses"]
    assert len(small["netcons"]["src"]) == 128 + 2
    d1 = W.config1()
    assert len(d1["parent"]) == 8 * 61
    d2 = W.config2(n_cell=4, ring_size=4)
    assert len(d2["parent"]) == 4 * 601


def test_invalid_descriptions_rejected():
    desc = W.config1()
    bad = dict(desc)
    bad["parent"] = desc["parent"].copy()
    bad["parent"][5] = 9          # parent after child
    with pytest.raises(ValueError):
        OracleModel(bad)
    bad = dict(desc)
    bad["parent"] = desc["parent"].copy()
    bad["parent"][62] = 3         # parent in another cell
    with pytest.raises(ValueError):
        OracleModel(bad)
