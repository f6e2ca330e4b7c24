/*
 * cn_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, sequential CPU fp64 oracle for the fixed-step time-integration
 * hot path of arxiv 1901.10975 (CoreNEURON):  event delivery -> matrix assembly
 * (nrn_cur + tree terms) -> Hines solve -> voltage update -> nrn_state ->
 * threshold detection   (Eq. 1, units L58-60).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, header or constant
 * table with the CUDA path under paper_1901_10975_b200/ and include/.
 *
 * Parity pins (tests/test_oracle_pins.py, P1..P16 of SURVEY.md 8(c)) check it
 * against closed forms, Thomas / dense LU solves, RK4 and exact ring timing.
 * The model-level plumbing ica -> cai -> SK of one_step (per-step zeroing of ica, accumulation
 * over several Ca channels, the order of cai dynamics and SK in nrn_state, the cai floor of
 * z_inf) is pinned by P9b.
 * "parity unpinned": the VALUES of the synthetic channel constants / network densities of
 * configs 3 and 5 have no external truth (every formula they enter is pinned: P7/P8/P9/P9b).
 */
#ifndef CN_ORACLE_H
#define CN_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* mechanism types (oracle's own numbering) */
enum {
  ORC_PAS = 1,      /* param: g, e                         (S/cm2, mV)            */
  ORC_HH = 2,       /* param: gnabar, gkbar, gl, el ; global: ena, ek             */
  ORC_EXPSYN = 3,   /* param: tau, e ; state g (uS)                                */
  ORC_EXP2SYN = 4,  /* param: tau1, tau2, e ; states A, B                          */
  ORC_ICLAMP = 5,   /* param: del, dur, amp (ms, ms, nA)                           */
  ORC_HHFORM = 6,   /* param: gbar ; global: p,q,E,to_ica, m(vh,k,t0,t1,vt,s), h(..)*/
  ORC_SK = 7,       /* param: gbar ; global: E, Kd, n, tau_z ; state z             */
  ORC_CADYN = 8,    /* no param ; global: gamma, depth, tau_d, cai_min ; state cai */
  ORC_AMPANMDA = 9, /* no param ; global: tau_r_A,tau_d_A,tau_r_N,tau_d_N,r_nmda,mg,e */
  ORC_GAP = 10      /* param: g (uS), peer (global node index, as a double) ; no state.
                       Gap junction of the fixed-step method: point current
                       i = g (v - v_peer) with v_peer the peer's voltage at the START of the step
                       (the voltages are exchanged once per step), conductance g              */
};

enum { ORC_OK = 0, ORC_ERR = -1 };

typedef struct {
  int32_t type;
  int64_t n;            /* instances */
  const int32_t *node;  /* [n] global node index */
  int32_t n_param;
  const double *param;  /* [n_param][n], SoA */
  int32_t n_global;
  const double *global;
} orc_mech;

typedef struct {
  int32_t n_cell;
  int64_t n_node;
  const int64_t *cell_first; /* [n_cell+1]; cell_first[c] is the root of cell c; gid = c */
  const int32_t *parent;     /* [n_node]; -1 for roots; parent[i] < i */
  const double *area;        /* um2 */
  const double *ri;          /* MOhm, node <-> parent */
  const double *cm;          /* uF/cm2 */
  double v_init, celsius;
  int32_t n_mech;
  const orc_mech *mech;
  int64_t n_netcon;
  const int32_t *nc_src;      /* source gid: cell (< n_cell) or scripted source (>= n_cell) */
  const int32_t *nc_tgt_mech; /* index into mech[] */
  const int64_t *nc_tgt_inst;
  const double *nc_weight;    /* uS */
  const double *nc_delay;     /* ms */
  const double *thr;          /* [n_cell] mV */
  int64_t n_stim;             /* scripted source spikes */
  const int32_t *stim_gid;    /* >= n_cell */
  const double *stim_t;       /* ms; step = llround(t/dt) */
} orc_desc;

typedef struct orc_model orc_model;

orc_model *orc_create(const orc_desc *desc); /* deep copy; NULL on invalid input */
void orc_destroy(orc_model *m);
int orc_run(orc_model *m, double tstop, double dt); /* to ABSOLUTE time; K = llround(tstop/dt) - done */
int64_t orc_steps_done(const orc_model *m);
int orc_get_v(const orc_model *m, double *out, int64_t n);
int64_t orc_n_spikes(const orc_model *m);
int orc_get_spikes(const orc_model *m, int32_t *gid, int64_t *step, int64_t cap);
double orc_min_margin(const orc_model *m); /* min over spikes of min(|v_new-thr|, |v_old-thr|) (R16) */
/* probes: v at the given nodes is appended after every step */
int orc_set_probes(orc_model *m, const int32_t *node, int64_t n);
int64_t orc_trace_steps(const orc_model *m);
int orc_get_trace(const orc_model *m, double *out, int64_t cap_steps); /* [steps][n_probe] */
/* state inspection: state s of mechanism table t -> out[n]; returns number of states of that type */
int orc_get_state(const orc_model *m, int32_t t, int32_t s, double *out, int64_t n);
int orc_get_cai(const orc_model *m, double *out, int64_t n);
/* per-node matrix coefficients a, b (S/cm2) */
int orc_get_ab(const orc_model *m, double *a, double *b, int64_t n);
/* the assembled system of the LAST step, saved before triangularisation (for residual pins) */
int orc_get_last_system(const orc_model *m, double *d, double *rhs, double *sol, int64_t n);

/* ---- pieces exposed for the pins (the model step is built from exactly these) ---- */
/* O4+O5: axial + capacitive terms added into d, rhs */
void orc_assemble_tree(int64_t n, const int32_t *parent, const double *a, const double *b,
                       const double *cm, double dt, const double *v, double *d, double *rhs);
/* O6+O7: Hines elimination; rhs becomes the solution */
void orc_hines(int64_t n, const int32_t *parent, const double *a, const double *b, double *d,
               double *rhs);
/* HH rate functions: out = {minf, mtau, hinf, htau, ninf, ntau} */
void orc_hh_rates(double v, double celsius, double *out6);
/* HHFORM gate: out = {xinf, xtau} for gate descriptor g6 = (vh,k,t0,t1,vt,s) */
void orc_hhform_gate(double v, const double *g6, double *out2);
/* number of states / params of a type */
int orc_n_state(int32_t type);
int orc_n_param(int32_t type);
/* one-instance mechanism calls: P params, S states, G globals */
void orc_mech_init(int32_t type, const double *G, const double *P, double *S, double v,
                   double celsius);
/* current (i) and conductance (g): distributed mA/cm2 & S/cm2, point nA & uS; ica part separately */
void orc_mech_cur(int32_t type, const double *G, const double *P, const double *S, double v,
                  double cai, double t_mid, double *i, double *g, double *ica);
void orc_mech_state(int32_t type, const double *G, const double *P, double *S, double v,
                    double dt, double celsius, double *cai, double ica);
/* event delivery onto one instance */
void orc_mech_receive(int32_t type, const double *G, const double *P, double *S, double w);
double orc_exp2syn_factor(double tau1, double tau2);

#ifdef __cplusplus
}
#endif
#endif
