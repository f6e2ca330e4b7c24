/*
 * cn_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see cn_oracle.h).
 *
 * Sequential fp64 restatement of the per-dt operations of PAPER.md L62-68:
 *   O1 deliver events (L64)           O6 Hines triangularisation (L62, L66)
 *   O2 zero rhs, d                    O7 back-substitution (L66)
 *   O3 mechanism currents (L65)       O8 v += rhs (L66)
 *   O4 axial terms (Eq. 1)       O9 mechanism states (L67)
 *   O5 diagonal cm/dt (Eq. 1)         O10 threshold detection (L68)
 * in the paper's order, in caller node order, no blocking / fusion / SIMD.
 * Units follow L58-60: mV, ms, uF/cm2, mA/cm2, S/cm2; point processes nA, uS,
 * converted by 100/area[um2] (L60: "division by the compartment area").
 * Readings R1..R22 of the silent points are listed in DESIGN.md.
 * Build: gcc -O2 -ffp-contract=off -std=c99 (R22).
 */
#include "cn_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define FARADAY 96485.33212 /* C/mol */

/* ------------------------------------------------------------------ */
/* mechanism definitions (SURVEY 8(c) "Mechanisms")                    */
/* ------------------------------------------------------------------ */

int orc_n_state(int32_t type) {
  switch (type) {
    case ORC_PAS: return 0;
    case ORC_HH: return 3;      /* m h n */
    case ORC_EXPSYN: return 1;  /* g */
    case ORC_EXP2SYN: return 2; /* A B */
    case ORC_ICLAMP: return 0;
    case ORC_HHFORM: return 2;  /* m h */
    case ORC_SK: return 1;      /* z */
    case ORC_CADYN: return 0;   /* cai lives in the per-node ion array */
    case ORC_AMPANMDA: return 4; /* A_ampa B_ampa A_nmda B_nmda */
    case ORC_GAP: return 0;
  }
  return -1;
}

int orc_n_param(int32_t type) {
  switch (type) {
    case ORC_PAS: return 2;
    case ORC_HH: return 4;
    case ORC_EXPSYN: return 2;
    case ORC_EXP2SYN: return 3;
    case ORC_ICLAMP: return 3;
    case ORC_HHFORM: return 1;
    case ORC_SK: return 1;
    case ORC_CADYN: return 0;
    case ORC_AMPANMDA: return 0;
    case ORC_GAP: return 2;
  }
  return -1;
}

static int n_global_of(int32_t type) {
  switch (type) {
    case ORC_PAS: return 0;
    case ORC_HH: return 2;
    case ORC_EXPSYN: return 0;
    case ORC_EXP2SYN: return 0;
    case ORC_ICLAMP: return 0;
    case ORC_HHFORM: return 16;
    case ORC_SK: return 4;
    case ORC_CADYN: return 4;
    case ORC_AMPANMDA: return 7;
    case ORC_GAP: return 0;
  }
  return -1;
}

static int is_point(int32_t type) {
  return type == ORC_EXPSYN || type == ORC_EXP2SYN || type == ORC_ICLAMP || type == ORC_AMPANMDA ||
         type == ORC_GAP;
}

/* x / (exp(x/y) - 1) with the removable singularity at x = 0 */
static double vtrap(double x, double y) {
  double u = x / y;
  if (fabs(u) < 1e-6) return y * (1.0 - u / 2.0);
  return x / (exp(u) - 1.0);
}

/* Hodgkin-Huxley 1952 squid axon, rest at -65 mV convention */
void orc_hh_rates(double v, double celsius, double *out6) {
  double q10 = pow(3.0, (celsius - 6.3) / 10.0);
  double alpha, beta, sum;
  alpha = 0.1 * vtrap(-(v + 40.0), 10.0);
  beta = 4.0 * exp(-(v + 65.0) / 18.0);
  sum = alpha + beta;
  out6[0] = alpha / sum;
  out6[1] = 1.0 / (q10 * sum);
  alpha = 0.07 * exp(-(v + 65.0) / 20.0);
  beta = 1.0 / (exp(-(v + 35.0) / 10.0) + 1.0);
  sum = alpha + beta;
  out6[2] = alpha / sum;
  out6[3] = 1.0 / (q10 * sum);
  alpha = 0.01 * vtrap(-(v + 55.0), 10.0);
  beta = 0.125 * exp(-(v + 65.0) / 80.0);
  sum = alpha + beta;
  out6[4] = alpha / sum;
  out6[5] = 1.0 / (q10 * sum);
}

/* HH-form gate: xinf = 1/(1+exp((vh-v)/k)), tau = t0 + t1/(exp((v-vt)/s)+exp(-(v-vt)/s)) */
void orc_hhform_gate(double v, const double *g6, double *out2) {
  double vh = g6[0], k = g6[1], t0 = g6[2], t1 = g6[3], vt = g6[4], s = g6[5];
  double u = (v - vt) / s;
  out2[0] = 1.0 / (1.0 + exp((vh - v) / k));
  out2[1] = t0 + t1 / (exp(u) + exp(-u));
}

static double ipow(double x, int p) {
  double r = 1.0;
  int j;
  for (j = 0; j < p; ++j) r *= x;
  return r;
}

double orc_exp2syn_factor(double tau1, double tau2) {
  double tp = (tau1 * tau2) / (tau2 - tau1) * log(tau2 / tau1);
  return 1.0 / (exp(-tp / tau2) - exp(-tp / tau1));
}

static double mgblock(double v, double mg) { return 1.0 / (1.0 + exp(-0.062 * v) * (mg / 3.57)); }

static double sk_zinf(const double *G, double cai) {
  if (cai < 1e-9) cai = 1e-9;
  return 1.0 / (1.0 + pow(G[1] / cai, G[2]));
}

void orc_mech_init(int32_t type, const double *G, const double *P, double *S, double v,
                   double celsius) {
  double r[6], g2[2];
  (void)P;
  switch (type) {
    case ORC_HH:
      orc_hh_rates(v, celsius, r);
      S[0] = r[0];
      S[1] = r[2];
      S[2] = r[4];
      break;
    case ORC_EXPSYN: S[0] = 0.0; break;
    case ORC_EXP2SYN: S[0] = S[1] = 0.0; break;
    case ORC_HHFORM:
      orc_hhform_gate(v, G + 4, g2);
      S[0] = g2[0];
      orc_hhform_gate(v, G + 10, g2);
      S[1] = g2[0];
      break;
    case ORC_SK: S[0] = 0.0; break; /* set from cai by the model after ion init */
    case ORC_AMPANMDA: S[0] = S[1] = S[2] = S[3] = 0.0; break;
    default: break;
  }
}

void orc_mech_cur(int32_t type, const double *G, const double *P, const double *S, double v,
                  double cai, double t_mid, double *i, double *g, double *ica) {
  double gna, gk, gg;
  (void)cai;
  *i = 0.0;
  *g = 0.0;
  *ica = 0.0;
  switch (type) {
    case ORC_PAS:
      *g = P[0];
      *i = P[0] * (v - P[1]);
      break;
    case ORC_HH:
      gna = P[0] * S[0] * S[0] * S[0] * S[1];
      gk = P[1] * S[2] * S[2] * S[2] * S[2];
      *i = gna * (v - G[0]) + gk * (v - G[1]) + P[2] * (v - P[3]);
      *g = gna + gk + P[2];
      break;
    case ORC_EXPSYN:
      *g = S[0];
      *i = S[0] * (v - P[1]);
      break;
    case ORC_EXP2SYN:
      *g = S[1] - S[0];
      *i = (S[1] - S[0]) * (v - P[2]);
      break;
    case ORC_ICLAMP:
      /* electrode current: i is negative membrane current; active iff del <= t_mid < del+dur (R10) */
      if (t_mid >= P[0] && t_mid < P[0] + P[1]) *i = -P[2];
      break;
    case ORC_HHFORM:
      gg = P[0] * ipow(S[0], (int)G[0]) * ipow(S[1], (int)G[1]);
      *g = gg;
      *i = gg * (v - G[2]);
      if (G[3] != 0.0) *ica = *i;
      break;
    case ORC_SK:
      *g = P[0] * S[0];
      *i = P[0] * S[0] * (v - G[0]);
      break;
    case ORC_AMPANMDA:
      gg = (S[1] - S[0]) + G[4] * (S[3] - S[2]) * mgblock(v, G[5]);
      *g = gg; /* CONDUCTANCE semantics (L160, R7): mg(v) held fixed */
      *i = gg * (v - G[6]);
      break;
    default: break;
  }
}

/* cnexp: y += (1 - exp(-dt/tau)) * (yinf - y) */
static double cnexp(double y, double yinf, double tau, double dt) {
  return y + (1.0 - exp(-dt / tau)) * (yinf - y);
}

void orc_mech_state(int32_t type, const double *G, const double *P, double *S, double v,
                    double dt, double celsius, double *cai, double ica) {
  double r[6], g2[2];
  switch (type) {
    case ORC_HH:
      orc_hh_rates(v, celsius, r);
      S[0] = cnexp(S[0], r[0], r[1], dt);
      S[1] = cnexp(S[1], r[2], r[3], dt);
      S[2] = cnexp(S[2], r[4], r[5], dt);
      break;
    case ORC_EXPSYN: S[0] = cnexp(S[0], 0.0, P[0], dt); break;
    case ORC_EXP2SYN:
      S[0] = cnexp(S[0], 0.0, P[0], dt);
      S[1] = cnexp(S[1], 0.0, P[1], dt);
      break;
    case ORC_HHFORM:
      if ((int)G[0] > 0) {
        orc_hhform_gate(v, G + 4, g2);
        S[0] = cnexp(S[0], g2[0], g2[1], dt);
      }
      if ((int)G[1] > 0) {
        orc_hhform_gate(v, G + 10, g2);
        S[1] = cnexp(S[1], g2[0], g2[1], dt);
      }
      break;
    case ORC_SK: S[0] = cnexp(S[0], sk_zinf(G, *cai), G[3], dt); break;
    case ORC_CADYN: {
      /* derivimplicit (L278): backward Euler, F(y) = y - y0 - dt*f(y) = 0 by Newton */
      double kappa = 1e4 * G[0] / (2.0 * FARADAY * G[1]);
      double y0 = *cai, y = y0;
      int it;
      for (it = 0; it < 50; ++it) {
        double f = -kappa * ica - (y - G[3]) / G[2];
        double F = y - y0 - dt * f;
        double dF = 1.0 + dt / G[2];
        double dy = F / dF;
        y -= dy;
        if (fabs(dy) <= 1e-12 * fabs(y)) break;
      }
      *cai = y;
      break;
    }
    case ORC_AMPANMDA:
      S[0] = cnexp(S[0], 0.0, G[0], dt);
      S[1] = cnexp(S[1], 0.0, G[1], dt);
      S[2] = cnexp(S[2], 0.0, G[2], dt);
      S[3] = cnexp(S[3], 0.0, G[3], dt);
      break;
    default: break;
  }
  (void)celsius;
}

void orc_mech_receive(int32_t type, const double *G, const double *P, double *S, double w) {
  double f;
  switch (type) {
    case ORC_EXPSYN: S[0] += w; break;
    case ORC_EXP2SYN:
      f = orc_exp2syn_factor(P[0], P[1]);
      S[0] += w * f;
      S[1] += w * f;
      break;
    case ORC_AMPANMDA:
      f = orc_exp2syn_factor(G[0], G[1]);
      S[0] += w * f;
      S[1] += w * f;
      f = orc_exp2syn_factor(G[2], G[3]);
      S[2] += w * f;
      S[3] += w * f;
      break;
    default: break;
  }
}

/* ------------------------------------------------------------------ */
/* tree matrix pieces                                                  */
/* ------------------------------------------------------------------ */

/* O4 axial rhs terms and O5 diagonal terms (Eq. 1 discretised; backward Euler in delta-v form) */
void orc_assemble_tree(int64_t n, const int32_t *parent, const double *a, const double *b,
                       const double *cm, double dt, const double *v, double *d, double *rhs) {
  int64_t i;
  for (i = 0; i < n; ++i) {
    int32_t p = parent[i];
    if (p >= 0) {
      double dv = v[p] - v[i];
      rhs[i] -= b[i] * dv;
      rhs[p] += a[i] * dv;
    }
  }
  for (i = 0; i < n; ++i) {
    int32_t p = parent[i];
    d[i] += 1e-3 * cm[i] / dt;
    if (p >= 0) {
      d[i] -= b[i];
      d[p] -= a[i];
    }
  }
}

/* O6 + O7: Gaussian elimination on the tree, children before parents (L62, L196 par[i]) */
void orc_hines(int64_t n, const int32_t *parent, const double *a, const double *b, double *d,
               double *rhs) {
  int64_t i;
  for (i = n - 1; i >= 0; --i) {
    int32_t p = parent[i];
    if (p >= 0) {
      double f = a[i] / d[i];
      d[p] -= f * b[i];
      rhs[p] -= f * rhs[i];
    }
  }
  for (i = 0; i < n; ++i) {
    int32_t p = parent[i];
    if (p < 0) {
      rhs[i] /= d[i];
    } else {
      rhs[i] -= b[i] * rhs[p];
      rhs[i] /= d[i];
    }
  }
}

/* ------------------------------------------------------------------ */
/* the model                                                           */
/* ------------------------------------------------------------------ */

typedef struct {
  int32_t type;
  int64_t n;
  int32_t *node;
  int32_t n_param, n_state, n_global;
  double *param; /* [n_param][n] */
  double *state; /* [n_state][n] */
  double *global;
} mech_t;

typedef struct {
  int64_t *ev; /* netcon indices */
  int64_t n, cap;
} slot_t;

struct orc_model {
  int32_t n_cell;
  int64_t n_node;
  int64_t *cell_first;
  int32_t *parent;
  double *area, *ri, *cm, *a, *b;
  double *v, *d, *rhs, *ica, *cai;
  double *d_saved, *rhs_saved;
  double v_init, celsius;
  int32_t n_mech;
  mech_t *mech;
  int64_t n_netcon;
  int32_t *nc_src, *nc_tgt_mech;
  int64_t *nc_tgt_inst;
  double *nc_weight, *nc_delay;
  int64_t *nc_dsteps;
  int32_t n_src; /* number of gids incl. scripted sources */
  int64_t *src_first, *src_list; /* CSR of netcons by source gid, in netcon order */
  double *thr;
  unsigned char *flag;
  int64_t n_stim;
  int32_t *stim_gid;
  double *stim_t;
  int64_t *stim_step;
  /* run state */
  double dt;
  int64_t k; /* steps done */
  int64_t W;
  slot_t *wheel;
  int32_t *sp_gid;
  int64_t *sp_step;
  int64_t n_sp, cap_sp;
  double min_margin;
  int64_t n_probe;
  int32_t *probe;
  double *trace;
  int64_t n_trace, cap_trace;
};

static void *dup_mem(const void *src, size_t bytes) {
  void *p = malloc(bytes ? bytes : 1);
  if (src && bytes) memcpy(p, src, bytes);
  return p;
}

orc_model *orc_create(const orc_desc *de) {
  orc_model *m;
  int64_t i, N;
  int32_t t, c;
  if (!de || de->n_cell < 0 || de->n_node < 0) return NULL;
  N = de->n_node;
  /* validation */
  for (c = 0; c < de->n_cell; ++c) {
    int64_t f = de->cell_first[c], l = de->cell_first[c + 1];
    if (l <= f) return NULL;
    if (de->parent[f] != -1) return NULL;
    for (i = f + 1; i < l; ++i)
      if (de->parent[i] < f || de->parent[i] >= i) return NULL;
  }
  if (de->n_cell > 0 && (de->cell_first[0] != 0 || de->cell_first[de->n_cell] != N)) return NULL;
  for (t = 0; t < de->n_mech; ++t) {
    const orc_mech *mt = &de->mech[t];
    if (orc_n_state(mt->type) < 0) return NULL;
    if (mt->n_param != orc_n_param(mt->type) || mt->n_global != n_global_of(mt->type)) return NULL;
    for (i = 0; i < mt->n; ++i)
      if (mt->node[i] < 0 || mt->node[i] >= N) return NULL;
    if (mt->type == ORC_GAP) /* the peer is a node of the model, given as an integral double */
      for (i = 0; i < mt->n; ++i) {
        double pr = mt->param[(int64_t)1 * mt->n + i];
        if (!(pr >= 0.0 && pr < (double)N) || pr != (double)(int64_t)pr) return NULL;
      }
  }
  for (i = 0; i < de->n_netcon; ++i) {
    int32_t tm = de->nc_tgt_mech[i];
    if (tm < 0 || tm >= de->n_mech) return NULL;
    if (de->nc_tgt_inst[i] < 0 || de->nc_tgt_inst[i] >= de->mech[tm].n) return NULL;
    if (de->nc_src[i] < 0) return NULL;
  }

  m = (orc_model *)calloc(1, sizeof(*m));
  m->n_cell = de->n_cell;
  m->n_node = N;
  m->cell_first = (int64_t *)dup_mem(de->cell_first, sizeof(int64_t) * (size_t)(de->n_cell + 1));
  m->parent = (int32_t *)dup_mem(de->parent, sizeof(int32_t) * (size_t)N);
  m->area = (double *)dup_mem(de->area, sizeof(double) * (size_t)N);
  m->ri = (double *)dup_mem(de->ri, sizeof(double) * (size_t)N);
  m->cm = (double *)dup_mem(de->cm, sizeof(double) * (size_t)N);
  m->a = (double *)calloc((size_t)N + 1, sizeof(double));
  m->b = (double *)calloc((size_t)N + 1, sizeof(double));
  m->v = (double *)calloc((size_t)N + 1, sizeof(double));
  m->d = (double *)calloc((size_t)N + 1, sizeof(double));
  m->rhs = (double *)calloc((size_t)N + 1, sizeof(double));
  m->ica = (double *)calloc((size_t)N + 1, sizeof(double));
  m->cai = (double *)calloc((size_t)N + 1, sizeof(double));
  m->d_saved = (double *)calloc((size_t)N + 1, sizeof(double));
  m->rhs_saved = (double *)calloc((size_t)N + 1, sizeof(double));
  m->v_init = de->v_init;
  m->celsius = de->celsius;

  /* per-model constants (R1): b = -100/(ri*area_i), a = -100/(ri*area_parent)  [S/cm2] */
  for (i = 0; i < N; ++i) {
    int32_t p = m->parent[i];
    if (p >= 0) {
      m->b[i] = -100.0 / (m->ri[i] * m->area[i]);
      m->a[i] = -100.0 / (m->ri[i] * m->area[p]);
    }
    m->v[i] = m->v_init;
    m->cai[i] = 1e-4; /* default intracellular Ca (mM) where no CADYN instance sits */
  }

  m->n_mech = de->n_mech;
  m->mech = (mech_t *)calloc((size_t)de->n_mech + 1, sizeof(mech_t));
  for (t = 0; t < de->n_mech; ++t) {
    const orc_mech *src = &de->mech[t];
    mech_t *mt = &m->mech[t];
    mt->type = src->type;
    mt->n = src->n;
    mt->n_param = src->n_param;
    mt->n_global = src->n_global;
    mt->n_state = orc_n_state(src->type);
    mt->node = (int32_t *)dup_mem(src->node, sizeof(int32_t) * (size_t)src->n);
    mt->param = (double *)dup_mem(src->param, sizeof(double) * (size_t)(src->n * src->n_param));
    mt->global = (double *)dup_mem(src->global, sizeof(double) * (size_t)src->n_global);
    mt->state = (double *)calloc((size_t)(src->n * mt->n_state) + 1, sizeof(double));
  }
  /* initial conditions (R11): ion pools first, then gates at their steady state */
  for (t = 0; t < m->n_mech; ++t) {
    mech_t *mt = &m->mech[t];
    if (mt->type == ORC_CADYN)
      for (i = 0; i < mt->n; ++i) m->cai[mt->node[i]] = mt->global[3];
  }
  for (t = 0; t < m->n_mech; ++t) {
    mech_t *mt = &m->mech[t];
    for (i = 0; i < mt->n; ++i) {
      double P[8], S[8];
      int j;
      for (j = 0; j < mt->n_param; ++j) P[j] = mt->param[(int64_t)j * mt->n + i];
      for (j = 0; j < mt->n_state; ++j) S[j] = 0.0;
      orc_mech_init(mt->type, mt->global, P, S, m->v_init, m->celsius);
      if (mt->type == ORC_SK) S[0] = sk_zinf(mt->global, m->cai[mt->node[i]]);
      for (j = 0; j < mt->n_state; ++j) mt->state[(int64_t)j * mt->n + i] = S[j];
    }
  }

  m->n_netcon = de->n_netcon;
  m->nc_src = (int32_t *)dup_mem(de->nc_src, sizeof(int32_t) * (size_t)de->n_netcon);
  m->nc_tgt_mech = (int32_t *)dup_mem(de->nc_tgt_mech, sizeof(int32_t) * (size_t)de->n_netcon);
  m->nc_tgt_inst = (int64_t *)dup_mem(de->nc_tgt_inst, sizeof(int64_t) * (size_t)de->n_netcon);
  m->nc_weight = (double *)dup_mem(de->nc_weight, sizeof(double) * (size_t)de->n_netcon);
  m->nc_delay = (double *)dup_mem(de->nc_delay, sizeof(double) * (size_t)de->n_netcon);
  m->nc_dsteps = (int64_t *)calloc((size_t)de->n_netcon + 1, sizeof(int64_t));
  m->n_stim = de->n_stim;
  m->stim_gid = (int32_t *)dup_mem(de->stim_gid, sizeof(int32_t) * (size_t)de->n_stim);
  m->stim_t = (double *)dup_mem(de->stim_t, sizeof(double) * (size_t)de->n_stim);
  m->stim_step = (int64_t *)calloc((size_t)de->n_stim + 1, sizeof(int64_t));
  /* CSR of netcons by source gid */
  m->n_src = m->n_cell;
  for (i = 0; i < m->n_netcon; ++i)
    if (m->nc_src[i] >= m->n_src) m->n_src = m->nc_src[i] + 1;
  for (i = 0; i < m->n_stim; ++i)
    if (m->stim_gid[i] >= m->n_src) m->n_src = m->stim_gid[i] + 1;
  m->src_first = (int64_t *)calloc((size_t)m->n_src + 2, sizeof(int64_t));
  m->src_list = (int64_t *)calloc((size_t)m->n_netcon + 1, sizeof(int64_t));
  for (i = 0; i < m->n_netcon; ++i) m->src_first[m->nc_src[i] + 1]++;
  for (c = 0; c < m->n_src; ++c) m->src_first[c + 1] += m->src_first[c];
  {
    int64_t *fill = (int64_t *)dup_mem(m->src_first, sizeof(int64_t) * (size_t)(m->n_src + 1));
    for (i = 0; i < m->n_netcon; ++i) m->src_list[fill[m->nc_src[i]]++] = i;
    free(fill);
  }
  m->thr = (double *)dup_mem(de->thr, sizeof(double) * (size_t)de->n_cell);
  m->flag = (unsigned char *)calloc((size_t)de->n_cell + 1, 1);
  for (c = 0; c < m->n_cell; ++c) m->flag[c] = (m->v_init > m->thr[c]);
  m->dt = 0.0;
  m->k = 0;
  m->min_margin = INFINITY;
  return m;
}

void orc_destroy(orc_model *m) {
  int32_t t;
  int64_t s;
  if (!m) return;
  free(m->cell_first); free(m->parent); free(m->area); free(m->ri); free(m->cm);
  free(m->a); free(m->b); free(m->v); free(m->d); free(m->rhs); free(m->ica); free(m->cai);
  free(m->d_saved); free(m->rhs_saved);
  for (t = 0; t < m->n_mech; ++t) {
    free(m->mech[t].node); free(m->mech[t].param); free(m->mech[t].state); free(m->mech[t].global);
  }
  free(m->mech);
  free(m->nc_src); free(m->nc_tgt_mech); free(m->nc_tgt_inst); free(m->nc_weight);
  free(m->nc_delay); free(m->nc_dsteps); free(m->stim_gid); free(m->stim_t); free(m->stim_step);
  free(m->src_first); free(m->src_list); free(m->thr); free(m->flag);
  if (m->wheel) {
    for (s = 0; s < m->W; ++s) free(m->wheel[s].ev);
    free(m->wheel);
  }
  free(m->sp_gid); free(m->sp_step); free(m->probe); free(m->trace);
  free(m);
}

static void push_event(orc_model *m, int64_t at_step, int64_t nc) {
  slot_t *s = &m->wheel[at_step % m->W];
  if (s->n == s->cap) {
    s->cap = s->cap ? 2 * s->cap : 8;
    s->ev = (int64_t *)realloc(s->ev, sizeof(int64_t) * (size_t)s->cap);
  }
  s->ev[s->n++] = nc;
}

/* a source (cell or scripted) fires with spike step ks: one event per NetCon at ks + d (R4, L156) */
static void fan_out(orc_model *m, int32_t gid, int64_t ks) {
  int64_t j;
  for (j = m->src_first[gid]; j < m->src_first[gid + 1]; ++j) {
    int64_t nc = m->src_list[j];
    push_event(m, ks + m->nc_dsteps[nc], nc);
  }
}

static int first_run_setup(orc_model *m, double dt) {
  int64_t i, maxd = 1;
  if (!(dt > 0.0)) return ORC_ERR;
  m->dt = dt;
  for (i = 0; i < m->n_netcon; ++i) {
    int64_t ds = llround(m->nc_delay[i] / dt);
    if (ds < 1) return ORC_ERR;
    m->nc_dsteps[i] = ds;
    if (ds > maxd) maxd = ds;
  }
  m->W = maxd + 1;
  m->wheel = (slot_t *)calloc((size_t)m->W, sizeof(slot_t));
  for (i = 0; i < m->n_stim; ++i) {
    m->stim_step[i] = llround(m->stim_t[i] / dt);
    if (m->stim_step[i] < 0) return ORC_ERR;
  }
  /* scripted spikes at step 0 exist before the first step */
  for (i = 0; i < m->n_stim; ++i)
    if (m->stim_step[i] == 0) fan_out(m, m->stim_gid[i], 0);
  return ORC_OK;
}

static void record_spike(orc_model *m, int32_t gid, int64_t step) {
  if (m->n_sp == m->cap_sp) {
    m->cap_sp = m->cap_sp ? 2 * m->cap_sp : 1024;
    m->sp_gid = (int32_t *)realloc(m->sp_gid, sizeof(int32_t) * (size_t)m->cap_sp);
    m->sp_step = (int64_t *)realloc(m->sp_step, sizeof(int64_t) * (size_t)m->cap_sp);
  }
  m->sp_gid[m->n_sp] = gid;
  m->sp_step[m->n_sp] = step;
  m->n_sp++;
}

static void one_step(orc_model *m) {
  const int64_t N = m->n_node, k = m->k;
  const double dt = m->dt;
  const double t_mid = ((double)k + 0.5) * dt; /* staggered grid: currents live at the midpoint (R10) */
  int64_t i;
  int32_t t, c;
  double P[8], S[8];
  int j;

  /* O1 deliver events due at step k (L64) */
  {
    slot_t *s = &m->wheel[k % m->W];
    for (i = 0; i < s->n; ++i) {
      int64_t nc = s->ev[i];
      mech_t *mt = &m->mech[m->nc_tgt_mech[nc]];
      int64_t q = m->nc_tgt_inst[nc];
      for (j = 0; j < mt->n_param; ++j) P[j] = mt->param[(int64_t)j * mt->n + q];
      for (j = 0; j < mt->n_state; ++j) S[j] = mt->state[(int64_t)j * mt->n + q];
      orc_mech_receive(mt->type, mt->global, P, S, m->nc_weight[nc]);
      for (j = 0; j < mt->n_state; ++j) mt->state[(int64_t)j * mt->n + q] = S[j];
    }
    s->n = 0;
  }
  /* O2 */
  for (i = 0; i < N; ++i) {
    m->rhs[i] = 0.0;
    m->d[i] = 0.0;
    m->ica[i] = 0.0;
  }
  /* O3 currents: tables in order, instances in table order (L65) */
  for (t = 0; t < m->n_mech; ++t) {
    mech_t *mt = &m->mech[t];
    int point = is_point(mt->type);
    for (i = 0; i < mt->n; ++i) {
      int32_t nd = mt->node[i];
      double cur, g, ica;
      for (j = 0; j < mt->n_param; ++j) P[j] = mt->param[(int64_t)j * mt->n + i];
      for (j = 0; j < mt->n_state; ++j) S[j] = mt->state[(int64_t)j * mt->n + i];
      orc_mech_cur(mt->type, mt->global, P, S, m->v[nd], m->cai[nd], t_mid, &cur, &g, &ica);
      if (mt->type == ORC_GAP) { /* L160, L228: the peer's voltage of the start of the step; all
                                    of v is still v^k here (O8 comes later) */
        cur = P[0] * (m->v[nd] - m->v[(int64_t)P[1]]);
        g = P[0];
      }
      if (point) { /* nA, uS -> mA/cm2, S/cm2 (L60) */
        m->rhs[nd] -= 100.0 * cur / m->area[nd];
        m->d[nd] += 100.0 * g / m->area[nd];
      } else {
        m->rhs[nd] -= cur;
        m->d[nd] += g;
        m->ica[nd] += ica;
      }
    }
  }
  /* O4 + O5 */
  orc_assemble_tree(N, m->parent, m->a, m->b, m->cm, dt, m->v, m->d, m->rhs);
  memcpy(m->d_saved, m->d, sizeof(double) * (size_t)N);
  memcpy(m->rhs_saved, m->rhs, sizeof(double) * (size_t)N);
  /* O6 + O7 */
  orc_hines(N, m->parent, m->a, m->b, m->d, m->rhs);
  /* O10 needs the old root voltages for the margin report only */
  /* O8 */
  for (c = 0; c < m->n_cell; ++c) {
    int64_t r = m->cell_first[c];
    m->d[r] = m->v[r]; /* stash old root v (d is dead after the solve) */
  }
  for (i = 0; i < N; ++i) m->v[i] += m->rhs[i];
  /* O9 states with the new v (L67) */
  for (t = 0; t < m->n_mech; ++t) {
    mech_t *mt = &m->mech[t];
    if (mt->n_state == 0 && mt->type != ORC_CADYN) continue;
    for (i = 0; i < mt->n; ++i) {
      int32_t nd = mt->node[i];
      for (j = 0; j < mt->n_param; ++j) P[j] = mt->param[(int64_t)j * mt->n + i];
      for (j = 0; j < mt->n_state; ++j) S[j] = mt->state[(int64_t)j * mt->n + i];
      orc_mech_state(mt->type, mt->global, P, S, m->v[nd], dt, m->celsius, &m->cai[nd],
                     m->ica[nd]);
      for (j = 0; j < mt->n_state; ++j) mt->state[(int64_t)j * mt->n + i] = S[j];
    }
  }
  /* O10 threshold on the root of each cell (L68, R5): spike step is k+1 */
  for (c = 0; c < m->n_cell; ++c) {
    int64_t r = m->cell_first[c];
    int above = m->v[r] > m->thr[c];
    if (above && !m->flag[c]) {
      double m1 = fabs(m->v[r] - m->thr[c]), m0 = fabs(m->d[r] - m->thr[c]);
      double mg = m1 < m0 ? m1 : m0;
      if (mg < m->min_margin) m->min_margin = mg;
      record_spike(m, c, k + 1);
      fan_out(m, c, k + 1);
    }
    m->flag[c] = (unsigned char)above;
  }
  for (i = 0; i < m->n_stim; ++i)
    if (m->stim_step[i] == k + 1) fan_out(m, m->stim_gid[i], k + 1);
  /* probes */
  if (m->n_probe > 0) {
    if (m->n_trace == m->cap_trace) {
      m->cap_trace = m->cap_trace ? 2 * m->cap_trace : 1024;
      m->trace = (double *)realloc(m->trace, sizeof(double) * (size_t)(m->cap_trace * m->n_probe));
    }
    for (i = 0; i < m->n_probe; ++i) m->trace[m->n_trace * m->n_probe + i] = m->v[m->probe[i]];
    m->n_trace++;
  }
  m->k = k + 1;
}

int orc_run(orc_model *m, double tstop, double dt) {
  int64_t target;
  if (!m || !(dt > 0.0)) return ORC_ERR;
  if (m->dt == 0.0) {
    if (first_run_setup(m, dt) != ORC_OK) return ORC_ERR;
  } else if (dt != m->dt) {
    return ORC_ERR;
  }
  target = llround(tstop / dt);
  while (m->k < target) one_step(m);
  return ORC_OK;
}

int64_t orc_steps_done(const orc_model *m) { return m->k; }

int orc_get_v(const orc_model *m, double *out, int64_t n) {
  if (n != m->n_node) return ORC_ERR;
  memcpy(out, m->v, sizeof(double) * (size_t)n);
  return ORC_OK;
}

int64_t orc_n_spikes(const orc_model *m) { return m->n_sp; }

int orc_get_spikes(const orc_model *m, int32_t *gid, int64_t *step, int64_t cap) {
  /* already sorted by (step, gid): steps ascend, and within a step cells are scanned in gid order */
  int64_t i, n = m->n_sp < cap ? m->n_sp : cap;
  for (i = 0; i < n; ++i) {
    gid[i] = m->sp_gid[i];
    step[i] = m->sp_step[i];
  }
  return ORC_OK;
}

double orc_min_margin(const orc_model *m) { return m->min_margin; }

int orc_set_probes(orc_model *m, const int32_t *node, int64_t n) {
  int64_t i;
  if (m->k != 0) return ORC_ERR;
  for (i = 0; i < n; ++i)
    if (node[i] < 0 || node[i] >= m->n_node) return ORC_ERR;
  free(m->probe);
  m->probe = (int32_t *)dup_mem(node, sizeof(int32_t) * (size_t)n);
  m->n_probe = n;
  return ORC_OK;
}

int64_t orc_trace_steps(const orc_model *m) { return m->n_trace; }

int orc_get_trace(const orc_model *m, double *out, int64_t cap_steps) {
  int64_t n = m->n_trace < cap_steps ? m->n_trace : cap_steps;
  memcpy(out, m->trace, sizeof(double) * (size_t)(n * m->n_probe));
  return ORC_OK;
}

int orc_get_state(const orc_model *m, int32_t t, int32_t s, double *out, int64_t n) {
  const mech_t *mt;
  if (t < 0 || t >= m->n_mech) return ORC_ERR;
  mt = &m->mech[t];
  if (s < 0 || s >= mt->n_state || n != mt->n) return ORC_ERR;
  memcpy(out, mt->state + (int64_t)s * mt->n, sizeof(double) * (size_t)n);
  return mt->n_state;
}

int orc_get_cai(const orc_model *m, double *out, int64_t n) {
  if (n != m->n_node) return ORC_ERR;
  memcpy(out, m->cai, sizeof(double) * (size_t)n);
  return ORC_OK;
}

int orc_get_ab(const orc_model *m, double *a, double *b, int64_t n) {
  if (n != m->n_node) return ORC_ERR;
  memcpy(a, m->a, sizeof(double) * (size_t)n);
  memcpy(b, m->b, sizeof(double) * (size_t)n);
  return ORC_OK;
}

int orc_get_last_system(const orc_model *m, double *d, double *rhs, double *sol, int64_t n) {
  if (n != m->n_node || m->k == 0) return ORC_ERR;
  memcpy(d, m->d_saved, sizeof(double) * (size_t)n);
  memcpy(rhs, m->rhs_saved, sizeof(double) * (size_t)n);
  memcpy(sol, m->rhs, sizeof(double) * (size_t)n);
  return ORC_OK;
}
