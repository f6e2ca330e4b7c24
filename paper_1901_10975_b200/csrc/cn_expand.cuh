// cn_expand.cuh -- first cn_run, interleaved groups: the tapes are EXPANDED ON THE DEVICE from the
// caller's compact arrays (cm, ri, area, the parameters of the distributed mechanisms: 60 B per HH
// compartment) instead of being laid out on the host and uploaded whole (125 B per compartment
// over PCIe plus the host passes that fill them).  cn_model_create starts the upload of the
// compact arrays while the host compiles the layout; finalize() launches the kernels below.
//
// Arithmetic: the row-normalised system of PAPER.md L150-L160 (R3):
//   c_i = 1e-3 cm_i / dt,  b_i = -100 / (ri_i area_i),  a_i = -100 / (ri_i area_parent),
//   a' = a_i / c_parent,  b' = b_i / c_i,  d' = (c_i - b_i - sum_children a_child + sum g_pas) / c_i,
//   r' = (sum g_pas e_pas) / c_i
// written with explicit round-to-nearest operations in one fixed order (no contraction into FMAs):
// the same bits as the host pass that fills the static rows of the warp-cooperative groups
// (cn_finalize.hpp), whatever kernel a cell runs on.
#pragma once

namespace cn {

// per class with interleaved groups: where its per-node tables start in ExpTables
struct ExpClass {
  int32_t n, node_off, child_off, chf_off;  // chf_off: the class's n + 1 entries of ch_first
};

// where a caller cell lives: group (warp-cooperative groups first) and slot
struct ExpCells {
  const int64_t *cell_first;   // [n_cell + 1]
  const int32_t *cell_grp, *cell_slot;
  const GroupInfo *grp;        // warp-cooperative groups
  const ClassInfo *ccls;       //   and their classes (nodeoff_off into node_off)
  const int32_t *node_off;
  const TapeGroup *tgrp;       // interleaved groups
  const ExpClass *ecls;        //   and their classes
  const uint32_t *row;
  int32_t n_cell, n_cgroup;
  int64_t n_ab;
};

__device__ __forceinline__ int32_t exp_cell_of(const ExpCells &C, int64_t node) {
  int32_t lo = 0, hi = C.n_cell;  // the cell with cell_first[c] <= node < cell_first[c + 1]
  while (hi - lo > 1) {
    const int32_t mid = (lo + hi) >> 1;
    if (C.cell_first[mid] <= node) lo = mid; else hi = mid;
  }
  return lo;
}

// caller node -> element of the voltage arena (the table cn_layout.hpp computes on the host;
// written here so that 8 B per node need not cross PCIe)
__global__ void expand_node_pos_kernel(ExpCells C, int64_t n_node, int64_t *__restrict__ node_pos) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_node) return;
  const int32_t c = exp_cell_of(C, i);
  const int32_t g = C.cell_grp[c], slot = C.cell_slot[c];
  const int32_t local = (int32_t)(i - C.cell_first[c]);
  if (g < C.n_cgroup) {
    const GroupInfo gi = C.grp[g];
    node_pos[i] = gi.ab_base + C.node_off[C.ccls[gi.cls].nodeoff_off + local] + slot;
  } else {
    const TapeGroup tg = C.tgrp[g - C.n_cgroup];
    node_pos[i] = C.n_ab + tg.tape_base + ((int64_t)C.row[C.ecls[tg.cls].node_off + local] + 4) * 32 + slot;
  }
}

struct ExpTables {
  const ExpClass *cls;       // [n_class]
  const uint32_t *row;       // [node_off + j]: first tape row of the record of local node j
  const int32_t *par;        // local parent (-1: root)
  const int32_t *vcopy;      // row of the copy of v at the head of the mechanism record, or -1
  const int32_t *cai;        // row of cai, or -1
  const int32_t *ch_first;   // [chf_off + j]: children of j (ascending index) in ch[]
  const int32_t *ch;         // [child_off + ...]
  const TapeGroup *tgrp;
  const int32_t *cell_of_pcell;
  const int64_t *cell_first;
  const double *cm, *ri, *area, *cai0;
  double *tape;
  double dt, v_init;
};

__device__ __forceinline__ double exp_invc(double cm, double dt) {
  return __ddiv_rn(1.0, __ddiv_rn(__dmul_rn(1e-3, cm), dt));
}

// one CTA per interleaved group, lane = cell, the warps share the nodes: a', b', the raw diagonal
// (before the passive conductances), v, the copies of v and cai.  The arena was zeroed before.
__global__ void __launch_bounds__(256) expand_static_kernel(ExpTables E) {
  const TapeGroup tg = E.tgrp[blockIdx.x];
  const ExpClass K = E.cls[tg.cls];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const bool real = lane < tg.ncell;
  const int64_t f = real ? E.cell_first[E.cell_of_pcell[tg.cell_base + lane]] : 0;
  double *T = E.tape + tg.tape_base + lane;
  const int32_t *chf = E.ch_first + K.chf_off;
  for (int j = w; j < K.n; j += nw) {
    double *rec = T + ((int64_t)E.row[K.node_off + j] + 4) * 32;
    const int32_t vc = E.vcopy[K.node_off + j], cr = E.cai[K.node_off + j];
    if (vc >= 0) T[(int64_t)vc * 32] = E.v_init;  // (idle lanes too)
    if (!real) {
      rec[-2 * 32] = 1.0;  // unit diagonal, everything else zero
      continue;
    }
    const int64_t i = f + j;
    const double c = __ddiv_rn(__dmul_rn(1e-3, E.cm[i]), E.dt);
    const double invc = __ddiv_rn(1.0, c);
    const double ar = E.area[i];
    double d = c, an = 0.0, bn = 0.0;
    const int32_t p = E.par[K.node_off + j];
    if (p >= 0) {
      const double r = E.ri[i];
      const double b = __ddiv_rn(-100.0, __dmul_rn(r, ar));
      const double a = __ddiv_rn(-100.0, __dmul_rn(r, E.area[f + p]));
      d = __dsub_rn(d, b);
      bn = __dmul_rn(b, invc);
      an = __dmul_rn(a, exp_invc(E.cm[f + p], E.dt));
    }
    for (int32_t q = chf[j]; q < chf[j + 1]; ++q) {
      const int64_t ci = f + E.ch[K.child_off + q];
      d = __dsub_rn(d, __ddiv_rn(-100.0, __dmul_rn(E.ri[ci], ar)));
    }
    rec[-4 * 32] = an;
    rec[-3 * 32] = bn;
    rec[-2 * 32] = d;
    rec[0] = E.v_init;
    if (cr >= 0) T[(int64_t)cr * 32] = E.cai0[i];
  }
}

// passive conductances of one table (at most one instance of a table per node): d += g, r += g e
__global__ void expand_pas_kernel(const int32_t *node, const double *param, int64_t n,
                                  const int64_t *node_pos, int64_t n_ab, double *v) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int64_t pos = node_pos[node[i]];
  if (pos < n_ab) return;  // a warp-cooperative cell: folded on the host
  const double g = param[i], e = param[n + i];
  v[pos - 64] = __dadd_rn(v[pos - 64], g);
  v[pos - 32] = __dadd_rn(v[pos - 32], __dmul_rn(g, e));
}

// d' = d / c, r' = r / c of every real lane
__global__ void __launch_bounds__(256) expand_norm_kernel(ExpTables E) {
  const TapeGroup tg = E.tgrp[blockIdx.x];
  const ExpClass K = E.cls[tg.cls];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if (lane >= tg.ncell) return;
  const int64_t f = E.cell_first[E.cell_of_pcell[tg.cell_base + lane]];
  double *T = E.tape + tg.tape_base + lane;
  for (int j = w; j < K.n; j += nw) {
    double *rec = T + ((int64_t)E.row[K.node_off + j] + 4) * 32;
    const double invc = exp_invc(E.cm[f + j], E.dt);
    rec[-2 * 32] = __dmul_rn(rec[-2 * 32], invc);
    rec[-1 * 32] = __dmul_rn(rec[-1 * 32], invc);
  }
}

// the records of one distributed table on the tapes: the caller's parameter rows, 1 / c of the
// node, the initial states (the same for every instance, or per instance from `s_inst`)
struct ExpMech {
  const int32_t *node;
  const double *param;     // [n_param][n] as the caller gave them
  const int32_t *tab_row;  // [class node_off + local node]: first row of the table's block, or -1
  const double *s_inst;    // [n_state][n] or NULL
  int64_t n;
  int32_t n_param, n_state;
  double s[CN_MAX_STATE];
};

__global__ void expand_mech_kernel(ExpMech X, ExpCells C, const double *cm, double dt, double *tape) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= X.n) return;
  const int64_t node = X.node[i];
  const int32_t c = exp_cell_of(C, node);
  const int32_t g = C.cell_grp[c];
  if (g < C.n_cgroup) return;  // a warp-cooperative cell: its instances live in the table arrays
  const TapeGroup tg = C.tgrp[g - C.n_cgroup];
  const int32_t r = X.tab_row[C.ecls[tg.cls].node_off + (int32_t)(node - C.cell_first[c])];
  if (r < 0) return;
  double *rec = tape + tg.tape_base + (int64_t)r * 32 + C.cell_slot[c];
  for (int j = 0; j < X.n_param; ++j) rec[(int64_t)j * 32] = X.param[(int64_t)j * X.n + i];
  rec[(int64_t)X.n_param * 32] = exp_invc(cm[node], dt);
  for (int j = 0; j < X.n_state; ++j)
    rec[(int64_t)(X.n_param + 1 + j) * 32] = X.s_inst ? X.s_inst[(int64_t)j * X.n + i] : X.s[j];
}

}  // namespace cn
