// cn_finalize.hpp -- finalize(): the part of the set-up that needs dt (first cn_run): row-normalised
// static rows, tapes, mechanism tables, NetCon tables, window buffers, uploads.  Included by
// cn_api.cu only.
#pragma once

// ---------------------------------------------------------------------------------------------
// first cn_run: dt-dependent constants (row-normalised system), initial states, upload
// ---------------------------------------------------------------------------------------------

// Elimination plan of the on-chip window kernel (cn_cell.cuh) for one class: the tree is cut into
// CHAINS, maximal unbranched paths x0 -> parent(x0) -> ... -> xk (x0 a leaf or a branch point,
// every later node with exactly one child); one thread eliminates a whole chain with the
// contribution travelling in registers.  A chain may start once all chains that end at the
// children of x0 are done: its LEVEL.  The chains of a level run side by side, one barrier per
// level; sibling contributions are summed by the parent's chain in a fixed order.  PLAN ORDER:
// chains sorted by level (longest first), the nodes of a chain side by side in elimination
// order, the root last; `perm` maps a local node to its position.
struct CellPlan {
  std::vector<CellSeg> segs;
  std::vector<uint16_t> child, dist;
  std::vector<int32_t> lvl, noff;
};

static void build_cell_plan(const cn_model *m, const HClass &K, int kc, CellClass &cc, CellPlan &P,
                            std::vector<uint16_t> &perm) {
  const int n = K.n;
  const int64_t f = m->cell_first[K.rep_cell];
  std::vector<int32_t> par(n, -1);
  std::vector<std::vector<int>> ch(n);
  for (int i = 1; i < n; ++i) {
    par[i] = (int32_t)(m->parent[f + i] - f);
    ch[par[i]].push_back(i);
  }
  struct Tmp { std::vector<int> nd; int level, par, x0; };
  std::vector<Tmp> tmp;
  std::vector<int> end_level(n, -1);  // level of the chain that ends at this node
  for (int x = n - 1; x >= 1; --x) {  // (children carry larger indices than their parents)
    if (ch[x].size() == 1) continue;  // interior of a chain
    Tmp t;
    t.x0 = x;
    t.level = 0;
    for (int c : ch[x]) t.level = std::max(t.level, end_level[c] + 1);
    int cur = x;
    t.nd.push_back(cur);
    while (par[cur] != 0 && ch[par[cur]].size() == 1) {
      cur = par[cur];
      t.nd.push_back(cur);
    }
    t.par = par[cur];
    end_level[cur] = t.level;
    tmp.push_back(std::move(t));
  }
  std::stable_sort(tmp.begin(), tmp.end(), [](const Tmp &a, const Tmp &b) {
    if (a.level != b.level) return a.level < b.level;
    return a.nd.size() > b.nd.size();
  });
  perm.assign(n, 0);
  int pos = 0;
  for (const Tmp &t : tmp)
    for (int x : t.nd) perm[x] = (uint16_t)pos++;
  perm[0] = (uint16_t)(n - 1);
  int nlev = 0;
  for (const Tmp &t : tmp) nlev = std::max(nlev, t.level + 1);
  cc.seg_off = (int32_t)P.segs.size();
  cc.n_seg = (int32_t)tmp.size();
  cc.n_lev = nlev;
  cc.lvl_off = (int32_t)P.lvl.size();
  cc.child_off = (int32_t)P.child.size();
  size_t li = 0;
  for (int L = 0; L <= nlev; ++L) {
    while (li < tmp.size() && tmp[li].level < L) ++li;
    P.lvl.push_back((int32_t)li);
  }
  for (const Tmp &t : tmp) {
    CellSeg sg{};
    sg.first = perm[t.nd[0]];
    sg.len = (uint16_t)t.nd.size();
    sg.nchild = (uint16_t)ch[t.x0].size();
    sg.par = perm[t.par];
    sg.child_off = (uint32_t)(P.child.size() - (size_t)cc.child_off);
    for (int c : ch[t.x0]) P.child.push_back(perm[c]);
    P.segs.push_back(sg);
  }
  cc.root_child_off = (int32_t)(P.child.size() - (size_t)cc.child_off);
  cc.root_nchild = (int32_t)ch[0].size();
  for (int c : ch[0]) P.child.push_back(perm[c]);
  cc.n_child = (int32_t)(P.child.size() - (size_t)cc.child_off);
  // where a position lives in the schedule-ordered arrays in HBM
  cc.noff_off = (int32_t)P.noff.size();
  P.noff.resize(P.noff.size() + (size_t)n);
  for (int x = 0; x < n; ++x) P.noff[(size_t)cc.noff_off + perm[x]] = K.node_off[x];
  // node positions of the instances of every distributed table (instance order of the class)
  cc.dist_base = (int32_t)P.dist.size();
  for (size_t t = 0; t < m->tab.size(); ++t) {
    const HTable &T = m->tab[t];
    cc.dist_off[t] = (int32_t)(P.dist.size() - (size_t)cc.dist_base);
    if (T.ti.point || T.type == CN_PAS) continue;
    const int32_t *nodes = m->dist_nodes.data() + T.cls_nodeoff[kc];
    for (int j = 0; j < T.cls_cnt[kc]; ++j) P.dist.push_back(perm[nodes[j]]);
  }
  cc.n_dist = (int32_t)(P.dist.size() - (size_t)cc.dist_base);
}

// ---------------------------------------------------------------------------------------------
// interleaved groups: the tapes are expanded on the device (cn_expand.cuh)
// ---------------------------------------------------------------------------------------------

// the caller's compact arrays -> device; arrays that are there already are left alone.  Runs on a
// thread of cn_model_create (from the caller's arrays) and, for what is still missing, in
// finalize() (from the model's copies).  Errors go to RawDev::err (fail() is per thread).
static void raw_upload(cn_model *m, int dev, int64_t N, const double *cm, const double *ri,
                       const double *area, const std::vector<RawSrc> &tabs) {
  RawDev &R = m->raw;
  if (cudaSetDevice(dev) != cudaSuccess) {
    R.err = cudaErrorInvalidDevice;
    return;
  }
  auto put = [&R](auto **dst, const auto *src, int64_t n) {
    if (*dst || R.err != cudaSuccess || R.cancel.load()) return;
    void *p = nullptr;
    cudaError_t e = cudaMalloc(&p, (size_t)std::max<int64_t>(n, 1) * sizeof(*src));
    if (e == cudaSuccess && n > 0)
      e = cudaMemcpy(p, src, (size_t)n * sizeof(*src), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
      if (p) cudaFree(p);
      R.err = e;
      return;
    }
    *dst = static_cast<std::remove_reference_t<decltype(*dst)>>(p);
  };
  put(&R.cm, cm, N);
  put(&R.ri, ri, N);
  put(&R.area, area, N);
  for (size_t t = 0; t < tabs.size(); ++t) {
    if (!tabs[t].want) continue;
    put(&R.node[t], tabs[t].node, tabs[t].n);
    put(&R.param[t], tabs[t].param, tabs[t].n * tabs[t].n_param);
  }
}

// initial states of an instance of a distributed table at v_init (nrn_init: every gate at its
// steady state)
static void dist_initial_states(const cn_model *m, const HTable &T, int32_t nd, double *S) {
  const double v = m->v_init;
  switch (T.type) {
    case CN_HH: {
      double al, be;
      al = 0.1 * h_vtrap(-(v + 40.0), 10.0); be = 4.0 * std::exp(-(v + 65.0) / 18.0);
      S[0] = al / (al + be);
      al = 0.07 * std::exp(-(v + 65.0) / 20.0); be = 1.0 / (std::exp(-(v + 35.0) / 10.0) + 1.0);
      S[1] = al / (al + be);
      al = 0.01 * h_vtrap(-(v + 55.0), 10.0); be = 0.125 * std::exp(-(v + 65.0) / 80.0);
      S[2] = al / (al + be);
      break;
    }
    case CN_HHFORM:
      S[0] = 1.0 / (1.0 + std::exp((T.glob[4] - v) / T.glob[5]));
      S[1] = 1.0 / (1.0 + std::exp((T.glob[10] - v) / T.glob[11]));
      break;
    case CN_SK: {
      double ca = m->any_cai ? m->cai0[nd] : 1e-4;
      if (ca < 1e-9) ca = 1e-9;
      S[0] = 1.0 / (1.0 + std::pow(T.glob[1] / ca, T.glob[2]));
      break;
    }
    default: break;
  }
}

template <class T, class A>
static int tmp_upload(cn_model *m, const std::vector<T, A> &h, const T **out) {
  void *p = nullptr;
  CU(cudaMalloc(&p, std::max<size_t>(h.size(), 1) * sizeof(T)));
  m->raw.tmp.push_back(p);
  if (!h.empty()) CU(cudaMemcpy(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
  *out = static_cast<const T *>(p);
  return CN_OK;
}

#define TUP(vec, ptr)                                  \
  do {                                                 \
    rc = tmp_upload(m, vec, &ptr);                     \
    if (rc != CN_OK) return rc;                        \
  } while (0)

// Layout tables of the set-up kernels (cn_expand.cuh): per class with interleaved groups the tape
// rows, local parents and children (ascending) of every node; per caller cell its group and slot.
// m->hm.grp / cls / node_off / tgrp must be on the device.  The arrays are temporary (RawDev::tmp).
static int exp_layout_tables(cn_model *m, ExpTables &E, ExpCells &C, std::vector<ExpClass> &ec) {
  ec.assign(m->cls.size(), ExpClass{0, 0, 0, 0});
  std::vector<uint32_t> row;
  std::vector<int32_t> par, vcopy, cai, chf, ch;
  std::vector<int32_t> fill;
  for (size_t kc = 0; kc < m->cls.size(); ++kc) {
    const HClass &K = m->cls[kc];
    const HTape &P = K.tp;
    if (P.n_groups == 0) continue;
    ec[kc] = ExpClass{K.n, (int32_t)row.size(), (int32_t)ch.size(), (int32_t)chf.size()};
    const int64_t f = m->cell_first[K.rep_cell];
    const size_t chf0 = chf.size(), ch0 = ch.size();
    chf.resize(chf0 + (size_t)K.n + 1, 0);
    for (int j = 0; j < K.n; ++j) {
      const int32_t p = j ? (int32_t)(m->parent[f + j] - f) : -1;
      row.push_back(P.row[P.pos_of[j]]);
      par.push_back(p);
      if (p >= 0) chf[chf0 + (size_t)p + 1]++;
      vcopy.push_back((size_t)j < P.vcopy_row.size() ? P.vcopy_row[j] : -1);
      cai.push_back(m->any_cai && (size_t)j < P.cai_row.size() ? P.cai_row[j] : -1);
    }
    for (int j = 0; j < K.n; ++j) chf[chf0 + (size_t)j + 1] += chf[chf0 + (size_t)j];
    ch.resize(ch0 + (size_t)std::max(K.n - 1, 0));
    fill.assign(chf.begin() + (std::ptrdiff_t)chf0, chf.begin() + (std::ptrdiff_t)(chf0 + (size_t)K.n));
    for (int j = 1; j < K.n; ++j) ch[ch0 + (size_t)fill[par[par.size() - (size_t)K.n + (size_t)j]]++] = j;
  }
  int rc;
  TUP(ec, E.cls); TUP(row, E.row); TUP(par, E.par); TUP(vcopy, E.vcopy); TUP(cai, E.cai);
  TUP(chf, E.ch_first); TUP(ch, E.ch);
  TUP(m->cell_first, E.cell_first);
  E.tgrp = m->hm.tgrp;
  C.cell_first = E.cell_first;
  TUP(m->cell_grp, C.cell_grp); TUP(m->cell_slot, C.cell_slot);
  C.grp = m->hm.grp;
  C.ccls = m->hm.cls;
  C.node_off = m->hm.node_off;
  C.tgrp = m->hm.tgrp;
  C.ecls = E.cls;
  C.row = E.row;
  C.n_cell = m->n_cell;
  C.n_cgroup = m->n_cgroup;
  C.n_ab = m->n_ab;
  return CN_OK;
}

// Fills the tapes (already zeroed) of all interleaved groups; m->hm.tgrp, m->d_node_pos and the
// arena must be on the device.  Asynchronous on the legacy default stream: finalize() synchronises
// at its end and releases the temporary arrays.
static int expand_tapes(cn_model *m, double dt, ExpTables E, const ExpCells &C,
                        const std::vector<ExpClass> &ec, const std::vector<int32_t> &cell_of_pcell) {
  const int nt = (int)m->tab.size();
  int dev = 0;
  CU(cudaGetDevice(&dev));
  RawDev &R = m->raw;
  if (R.err != cudaSuccess) {  // the early upload failed: once more, from the model's copies
    for (double **p : {&R.cm, &R.ri, &R.area})
      if (*p) { cudaFree(*p); *p = nullptr; }
    for (double *&p : R.param)
      if (p) { cudaFree(p); p = nullptr; }
    for (int32_t *&p : R.node)
      if (p) { cudaFree(p); p = nullptr; }
    R.err = cudaSuccess;
  }
  R.cancel.store(false);
  if (R.param.empty()) {
    R.param.assign((size_t)nt, nullptr);
    R.node.assign((size_t)nt, nullptr);
  }
  std::vector<RawSrc> src((size_t)nt);
  for (int t = 0; t < nt; ++t) {
    const HTable &T = m->tab[t];
    src[t] = RawSrc{T.node.data(), T.param.data(), T.n, T.ti.n_param,
                    !T.ti.point && T.ti.n_param > 0 && T.n > 0};
  }
  for (int t = 0; t < nt; ++t)
    if (src[t].want && !R.param[t] && m->tab[t].param.empty())
      return fail(CN_ERR_ARG, "internal: the parameters of table %d are neither on the device nor on the host", t);
  if (!m->node_arrays_host && !(R.cm && R.ri && R.area))
    return fail(CN_ERR_ARG, "internal: the node arrays are neither on the device nor on the host");
  raw_upload(m, dev, m->N, m->cm.data(), m->ri.data(), m->area.data(), src);
  if (R.err != cudaSuccess)
    return fail(R.err == cudaErrorMemoryAllocation ? CN_ERR_NOMEM : CN_ERR_CUDA,
                "upload of the model arrays failed: %s", cudaGetErrorString(R.err));
  int rc;
  TUP(cell_of_pcell, E.cell_of_pcell);
  E.cai0 = nullptr;
  if (m->any_cai) TUP(m->cai0, E.cai0);
  E.cm = R.cm; E.ri = R.ri; E.area = R.area;
  E.tape = m->d_v + m->n_ab;
  E.dt = dt;
  E.v_init = m->v_init;
  const int ntg = (int)m->tgrp.size();
  expand_static_kernel<<<ntg, 256>>>(E);
  for (int t = 0; t < nt; ++t) {  // (table after table: the order of the sums is part of the result)
    const HTable &T = m->tab[t];
    if (T.type != CN_PAS || T.n == 0) continue;
    expand_pas_kernel<<<(unsigned)((T.n + 255) / 256), 256>>>(R.node[t], R.param[t], T.n,
                                                              m->d_node_pos, m->n_ab, m->d_v);
  }
  expand_norm_kernel<<<ntg, 256>>>(E);
  for (int t = 0; t < nt; ++t) {
    const HTable &T = m->tab[t];
    if (T.ti.point || T.n == 0 || tape_rows_of(T.ti, T.type) == 0) continue;
    // first row of the table's block per (class, local node)
    std::vector<int32_t> tab_row;
    bool any = false;
    for (size_t kc = 0; kc < m->cls.size(); ++kc) {
      const HClass &K = m->cls[kc];
      if (K.tp.n_groups == 0) continue;
      tab_row.resize((size_t)ec[kc].node_off + (size_t)K.n, -1);
      if ((size_t)t >= K.tp.tab_row.size() || K.tp.tab_row[t].empty()) continue;
      for (int j = 0; j < K.n; ++j) {
        tab_row[(size_t)ec[kc].node_off + (size_t)j] = K.tp.tab_row[t][j];
        any = any || K.tp.tab_row[t][j] >= 0;
      }
    }
    if (!any) continue;
    ExpMech X{};
    X.node = R.node[t];
    X.param = R.param[t];
    X.n = T.n;
    X.n_param = T.ti.n_param;
    X.n_state = T.ti.n_state;
    TUP(tab_row, X.tab_row);
    X.s_inst = nullptr;
    if (T.type == CN_SK) {  // the one type whose initial state depends on the node (cai)
      uvec<double> s((size_t)T.n * T.ti.n_state);
      par_for(T.n, 1 << 14, [&](int64_t i0, int64_t i1) {
        for (int64_t i = i0; i < i1; ++i) {
          double S[CN_MAX_STATE] = {0.0};
          dist_initial_states(m, T, T.node[i], S);
          for (int j = 0; j < T.ti.n_state; ++j) s[(size_t)j * T.n + i] = S[j];
        }
      });
      TUP(s, X.s_inst);
    } else {
      dist_initial_states(m, T, -1, X.s);
    }
    expand_mech_kernel<<<(unsigned)((T.n + 255) / 256), 256>>>(X, C, R.cm, dt, m->d_v + m->n_ab);
  }
  CU(cudaGetLastError());
  return CN_OK;
}
#undef TUP

static int finalize(cn_model *m, double dt) {
  const bool dbg = m->opt("debug") && std::atoi(m->opt("debug")) != 0;
  auto t_prev = std::chrono::steady_clock::now();
  auto lap = [&](const char *what) {
    if (!dbg) return;
    const auto t = std::chrono::steady_clock::now();
    fprintf(stderr, "[cn] finalize %-32s %7.1f ms\n", what,
            std::chrono::duration<double, std::milli>(t - t_prev).count());
    t_prev = t;
  };
  const int64_t N = m->N;
  const int nt = (int)m->tab.size();
  const int ng = (int)m->grp.size();
  int dev_count = 0;
  if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0)
    return fail(CN_ERR_CUDA, "no CUDA device: libcn has no CPU fallback");
  // delays
  std::vector<int32_t> dsteps((size_t)m->n_netcon);
  int64_t mind = INT32_MAX, maxd = 1;
  for (int64_t i = 0; i < m->n_netcon; ++i) {
    const long long ds = llround(m->nc_delay[i] / dt);
    if (ds < 1) return fail(CN_ERR_NETCON, "netcon %lld: delay %.6g ms is < 1 step of %.6g ms",
                            (long long)i, m->nc_delay[i], dt);
    if (ds > 1000000) return fail(CN_ERR_NETCON, "netcon %lld: delay too long", (long long)i);
    dsteps[i] = (int32_t)ds;
    mind = std::min<int64_t>(mind, ds);
    maxd = std::max<int64_t>(maxd, ds);
  }
  if (m->n_netcon == 0) mind = 1;
  // Row-normalised static arrays of the WARP-COOPERATIVE groups (the tapes of the interleaved groups
  // are expanded on the device from the compact arrays, cn_expand.cuh: same operations, same order):
  //   c_i = 1e-3 cm_i/dt,  b' = b/c_i,  a' = a/c_parent,
  //   dstat = (c - b - sum_children a + sum static g)/c,  rstat = (sum static g*e)/c
  const bool host_rows = m->n_cgroup > 0;
  const int64_t NH = host_rows ? N : 0;
  uvec<double> invc((size_t)NH), bn((size_t)NH), an((size_t)NH);
  uvec<double> dstat((size_t)m->n_pnode), rstat((size_t)m->n_pnode);
  par_for(m->n_pnode, 1 << 20, [&](int64_t i0, int64_t i1) {
    std::fill(dstat.begin() + i0, dstat.begin() + i1, 1.0);
    std::fill(rstat.begin() + i0, rstat.begin() + i1, 0.0);
  });
  uvec<double> v0((size_t)m->n_ab);  // schedule-ordered v of the cooperative groups
  uvec<double> dsum((size_t)NH), rsum((size_t)NH);
  uvec<int32_t> cell_of_node((size_t)NH);
  par_for((int64_t)v0.size(), 1 << 20, [&](int64_t i0, int64_t i1) {
    std::fill(v0.begin() + i0, v0.begin() + i1, 0.0);
  });
  par_for(NH, 1 << 20, [&](int64_t i0, int64_t i1) {
    std::fill(bn.begin() + i0, bn.begin() + i1, 0.0);
    std::fill(an.begin() + i0, an.begin() + i1, 0.0);
    std::fill(rsum.begin() + i0, rsum.begin() + i1, 0.0);
  });
  // cells are independent (a parent sits in the same cell): all host cores
  if (host_rows)
   par_for(m->n_cell, 256, [&](int64_t c0, int64_t c1) {
    const int64_t i0 = m->cell_first[c0], i1 = m->cell_first[c1];
    for (int64_t c = c0; c < c1; ++c)
      for (int64_t i = m->cell_first[c]; i < m->cell_first[c + 1]; ++i) cell_of_node[i] = (int32_t)c;
    for (int64_t i = i0; i < i1; ++i) {
      const double c = 1e-3 * m->cm[i] / dt;
      invc[i] = 1.0 / c;
      dsum[i] = c;
    }
    for (int64_t i = i0; i < i1; ++i) {
      const int32_t p = m->parent[i];
      if (p >= 0) {
        const double b = -100.0 / (m->ri[i] * m->area[i]);
        const double a = -100.0 / (m->ri[i] * m->area[p]);
        dsum[i] -= b;
        dsum[p] -= a;
        bn[i] = b * invc[i];
        an[i] = a * invc[p];
      }
    }
   });
  if (host_rows)
   for (const HTable &T : m->tab)
    if (T.type == CN_PAS)  // (at most one instance of a table per node: no two threads meet)
      par_for(T.n, 65536, [&](int64_t q0, int64_t q1) {
        for (int64_t i = q0; i < q1; ++i) {
          const double g = T.param[i], e = T.param[T.n + i];
          dsum[T.node[i]] += g;
          rsum[T.node[i]] += g * e;
        }
      });
  // a caller node that sits on a tape (node_pos: element of the arena, the tapes come last)
  auto on_tape = [&](int64_t i) { return m->node_pos[i] >= m->n_ab; };
  // inverse map: (group, slot) -> caller cell
  std::vector<int32_t> cell_of_pcell((size_t)m->n_pcell, -1);
  for (int32_t c = 0; c < m->n_cell; ++c) {
    const int g = m->cell_grp[c];
    const int32_t cb = g < m->n_cgroup ? m->grp[g].cell_base : m->tgrp[g - m->n_cgroup].cell_base;
    cell_of_pcell[cb + m->cell_slot[c]] = c;
  }
  if (host_rows)
    par_for(N, 65536, [&](int64_t i0, int64_t i1) {
      for (int64_t i = i0; i < i1; ++i) {
        if (on_tape(i)) continue;
        const int64_t q = m->node_pos[i];
        dstat[q] = dsum[i] * invc[i];
        rstat[q] = rsum[i] * invc[i];
        v0[q] = m->v_init;
      }
    });
  lap("static rows");
  // schedule-ordered off-diagonals
  uvec<double> a_s((size_t)m->n_ab), b_s((size_t)m->n_ab);
  par_for(m->n_ab, 1 << 20, [&](int64_t i0, int64_t i1) {
    std::fill(a_s.begin() + i0, a_s.begin() + i1, 0.0);
    std::fill(b_s.begin() + i0, b_s.begin() + i1, 0.0);
  });
  std::vector<uint32_t> sched_all;
  std::vector<int32_t> nodeoff_all;
  std::vector<ClassInfo> cinfo(m->cls.size());
  for (size_t kc = 0; kc < m->cls.size(); ++kc) {
    const HClass &K = m->cls[kc];
    cinfo[kc] = ClassInfo{K.n, K.G, K.lgG, K.rounds, K.sched_off, K.needs_ica, K.nodeoff_off, 0};
    sched_all.insert(sched_all.end(), K.sched.begin(), K.sched.end());
    nodeoff_all.insert(nodeoff_all.end(), K.node_off.begin(), K.node_off.end());
  }
  par_for(ng, 64, [&](int64_t g0, int64_t g1) {  // (every group writes its own slots)
   for (int64_t g = g0; g < g1; ++g) {
    const GroupInfo &gi = m->grp[g];
    const HClass &K = m->cls[gi.cls];
    const int P = 32 / K.G;
    for (int c = 0; c < gi.ncell; ++c) {
      const int32_t cell = cell_of_pcell[gi.cell_base + c];
      const int64_t f = m->cell_first[cell];
      for (int r = 0; r < K.rounds; ++r)
        for (int p = 0; p < P; ++p) {
          const uint32_t e = K.sched[(size_t)r * P + p];
          if ((e & 0xFFFFu) == CN_IDLE) continue;
          const int64_t i = f + (e & 0xFFFFu);
          const int64_t pos = gi.ab_base + (int64_t)r * 32 + p * K.G + c;
          a_s[pos] = an[i];
          b_s[pos] = bn[i];
        }
    }
   }
  });
  lap("coop schedule arrays");
  // thresholds, flags, gids per permuted cell
  std::vector<double> thr((size_t)m->n_pcell, 0.0);
  std::vector<unsigned char> flag((size_t)m->n_pcell, 0);
  std::vector<int32_t> gid_of((size_t)m->n_pcell, -1);
  par_for(m->n_pcell, 1 << 14, [&](int64_t p0, int64_t p1) {
    for (int64_t pc = p0; pc < p1; ++pc) {
      const int32_t c = cell_of_pcell[pc];
      if (c < 0) continue;
      thr[pc] = m->thr[c];
      flag[pc] = m->v_init > m->thr[c];
      gid_of[pc] = c;
    }
  });
  // cai per node of the cooperative groups
  std::vector<double> cai;
  if (m->any_cai) {
    cai.assign((size_t)m->n_pnode, 1e-4);
    par_for(N, 1 << 16, [&](int64_t i0, int64_t i1) {
      for (int64_t i = i0; i < i1; ++i)
        if (!on_tape(i)) cai[m->node_pos[i]] = m->cai0[i];
    });
  }

  DModel &H = m->hm;
  H.warp_smem_doubles = m->warp_smem_doubles;
  H.dt = dt;
  H.celsius = m->celsius;
  H.q10 = std::pow(3.0, (m->celsius - 6.3) / 10.0);
  int rc;
#define UP(vec, ptr)                                            \
  do {                                                          \
    rc = dev_upload(m, vec, &ptr);                              \
    if (rc != CN_OK) return rc;                                 \
  } while (0)
  {
    GroupInfo *dg; ClassInfo *dc; uint32_t *ds; int32_t *dn;
    UP(m->grp, dg); UP(cinfo, dc); UP(sched_all, ds); UP(m->dist_nodes, dn);
    H.grp = dg; H.cls = dc; H.sched = ds; H.dist_nodes = dn;
    int32_t *dno; UP(nodeoff_all, dno); H.node_off = dno;
    double *p;
    // nodes of warp-cooperative cells that carry point processes: negative static diagonal
    // (one pass per node, not per instance: several point processes may share a node)
    if (m->n_cgroup > 0) {
      std::vector<uint8_t> has_pp((size_t)N, 0);
      for (const HTable &T : m->tab)
        if (T.ti.point)
          par_for(T.n, 1 << 16, [&](int64_t i0, int64_t i1) {
            for (int64_t i = i0; i < i1; ++i) has_pp[T.node[i]] = 1;  // (all writers store 1)
          });
      par_for(N, 1 << 16, [&](int64_t i0, int64_t i1) {
        for (int64_t i = i0; i < i1; ++i)
          if (has_pp[i] && !on_tape(i)) {
            double &d = dstat[m->node_pos[i]];
            d = -std::fabs(d);
          }
      });
    }
    UP(dstat, p); H.dstat = p;
    H.ppdr = nullptr;
    {  // point processes on warp-cooperative groups: their conductance / current rows
      bool any = false;
      for (const HTable &T : m->tab)
        if (T.ti.point && T.pp_tape_begin > 0) any = true;
      if (any) {
        rc = dev_alloc(m, (size_t)(2 * m->n_pnode + 64), &H.ppdr);
        if (rc != CN_OK) return rc;
      }
    }
    UP(rstat, p); H.rstat = p;
    UP(a_s, p); H.a_s = p;
    UP(b_s, p); H.b_s = p;
    if (m->any_cai) { UP(cai, m->d_cai); H.cai = m->d_cai; } else H.cai = nullptr;
    UP(thr, p); H.thr = p;
    unsigned char *pf; UP(flag, pf); H.flag = pf;
    int32_t *pg; UP(gid_of, pg); H.gid_of_pcell = pg;
  }
  lap("small uploads");
  // mechanism tables
  for (int t = 0; t < nt; ++t) {
    HTable &T = m->tab[t];
    DTable &D = H.tab[t];
    memset(&D, 0, sizeof(D));
    D.type = T.type;
    D.is_point = T.ti.point;
    D.n_param = T.ti.n_dev_param;
    D.n_state = T.ti.n_state;
    for (size_t j = 0; j < T.glob.size(); ++j) D.glob[j] = T.glob[j];
    if (T.type == CN_AMPANMDA) {
      D.glob[7] = h_exp2_factor(T.glob[0], T.glob[1]);
      D.glob[8] = h_exp2_factor(T.glob[2], T.glob[3]);
      for (int c = 0; c < 4; ++c) D.glob[9 + c] = 1.0 - std::exp(-dt / T.glob[c]);  // cnexp factors
    }
    if (T.type == CN_PAS) continue;  // folded
    const int64_t nd = T.n_dev;
    std::vector<uvec<double>> par(T.ti.n_dev_param), st(T.ti.n_state);
    for (auto &x : par) x.resize((size_t)nd);
    for (auto &x : st) x.resize((size_t)nd);
    par_for(nd, 1 << 18, [&](int64_t i0, int64_t i1) {
      for (int j = 0; j < T.ti.n_dev_param; ++j)  // benign padding for distributed tables
        std::fill(par[j].begin() + i0, par[j].begin() + i1,
                  !T.ti.point && j == T.ti.n_dev_param - 1 ? 1.0 : 0.0);
      for (auto &x : st) std::fill(x.begin() + i0, x.begin() + i1, 0.0);
    });
    // instances are independent (each writes its own elements): all host cores.  (The instances
    // of a distributed table that live on tapes are written by expand_mech_kernel.)
    if (T.ti.point || nd > 0)
     par_for(T.n, 4096, [&](int64_t ii0, int64_t ii1) {
     for (int64_t i = ii0; i < ii1; ++i) {
      if (T.inst_pos[i] < 0 || (!T.ti.point && T.tape_loc[i] >= 0)) continue;
      const int32_t nd_i = T.node[i];
      double P[CN_MAX_PARAM] = {0.0}, S[CN_MAX_STATE] = {0.0};
      for (int j = 0; j < T.ti.n_param; ++j) P[j] = T.param[(size_t)j * T.n + i];
      // (node arrays off the host: every distributed instance is on a tape and was skipped above)
      const double cm_i = m->node_arrays_host ? m->cm[nd_i] : T.pp_cm[i];
      const double area_i = m->node_arrays_host ? m->area[nd_i] : T.pp_area[i];
      const double ic = 1.0 / (1e-3 * cm_i / dt);
      const double scale = 100.0 / area_i * ic;
      switch (T.type) {
        case CN_HH:
          P[4] = ic;
          dist_initial_states(m, T, nd_i, S);
          break;
        case CN_EXPSYN:  // tau -> the cnexp factor 1 - exp(-dt/tau) (the device never needs tau)
          P[2] = scale;
          P[0] = 1.0 - std::exp(-dt / P[0]);
          break;
        case CN_EXP2SYN:
          P[3] = scale;
          P[4] = h_exp2_factor(P[0], P[1]);
          P[0] = 1.0 - std::exp(-dt / P[0]);
          P[1] = 1.0 - std::exp(-dt / P[1]);
          break;
        case CN_ICLAMP: P[3] = scale; break;
        case CN_HHFORM:
        case CN_SK:
          P[1] = ic;
          dist_initial_states(m, T, nd_i, S);
          break;
        case CN_AMPANMDA: P[0] = scale; break;
        case CN_GAP:  // positions in the voltage arena (exact in a double: < 2^53)
          P[0] *= scale;
          P[1] = (double)m->node_pos[(int64_t)P[1]];
          break;
        default: break;
      }
      const int64_t q = T.inst_pos[i];
      for (int j = 0; j < T.ti.n_dev_param; ++j) par[j][q] = P[j];
      for (int j = 0; j < T.ti.n_state; ++j) st[j][q] = S[j];
     }
    });
    for (int j = 0; j < T.ti.n_dev_param; ++j) { UP(par[j], T.d_param[j]); D.param[j] = T.d_param[j]; }
    for (int j = 0; j < T.ti.n_state; ++j) { UP(st[j], T.d_state[j]); D.state[j] = T.d_state[j]; }
    if (T.ti.point) {
      UP(T.pp_first, T.d_pp_first); UP(T.pp_slot, T.d_pp_slot); UP(T.pp_wslot, T.d_pp_wslot);
      D.pp_first = T.d_pp_first; D.pp_slot = T.d_pp_slot; D.pp_wslot = T.d_pp_wslot;
      D.pp_goff = m->win_ninst;
      m->win_ninst += T.n;
    } else {
      UP(T.cls_cnt, T.d_cls_cnt); UP(T.cls_nodeoff, T.d_cls_nodeoff);
      UP(T.grp_instbase, T.d_grp_instbase);
      D.cls_cnt = T.d_cls_cnt; D.cls_nodeoff = T.d_cls_nodeoff; D.grp_instbase = T.d_grp_instbase;
    }
  }
  lap("mechanism tables");
  // the arena [schedule-ordered v of the cooperative groups | tapes of the interleaved groups] and
  // the programs; the tapes are expanded on the device once the group table is there (below)
  {
    {
      void *p = nullptr;
      CU(cudaMalloc(&p, (size_t)std::max<int64_t>(m->n_ab + m->n_tape, 1) * sizeof(double)));
      m->dev_allocs.push_back(p);
      m->d_v = static_cast<double *>(p);
      if (m->n_ab > 0)
        CU(cudaMemcpy(m->d_v, v0.data(), (size_t)m->n_ab * sizeof(double), cudaMemcpyHostToDevice));
      if (m->n_tape > 0)
        CU(cudaMemsetAsync(m->d_v + m->n_ab, 0, (size_t)m->n_tape * sizeof(double), 0));
    }
    H.v = m->d_v;
    H.tape = m->d_v + m->n_ab;
    std::vector<TapeClass> tcls(m->cls.size());
    std::vector<TapeTask> ttask(m->cls.size() * (size_t)m->tape_W);
    std::vector<uint4> prog;
    for (size_t kc = 0; kc < m->cls.size(); ++kc) {
      const HClass &K = m->cls[kc];
      const HTape &P = K.tp;
      tcls[kc] = TapeClass{K.n, P.prog_off, (int32_t)P.prog.size(), P.n_bar};
      if (P.n_groups == 0) continue;
      if ((int)prog.size() != P.prog_off) return fail(CN_ERR_ARG, "internal: program offsets");
      prog.insert(prog.end(), P.prog.begin(), P.prog.end());
      for (int w = 0; w < m->tape_W; ++w) {
        const HTask &Tk = P.task[w];
        // program positions are relative to the class's program (as it sits in shared memory)
        ttask[kc * (size_t)m->tape_W + w] =
            TapeTask{Tk.p0, Tk.p1, Tk.b0, Tk.b1, Tk.nchunk, Tk.tm_base, Tk.row0, Tk.head, Tk.nrows,
                     (uint32_t)Tk.pp0};
      }
    }
    TapeGroup *dtg; TapeClass *dtc; uint4 *dpg; TapeTask *dtt;
    UP(m->tgrp, dtg); UP(tcls, dtc); UP(prog, dpg); UP(ttask, dtt);
    H.tgrp = dtg; H.tcls = dtc; H.prog = dpg; H.ttask = dtt;
    lap("arena, programs");
    // caller node -> arena element on the device (cn_get_v, probes, the expansion): computed
    // there from the per-cell and per-class tables instead of uploading 8 B per node
    ExpTables E{};
    ExpCells C{};
    std::vector<ExpClass> ec;
    rc = exp_layout_tables(m, E, C, ec);
    if (rc != CN_OK) return rc;
    rc = dev_alloc(m, (size_t)std::max<int64_t>(N, 1), &m->d_node_pos, false);
    if (rc != CN_OK) return rc;
    if (N > 0) expand_node_pos_kernel<<<(unsigned)((N + 255) / 256), 256>>>(C, N, m->d_node_pos);
    lap("layout tables, node positions");
    if (m->n_tape > 0) {
      rc = expand_tapes(m, dt, E, C, ec, cell_of_pcell);
      if (rc != CN_OK) return rc;
    }
    H.tape_W = m->tape_W;
    H.tape_S = m->tape_S;
    H.tape_CH = m->tape_CH;
    H.tape_prog_cap = std::max(m->tape_prog_cap, 1);
    H.tape_sys_cap = std::max(m->tape_sys_cap, 1);
    H.tape_bar_cap = m->tape_bar_cap;
    H.tape_pf = 0;  // measured on config 4: prefetching ahead of the ring only costs (0: off)
    if (const char *e = m->opt("tape_pf")) H.tape_pf = std::max(0, std::min(4096, std::atoi(e)));
    for (int t = 0; t < nt; ++t) {
      H.tab[t].pp_tape_begin = m->tab[t].pp_tape_begin;
      H.tab[t].pp_tape_end = m->tab[t].ti.point ? m->tab[t].n : 0;
    }
  }
  // PAS tables still need (empty) layout pointers so the kernel's table loop can skip them
  for (int t = 0; t < nt; ++t) {
    HTable &T = m->tab[t];
    if (T.type != CN_PAS) continue;
    std::vector<int32_t> zc(m->cls.size(), 0);
    std::vector<int64_t> zg((size_t)ng, 0);
    UP(zc, T.d_cls_cnt); UP(zc, T.d_cls_nodeoff); UP(zg, T.d_grp_instbase);
    H.tab[t].cls_cnt = T.d_cls_cnt; H.tab[t].cls_nodeoff = T.d_cls_nodeoff;
    H.tab[t].grp_instbase = T.d_grp_instbase;
  }
  lap("tape expansion (launches)");
  // NetCons: CSR by source gid, sorted by delay steps (stable in caller order)
  {
    // (a stable counting sort by source on all cores, then every source's few NetCons by delay)
    std::vector<int64_t> src_first;
    uvec<int64_t> rank, order((size_t)m->n_netcon);
    par_bucket(m->n_netcon, m->n_src, [&](int64_t i) { return m->nc_src[i]; }, src_first, rank);
    par_for(m->n_netcon, 1 << 16, [&](int64_t i0, int64_t i1) {
      for (int64_t i = i0; i < i1; ++i) order[rank[i]] = i;
    });
    par_for(m->n_src, 1024, [&](int64_t s0, int64_t s1) {
      const auto by_delay = [&](int64_t x, int64_t y) { return dsteps[x] < dsteps[y]; };
      for (int64_t sg = s0; sg < s1; ++sg) {
        auto b = order.begin() + src_first[sg], e = order.begin() + src_first[sg + 1];
        if (!std::is_sorted(b, e, by_delay)) std::stable_sort(b, e, by_delay);
      }
    });
    uvec<int32_t> nd((size_t)m->n_netcon), ntab((size_t)m->n_netcon);
    uvec<int64_t> ninst((size_t)m->n_netcon);
    uvec<double> nw((size_t)m->n_netcon);
    par_for(m->n_netcon, 1 << 16, [&](int64_t j0, int64_t j1) {
      for (int64_t j = j0; j < j1; ++j) {
        const int64_t i = order[j];
        nd[j] = dsteps[i];
        ntab[j] = m->nc_tgt_mech[i];
        ninst[j] = m->tab[m->nc_tgt_mech[i]].inst_pos[m->nc_tgt_inst[i]];
        nw[j] = m->nc_w[i];
      }
    });
    lap("netcons: sort");
    {  // fixed-point scale of the event-weight sums: the largest sum of |w| on one synapse < 2^62
      std::vector<int64_t> toff(m->tab.size() + 1, 0);  // (point tables only: the others get no events)
      for (size_t t = 0; t < m->tab.size(); ++t)
        toff[t + 1] = toff[t] + (m->tab[t].ti.point ? m->tab[t].n : 0);
      std::vector<double> wsum((size_t)toff.back(), 0.0);
      for (int64_t i = 0; i < m->n_netcon; ++i)
        wsum[(size_t)(toff[m->nc_tgt_mech[i]] + m->nc_tgt_inst[i])] += std::fabs(m->nc_w[i]);
      double wmax = 1e-300;
      for (double x : wsum) wmax = std::max(wmax, x);
      int ex = 0;
      std::frexp(wmax, &ex);  // wmax < 2^ex
      ex = std::max(-400, std::min(400, ex));
      H.fxw_scale = std::ldexp(1.0, 62 - ex);
      H.fxw_inv = std::ldexp(1.0, ex - 62);
    }
    int64_t *p64; int32_t *p32; double *pd;
    UP(src_first, p64); H.src_first = p64;
    UP(nd, p32); H.nc_d = p32;
    UP(ntab, p32); H.nc_tab = p32;
    UP(ninst, p64); H.nc_inst = p64;
    UP(nw, pd); H.nc_w = pd;
    H.mind = (int32_t)mind;
    H.maxd = (int32_t)maxd;
    H.wr = (int32_t)(maxd + 2);
    rc = dev_alloc(m, (size_t)H.wr, &H.sp_end);
    if (rc != CN_OK) return rc;
    // scripted sources sorted by step
    const int64_t ns = (int64_t)m->stim_gid.size();
    std::vector<int64_t> sstep((size_t)ns), so((size_t)ns);
    for (int64_t i = 0; i < ns; ++i) sstep[i] = llround(m->stim_t[i] / dt);
    std::iota(so.begin(), so.end(), 0);
    std::stable_sort(so.begin(), so.end(), [&](int64_t x, int64_t y) { return sstep[x] < sstep[y]; });
    std::vector<int32_t> sg((size_t)ns);
    std::vector<int64_t> ss((size_t)ns);
    for (int64_t j = 0; j < ns; ++j) { sg[j] = m->stim_gid[so[j]]; ss[j] = sstep[so[j]]; }
    UP(sg, p32); H.stim_gid = p32;
    UP(ss, p64); H.stim_step = p64;
    H.n_stim = ns;
  }
  lap("netcons");
  // window mode: every cell on the interleaved kernel, no point process whose current depends on
  // v (AMPA+NMDA, gap junctions); a window is at most the smallest delay long (probes are
  // recorded by the kernel itself then)
  {
    bool ok = m->hm.n_tgroup > 0 && m->grp.empty();
    for (const HTable &T : m->tab)
      if ((T.type == CN_AMPANMDA || T.type == CN_GAP) && T.n > 0) ok = false;
    if (const char *e = m->opt("tape_window")) ok = ok && std::atoi(e) != 0;
    int64_t wn = m->n_netcon > 0 ? std::min<int64_t>(H.mind, 64) : 32;
    if (wn < 2) ok = false;
    if (ok && (m->win_stride + m->win_ninst) * wn * 8 > ((int64_t)4 << 30)) ok = false;
    m->window = ok;
    m->win_steps = (int)wn;
    H.win_stride = m->win_stride;
    H.win_ninst = m->win_ninst;
    if (ok) {
      rc = dev_alloc(m, (size_t)(m->win_stride * wn + 128), &H.win_rows);  // (+ prefetch overrun)
      if (rc != CN_OK) return rc;
      rc = dev_alloc(m, (size_t)std::max<int64_t>(m->win_ninst * wn, 1), &H.win_deliv);
      if (rc != CN_OK) return rc;
      rc = dev_alloc(m, (size_t)std::max<int64_t>(m->win_ninst, 1), &H.win_mask);
      if (rc != CN_OK) return rc;
      rc = dev_alloc(m, (size_t)m->hm.n_tgroup, &H.win_done); if (rc != CN_OK) return rc;
      rc = dev_alloc(m, 1, &H.win_ticket); if (rc != CN_OK) return rc;
      H.win_mark_cap = H.maxd + 64;
      rc = dev_alloc(m, (size_t)H.win_mark_cap, &H.win_mark_step); if (rc != CN_OK) return rc;
      rc = dev_alloc(m, (size_t)H.win_mark_cap, &H.win_mark_nsp); if (rc != CN_OK) return rc;
    }
  }
  // cell-window mode (cn_cell.cuh): every cell on the warp-cooperative layout with one
  // cell per warp, no gap junctions, the largest cell fits the shared memory of a CTA; chosen
  // automatically when the whole model is resident on the device at once, or forced by onchip=1
  {
    int onchip = -1;
    if (const char *e = m->opt("onchip")) onchip = std::atoi(e);
    bool ok = onchip != 0 && m->hm.n_tgroup == 0 && !m->grp.empty();
    for (const HClass &K : m->cls)
      if (K.count - K.tp.n_cells > 0 && K.G != 1) ok = false;
    for (const HTable &T : m->tab)
      if (T.type == CN_GAP && T.n > 0) ok = false;
    const int64_t wn = m->n_netcon > 0 ? std::min<int64_t>(H.mind, 64) : 32;
    if (wn < 2 && onchip != 1) ok = false;
    if (ok && m->win_ninst * wn * 8 > ((int64_t)4 << 30)) ok = false;
    std::vector<CellClass> ccls(m->cls.size());
    CellPlan plan;
    std::vector<std::vector<uint16_t>> perm(m->cls.size());  // local node -> plan position
    size_t max_bytes = 0;
    if (ok) {
      for (size_t kc = 0; kc < m->cls.size(); ++kc) {
        const HClass &K = m->cls[kc];
        int off = 0;
        for (int t = 0; t < nt; ++t) {
          const HTable &T = m->tab[t];
          ccls[kc].mech_off[t] = off;
          if (T.ti.point || T.type == CN_PAS) continue;
          off += (T.ti.n_dev_param + T.ti.n_state) * T.cls_cnt[kc];
        }
        ccls[kc].mech_doubles = off;
        if (K.count - K.tp.n_cells > 0) {
          CellClass &cc = ccls[kc];
          build_cell_plan(m, K, (int)kc, cc, plan, perm[kc]);
          const size_t plan_bytes = (size_t)cc.n_seg * sizeof(CellSeg) + (size_t)(cc.n_lev + 1) * 4 +
                                    (size_t)(cc.n_child + cc.n_dist) * 2 + 16;
          max_bytes = std::max(max_bytes, ((size_t)K.n * (9 + (K.needs_ica ? 1 : 0) + (m->any_cai ? 1 : 0)) + off) * 8 + plan_bytes);
        }
      }
      if (max_bytes > 220 * 1024) ok = false;
    }
    if (ok) {
      int dev = 0, sms = 0;
      CU(cudaGetDevice(&dev));
      CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
      int max_n = 1;
      for (const HClass &K : m->cls)
        if (K.count - K.tp.n_cells > 0) max_n = std::max(max_n, K.n);
      m->cwin_threads = max_n <= 128 ? 64 : max_n <= 320 ? 128 : 256;
      const int per_sm = (int)std::max<size_t>(
          1, std::min<size_t>(std::min(32, 2048 / m->cwin_threads), (227 * 1024) / (max_bytes + 1024)));
      if (onchip == -1 && ng > sms * per_sm) ok = false;  // auto: only when everything is resident at once
      m->cwin_grid = std::min(ng, sms * per_sm);
      m->cwin_smem = max_bytes;
    }
    m->cwindow = ok;
    if (ok) {
      m->win_steps = (int)std::max<int64_t>(wn, 1);
      H.win_stride = 0;
      H.win_ninst = m->win_ninst;
      if (m->n_netcon > 0) {
        rc = dev_alloc(m, (size_t)std::max<int64_t>(m->win_ninst * m->win_steps, 1), &H.win_deliv);
        if (rc != CN_OK) return rc;
      }
      H.win_mark_cap = H.maxd + 64;
      rc = dev_alloc(m, (size_t)H.win_mark_cap, &H.win_mark_step); if (rc != CN_OK) return rc;
      rc = dev_alloc(m, (size_t)H.win_mark_cap, &H.win_mark_nsp); if (rc != CN_OK) return rc;
      CellClass *dcc;
      rc = dev_upload(m, ccls, &dcc); if (rc != CN_OK) return rc;
      H.ccls = dcc;
      CellSeg *dsg; uint16_t *dsc, *dsd; int32_t *dsl, *dno;
      rc = dev_upload(m, plan.segs, &dsg); if (rc != CN_OK) return rc;
      rc = dev_upload(m, plan.child, &dsc); if (rc != CN_OK) return rc;
      rc = dev_upload(m, plan.dist, &dsd); if (rc != CN_OK) return rc;
      rc = dev_upload(m, plan.lvl, &dsl); if (rc != CN_OK) return rc;
      rc = dev_upload(m, plan.noff, &dno); if (rc != CN_OK) return rc;
      H.cseg = dsg; H.cseg_child = dsc; H.cdist = dsd; H.cseg_lvl = dsl; H.cplan_noff = dno;
      m->cwin_perm = perm;
      rc = dev_alloc(m, 256, &H.cwin_smctr); if (rc != CN_OK) return rc;
      for (int t = 0; t < nt; ++t) {
        HTable &T = m->tab[t];
        if (!T.ti.point) continue;
        // the node of every instance as a plan position of its cell's class
        uvec<int32_t> ppos((size_t)T.n);
        par_for(T.n, 1 << 16, [&](int64_t i0, int64_t i1) {
          for (int64_t i = i0; i < i1; ++i) {
            const int32_t c = cell_of_node[T.node[i]];
            ppos[T.inst_pos[i]] = perm[m->cell_cls[c]][T.node[i] - m->cell_first[c]];
          }
        });
        rc = dev_upload(m, ppos, &T.d_pp_local); if (rc != CN_OK) return rc;
        H.tab[t].pp_local = T.d_pp_local;
      }
      if (max_bytes > 48 * 1024) {
        CU(cudaFuncSetAttribute(cell_window_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_bytes));
        CU(cudaFuncSetAttribute(cell_window_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_bytes));
        CU(cudaFuncSetAttribute(cell_window_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_bytes));
      }
    }
  }
  rc = dev_alloc(m, 2, &H.step_ctr); if (rc != CN_OK) return rc;
  if (const char *e = m->opt("graph")) m->graph_on = std::atoi(e) != 0;
  // spikes
  rc = dev_alloc(m, (size_t)m->sp_cap, &m->d_sp_gid, false); if (rc) return rc;
  rc = dev_alloc(m, (size_t)m->sp_cap, &m->d_sp_step, false); if (rc) return rc;
  rc = dev_alloc(m, 1, &m->d_nsp); if (rc) return rc;
  rc = dev_alloc(m, 1, &m->d_overflow); if (rc) return rc;
  H.sp_gid = m->d_sp_gid; H.sp_step = m->d_sp_step; H.n_sp = m->d_nsp; H.sp_cap = m->sp_cap;
  H.overflow = m->d_overflow;
  lap("window buffers, spikes");
  // caller-order gather buffer for cn_get_v, probes
  rc = dev_alloc(m, (size_t)std::max<int64_t>(N, 1), &m->d_gather, false); if (rc) return rc;
  if (!m->probe.empty()) {
    std::vector<int64_t> pp(m->probe.size());
    for (size_t j = 0; j < pp.size(); ++j) pp[j] = m->node_pos[m->probe[j]];
    UP(pp, m->d_probe_pos);
    rc = dev_alloc(m, (size_t)(m->probe_cap * (int64_t)m->probe.size()), &m->d_trace, false);
    if (rc) return rc;
    if (m->cwindow) {  // the probes of every cell: the cell-window kernel records them per step
      std::vector<int32_t> first((size_t)ng + 1, 0), col(m->probe.size());
      std::vector<int64_t> pos(m->probe.size());
      std::vector<int32_t> grp_of(m->probe.size());
      for (size_t j = 0; j < m->probe.size(); ++j) {
        const int64_t nd = m->probe[j];
        const int32_t c = (int32_t)(std::upper_bound(m->cell_first.begin(), m->cell_first.end(), nd) -
                                    m->cell_first.begin()) - 1;
        grp_of[j] = m->cell_grp[c];
        first[grp_of[j] + 1]++;
      }
      for (int g = 0; g < ng; ++g) first[g + 1] += first[g];
      std::vector<int32_t> fill(first.begin(), first.end() - 1);
      for (size_t j = 0; j < m->probe.size(); ++j) {
        const int32_t q = fill[grp_of[j]]++;
        const int32_t c = (int32_t)(std::upper_bound(m->cell_first.begin(), m->cell_first.end(),
                                                     (int64_t)m->probe[j]) - m->cell_first.begin()) - 1;
        pos[q] = m->cwin_perm[m->cell_cls[c]][m->probe[j] - m->cell_first[c]];  // plan position
        col[q] = (int32_t)j;
      }
      int32_t *df, *dc;
      int64_t *dp;
      UP(first, df); UP(pos, dp); UP(col, dc);
      H.wp_first = df; H.wp_pos = dp; H.wp_col = dc;
      H.trace = m->d_trace;
      H.trace_cap = m->probe_cap;
      H.n_probe = (int32_t)m->probe.size();
    }
    if (m->window) {  // the probes of every group: the interleaved kernel records them per step
      const int ntg = (int)m->tgrp.size();
      std::vector<int32_t> first((size_t)ntg + 1, 0), col(m->probe.size());
      std::vector<int64_t> pos(m->probe.size());
      std::vector<int32_t> grp_of(m->probe.size());
      for (size_t j = 0; j < m->probe.size(); ++j) {
        const int64_t nd = m->probe[j];
        const int32_t c = (int32_t)(std::upper_bound(m->cell_first.begin(), m->cell_first.end(), nd) -
                                    m->cell_first.begin()) - 1;
        grp_of[j] = m->cell_grp[c] - m->n_cgroup;
        first[grp_of[j] + 1]++;
      }
      for (int g = 0; g < ntg; ++g) first[g + 1] += first[g];
      std::vector<int32_t> fill(first.begin(), first.end() - 1);
      for (size_t j = 0; j < m->probe.size(); ++j) {
        const int32_t q = fill[grp_of[j]]++;
        pos[q] = pp[j];
        col[q] = (int32_t)j;
      }
      int32_t *df, *dc;
      int64_t *dp;
      UP(first, df); UP(pos, dp); UP(col, dc);
      H.wp_first = df; H.wp_pos = dp; H.wp_col = dc;
      H.trace = m->d_trace;
      H.trace_cap = m->probe_cap;
      H.n_probe = (int32_t)m->probe.size();
    }
  }
#undef UP
  // The uploads and memsets above ran on the legacy default stream; the model's stream may be a
  // non-blocking one (torch's are) that does not wait for it: everything lands before the first launch.
  lap("probes");
  CU(cudaDeviceSynchronize());
  lap("device synchronize");
  m->raw.release();
  lap("release of the compact arrays");
  CU(cudaEventCreate(&m->ev0));
  CU(cudaEventCreate(&m->ev1));
  m->dt = dt;
  m->uploaded = true;
  return CN_OK;
}

