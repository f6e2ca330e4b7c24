// cn_tape_program.hpp -- host side of the interleaved kernel (cn_tape.cuh): compiles the tree of one
// shape class into the W record lists the kernel interprets (static schedule, hand-over kinds,
// dependencies, tape rows, chunks, backward program) and dry-runs them.  Included by cn_layout.hpp
// after the host model structures (cn_model, HClass, HTape, HTask); not a stand-alone unit.
#pragma once

// Program of the interleaved kernel for one class: a static schedule of the cell's elimination
// over W warps (children before parents, L196).
//   1. The tree is cut into tasks: whole subtrees small enough to balance (visited depth-first,
//      the heaviest child last so that it hands over to the parent in registers) and, above them,
//      single nodes.  The tasks are list-scheduled on W warps, deepest first; a warp that
//      completes the last child of a node continues with that node.
//   2. Every node with distributed mechanisms gets a MECH record (nrn_state of the previous step,
//      nrn_cur); these come first on every warp, spread evenly in the order the elimination
//      needs them.
//   3. Contributions that are not handed over in registers meet in the parent's row of the
//      shared-memory system: the first contributor stores, the others add, one after the other
//      in the order of the simulated schedule.  Dependencies between warps become WAIT records /
//      signal flags on per-warp progress counters.  All dependencies point backwards in simulated
//      time (MECH records depend on nothing), so the program cannot deadlock; a host-side dry run
//      checks that anyway.
//   4. Each warp's records get consecutive rows of the group's tape, padded so that no record
//      wraps around the warp's ring; the chunk bookkeeping of the ring is precomputed.
static int build_tape_program(cn_model *m, HClass &K) {
  HTape &P = K.tp;
  const int n = K.n;
  const int nt = (int)m->tab.size();
  const int W = m->tape_W;
  const uint32_t CH = (uint32_t)m->tape_CH;
  const int64_t f = m->cell_first[K.rep_cell];
  auto give_up = [&]() {  // this class stays on the cooperative kernel
    P.n_groups = 0;
    P.n_cells = 0;
    return CN_OK;
  };
  if (n > 1023) return give_up();  // 10-bit system rows
  std::vector<int32_t> par(n, -1);
  std::vector<std::vector<int32_t>> ch(n);
  for (int i = 1; i < n; ++i) {
    par[i] = (int32_t)(m->parent[f + i] - f);
    ch[par[i]].push_back(i);
  }
  // which local nodes carry which distributed table (from the representative cell), cost weights
  P.tab_row.assign(nt, std::vector<int32_t>());
  std::vector<uint32_t> node_mask(n, 0);
  std::vector<uint8_t> has_cai(n, 0), need_ica(n, 0);
  std::vector<double> ecost(n, 1.0), mcost(n, 0.0);
  for (int t = 0; t < nt; ++t) {
    const HTable &T = m->tab[t];
    if (T.ti.point) continue;
    P.tab_row[t].assign(n, -1);
    if (T.type == CN_PAS) continue;  // folded into the static rows
    for (int64_t q = T.cell_first[K.rep_cell]; q < T.cell_first[K.rep_cell + 1]; ++q) {
      const int x = (int)(T.node[T.inst(q)] - f);
      node_mask[x] |= 1u << t;
      if (T.type == CN_CADYN) has_cai[x] = need_ica[x] = 1;
      if (T.type == CN_SK) has_cai[x] = 1;
      mcost[x] += (T.type == CN_HH ? 12.0 : T.type == CN_HHFORM ? 8.0 : T.type == CN_SK ? 6.0 : 1.0) *
                  m->tape_mcost_scale;
    }
  }
  for (int x = 0; x < n; ++x)
    if (P.has_pp[x]) ecost[x] += 0.3;
  for (int x = 0; x < n; ++x)  // a node where contributions meet costs more than a chain node
    if (ch[x].size() > 1 || node_mask[x]) ecost[x] += m->tape_bcost;
  std::vector<double> sw(ecost), bl(n, 0.0);
  for (int x = n - 1; x >= 1; --x) sw[par[x]] += sw[x];
  for (int x = 0; x < n; ++x) bl[x] = ecost[x] + (x ? bl[par[x]] : 0.0);

  // ---- 1. tasks ---------------------------------------------------------------------------
  struct Task {
    std::vector<int32_t> nodes;  // in visiting order, top node last
    int ptask = -1, pending = 0, warp = -1;
    double cost = 0.0, ready = 0.0, prio = 0.0, t0 = 0.0, t1 = 0.0;
    std::vector<int> kids;
  };
  std::vector<Task> tasks;
  std::vector<int32_t> task_of(n, -1);
  const double gran = W > 1 ? sw[0] / (m->tape_gran * W) : 1e300;
  for (int x = 0; x < n; ++x) {
    if (sw[x] > gran) {  // upper node: a task of its own
      task_of[x] = (int)tasks.size();
      tasks.emplace_back();
      tasks.back().nodes.push_back(x);
    } else if (x == 0 || sw[par[x]] > gran) {  // root of a small subtree: depth-first post-order
      const int id = (int)tasks.size();
      tasks.emplace_back();
      std::vector<std::pair<int32_t, uint32_t>> st;
      st.emplace_back(x, 0u);
      while (!st.empty()) {
        auto &top = st.back();
        auto &c = ch[top.first];
        if (top.second == 0 && c.size() > 1)
          std::stable_sort(c.begin(), c.end(), [&](int p, int q) { return sw[p] < sw[q]; });
        if (top.second < c.size()) {
          const int32_t y = c[top.second++];
          st.emplace_back(y, 0u);
        } else {
          tasks[id].nodes.push_back(top.first);
          task_of[top.first] = id;
          st.pop_back();
        }
      }
    }
  }
  const int ntask = (int)tasks.size();
  for (int id = 0; id < ntask; ++id) {
    Task &T = tasks[id];
    const int top = T.nodes.back();
    for (int32_t x : T.nodes) T.cost += ecost[x];
    T.prio = bl[top];
    T.ptask = top ? task_of[par[top]] : -1;
  }
  for (int id = 0; id < ntask; ++id)
    if (tasks[id].ptask >= 0) tasks[tasks[id].ptask].kids.push_back(id);
  // when a task may start on warp w: all children done, plus a hand-over cost for every child
  // that ran on another warp (signal, wake-up, contribution through shared memory)
  const double hcost = m->tape_hcost;
  auto ready_on = [&](const Task &T, int w) {
    double r = 0.0;
    for (int c : T.kids) r = std::max(r, tasks[c].t1 + (tasks[c].warp == w ? 0.0 : hcost));
    return r;
  };
  // ---- list scheduling (two passes: the second one knows the mechanism load of each warp) ----
  std::vector<double> mload(W, 0.0), t_end(n, 0.0), mt_end(n, 0.0);
  std::vector<int> e_warp(n, 0), m_warp(n, -1);
  std::vector<std::vector<int32_t>> elist(W), mlist(W);
  for (int pass = 0; pass < 2; ++pass) {
    for (Task &T : tasks) { T.pending = 0; T.warp = -1; T.ready = 0.0; }
    for (const Task &T : tasks)
      if (T.ptask >= 0) tasks[T.ptask].pending++;
    std::vector<double> wt(mload);
    std::vector<int> last(W, -1);
    for (auto &l : elist) l.clear();
    int done0 = 0;
    auto place = [&](int id, int w) {
      Task &T = tasks[id];
      T.warp = w;
      T.t0 = std::max(wt[w], ready_on(T, w));
      double t = T.t0;
      for (int32_t x : T.nodes) {
        t += ecost[x];
        t_end[x] = t;
        e_warp[x] = w;
        elist[w].push_back(x);
      }
      wt[w] = t;
      T.t1 = t;
      last[w] = id;
      if (T.ptask >= 0) {
        tasks[T.ptask].pending--;
        tasks[T.ptask].ready = std::max(tasks[T.ptask].ready, t);
      }
    };
    // the whole subtrees first, largest first to the least loaded warp: in the backward sweep
    // (the reverse of each warp's list) the upper nodes, which every warp waits for, then come
    // before any subtree
    if (W > 1 && m->tape_leaf_first) {
      std::vector<int> leafs;
      for (int id = 0; id < ntask; ++id)
        if (sw[tasks[id].nodes.back()] <= gran) leafs.push_back(id);
      std::stable_sort(leafs.begin(), leafs.end(),
                       [&](int a, int b) { return tasks[a].cost > tasks[b].cost; });
      for (int id : leafs) {
        const int w = (int)(std::min_element(wt.begin(), wt.end()) - wt.begin());
        place(id, w);
        ++done0;
      }
    }
    for (int done = done0; done < ntask; ++done) {
      // the earliest free warp; among equals one that can continue with the parent of its last task
      auto affinity = [&](int w) {
        if (last[w] < 0) return -1;
        const int pt = tasks[last[w]].ptask;
        if (pt >= 0 && tasks[pt].warp < 0 && tasks[pt].pending == 0 &&
            ready_on(tasks[pt], w) <= wt[w] + 1e-9)
          return pt;
        return -1;
      };
      int w = 0;
      for (int u = 1; u < W; ++u)
        if (wt[u] < wt[w] - 1e-9 || (std::fabs(wt[u] - wt[w]) <= 1e-9 && affinity(w) < 0 &&
                                     affinity(u) >= 0))
          w = u;
      int cand = affinity(w);
      if (cand < 0) {
        int best_now = -1, best_later = -1;
        for (int id = 0; id < ntask; ++id) {
          const Task &T = tasks[id];
          if (T.warp >= 0 || T.pending > 0) continue;
          if (T.ready <= wt[w] + 1e-9) {
            if (best_now < 0 || T.prio > tasks[best_now].prio) best_now = id;
          } else if (best_later < 0 || T.ready < tasks[best_later].ready - 1e-9 ||
                     (T.ready <= tasks[best_later].ready + 1e-9 &&
                      T.prio > tasks[best_later].prio)) {
            best_later = id;
          }
        }
        if (best_now < 0 && best_later >= 0) {
          // nothing to do yet: wait until the next task becomes ready, then decide again (the warp
          // that completes its last child may want to continue with it)
          bool other_busy = false;
          for (int u = 0; u < W; ++u)
            if (u != w && wt[u] > wt[w] + 1e-9) other_busy = true;
          if (other_busy && wt[w] < tasks[best_later].ready - 1e-9) {
            wt[w] = tasks[best_later].ready;
            --done;
            continue;
          }
        }
        cand = best_now >= 0 ? best_now : best_later;
      }
      if (cand < 0) return fail(CN_ERR_TOPOLOGY, "internal: tape scheduler found no task");
      place(cand, w);
    }
    P.sim_makespan = *std::max_element(wt.begin(), wt.end());
    if (pass == 1) break;
    // ---- 2. mechanism records: in the order the elimination needs them, to the least loaded ----
    std::vector<int32_t> mn;
    for (int x = 0; x < n; ++x)
      if (node_mask[x]) mn.push_back(x);
    if (mn.empty()) break;
    std::stable_sort(mn.begin(), mn.end(), [&](int p, int q) { return t_end[p] < t_end[q]; });
    for (int32_t x : mn) {
      const int w = (int)(std::min_element(mload.begin(), mload.end()) - mload.begin());
      mload[w] += mcost[x];
      mt_end[x] = mload[w];
      m_warp[x] = w;
      mlist[w].push_back(x);
    }
  }
  P.sim_work = sw[0];
  for (int x = 0; x < n; ++x) P.sim_work += mcost[x];
  // Which list runs on which warp is free.  Warps w and w + 4 share a quarter of the tensor
  // memory (64 row slots): pair the longest list with the shortest, and so on, so that as few
  // private rows as possible overflow into shared memory.
  if (W > 4 && W <= 8) {
    std::vector<int> rank(W);
    std::iota(rank.begin(), rank.end(), 0);
    std::stable_sort(rank.begin(), rank.end(),
                     [&](int a, int b) { return elist[a].size() > elist[b].size(); });
    std::vector<int> slot(W);
    for (int r = 0; r < W; ++r) slot[rank[r]] = r < 4 ? r : 4 + (W - 1 - r);
    std::vector<std::vector<int32_t>> e2(W), m2(W);
    for (int w = 0; w < W; ++w) {
      e2[slot[w]].swap(elist[w]);
      m2[slot[w]].swap(mlist[w]);
    }
    elist.swap(e2);
    mlist.swap(m2);
    for (int x = 0; x < n; ++x) {
      e_warp[x] = slot[e_warp[x]];
      if (m_warp[x] >= 0) m_warp[x] = slot[m_warp[x]];
    }
  }

  // ---- 3. records, hand-over kinds, dependencies ----------------------------------------------
  struct Rec {
    int type = 0;      // 0 ELIM, 1 MECH
    int32_t node = 0;
    uint32_t flags = 0;
    std::vector<std::pair<int, int>> deps;  // (warp, pre-index) this record waits for, forward
    int bw_warp = -1, bw_pre = -1;          // backward: the parent's record on another warp
    int fidx = 0;                           // index in the final list (WAIT records included)
    uint32_t row = 0, len = 0, ring = 0;    // first tape row, rows, byte offset in the ring
    uint32_t srow = 0;                      // row of the shared-memory system, or TMEM slot
    bool tm = false;
    int unit = -1;                          // backward unit (RUN or single ELIM record) of the node
    int sig = 0;                            // mbarrier the record arrives on (RF_SIG_F)
  };
  std::vector<std::vector<Rec>> recs(W);
  std::vector<int> e_pre(n, -1), m_pre(n, -1);  // pre-index of a node's records in its warp's list
  for (int w = 0; w < W; ++w) {
    for (int32_t x : mlist[w]) {
      m_pre[x] = (int)recs[w].size();
      Rec r;
      r.type = 1;
      r.node = x;
      r.flags = RT_MECH | (has_cai[x] ? RM_HAS_CAI : 0) | (need_ica[x] ? RM_NEED_ICA : 0);
      recs[w].push_back(r);
    }
    for (int32_t x : elist[w]) {
      e_pre[x] = (int)recs[w].size();
      Rec r;
      r.node = x;
      recs[w].push_back(r);
    }
  }
  auto erec = [&](int x) -> Rec & { return recs[e_warp[x]][e_pre[x]]; };
  std::vector<uint8_t> fwd(n, 0);
  for (int w = 0; w < W; ++w)
    for (size_t i = 0; i + 1 < elist[w].size(); ++i)
      if (par[elist[w][i]] == elist[w][i + 1]) fwd[elist[w][i]] = 1;
  auto add_dep = [&](Rec &r, int rw, int w2, int pre2) {
    if (w2 == rw) return;  // program order
    r.deps.emplace_back(w2, pre2);
    recs[w2][pre2].flags |= RF_SIG_F;
  };
  for (int x = 0; x < n; ++x) {
    Rec &r = erec(x);
    if (x == 0) r.flags |= RK_ROOT;
    else if (fwd[x]) r.flags |= RK_FWD;
    if (P.has_pp[x]) r.flags |= RF_HAS_PP;
    if (node_mask[x]) r.flags |= RF_MECHV;
    // contributors to x's system row: its mechanism record first, then the children that do not
    // hand over in registers, in the order of the simulated schedule
    std::vector<int32_t> cs;
    for (int32_t c : ch[x]) {
      if (fwd[c]) r.flags |= RF_FWD_IN;
      else cs.push_back(c);
    }
    std::stable_sort(cs.begin(), cs.end(), [&](int p, int q) {
      if (t_end[p] != t_end[q]) return t_end[p] < t_end[q];
      if (e_warp[p] != e_warp[q]) return e_warp[p] < e_warp[q];
      return e_pre[p] < e_pre[q];
    });
    int lw = -1, lp = -1;  // last contributor so far
    if (node_mask[x]) {
      lw = m_warp[x];
      lp = m_pre[x];
    }
    for (int32_t c : cs) {
      Rec &rc = erec(c);
      rc.flags |= lw < 0 ? RK_STORE : RK_ADD;
      if (lw >= 0) add_dep(rc, e_warp[c], lw, lp);
      lw = e_warp[c];
      lp = e_pre[c];
    }
    if (lw >= 0) {
      r.flags |= RF_HAS_ACC;
      add_dep(r, e_warp[x], lw, lp);
    }
  }
  // ---- 4. tape rows: each warp's records get consecutive rows, padded so that no record wraps
  // around the warp's ring; system rows in the same order ----------------------------------------
  P.order.clear();
  P.pos_of.assign(n, 0);
  P.row.assign(n, 0);
  P.cai_row.assign(n, -1);
  P.ica_row.assign(n, -1);
  P.pp_row.assign(n, -1);
  P.vcopy_row.assign(n, -1);
  P.task.assign(W, HTask());
  P.prog.clear();
  // point-process nodes are numbered in the order the warps meet them (window mode prefetches
  // the rows of the next one while it works on the current one)
  P.pp_ord.assign(n, -1);
  P.n_pp = 0;
  for (int w = 0; w < W; ++w) {
    P.task[w].pp0 = P.n_pp;
    for (int32_t x : elist[w]) {
      P.pos_of[x] = (int32_t)P.order.size();
      P.order.push_back(x);
      if (P.has_pp[x]) P.pp_ord[x] = P.n_pp++;
    }
  }
  if (P.n_pp > 1023) return give_up();
  // Where (multiplier, reduced rhs) of a node wait for the back-substitution: a node without
  // contributions from mechanisms or from children that do not hand over in registers (its row
  // is written and read by its own warp only) gets a slot of the warp's share of tensor
  // memory (each quarter of the CTA's 256 TMEM columns = 64 slots, shared by the warps w, w + 4, ...
  // that can address it); every other node, and what does not fit, a row of the shared-memory
  // system.
  {
    std::vector<int> plain_cnt(W, 0), cap(W, 0);
    auto is_plain = [&](const Rec &r) {  // nobody else touches the node's row
      return r.type == 0 && !(r.flags & RF_HAS_ACC);
    };
    for (int w = 0; w < W; ++w)
      for (const Rec &r : recs[w]) plain_cnt[w] += is_plain(r) ? 1 : 0;
    const int tm_slots = m->tape_tmem ? 64 : 0;
    for (int q = 0; q < 4 && q < W; ++q) {
      int tot = 0;
      for (int w = q; w < W; w += 4) tot += plain_cnt[w];
      int base = 0;
      for (int w = q; w < W; w += 4) {
        cap[w] = tot <= tm_slots ? plain_cnt[w] : (int)((int64_t)plain_cnt[w] * tm_slots / tot);
        P.task[w].tm_base = base;
        base += cap[w];
      }
    }
    uint32_t ns = 0;
    for (int w = 0; w < W; ++w) {
      int used = 0;
      for (Rec &r : recs[w]) {
        if (r.type != 0) continue;
        if (is_plain(r) && used < cap[w]) {
          r.tm = true;
          r.srow = (uint32_t)used++;
        } else {
          r.srow = ns++;
        }
      }
    }
    for (int w = 0; w < W; ++w)
      for (Rec &r : recs[w])
        if (r.type == 1) r.srow = erec(r.node).srow;  // a mechanism record writes the node's row
    if (ns > 1023) return give_up();
    P.n_srow = (int)ns;
  }
  uint32_t row = 0;
  for (int w = 0; w < W; ++w) {
    HTask &Tk = P.task[w];
    Tk.row0 = row;
    for (Rec &r : recs[w]) {
      const int x = r.node;
      uint32_t ln;
      if (r.type == 1) {
        ln = 1 + (has_cai[x] ? 1 : 0) + (need_ica[x] ? 1 : 0);
        for (int t = 0; t < nt; ++t)
          if (node_mask[x] & (1u << t)) ln += (uint32_t)tape_rows_of(m->tab[t].ti, m->tab[t].type);
      } else {
        ln = 5 + (P.has_pp[x] ? 2 : 0);
      }
      if (ln > CH) return give_up();  // a record must fit a chunk (build_layout sizes CH for it)
      r.row = row;
      r.len = ln;
      row += ln;
      if (r.type == 1) {
        uint32_t q = r.row;
        P.vcopy_row[x] = (int32_t)q++;
        if (has_cai[x]) P.cai_row[x] = (int32_t)q++;
        if (need_ica[x]) P.ica_row[x] = (int32_t)q++;
        for (int t = 0; t < nt; ++t)
          if (node_mask[x] & (1u << t)) {
            P.tab_row[t][x] = (int32_t)q;
            q += (uint32_t)tape_rows_of(m->tab[t].ti, m->tab[t].type);
          }
      } else {
        P.row[P.pos_of[x]] = r.row;
        if (P.has_pp[x]) P.pp_row[x] = (int32_t)(r.row + 5);
      }
    }
    Tk.nrows = row - Tk.row0;
    if (row > 65535) return give_up();  // 16-bit tape rows
  }
  P.n_rows = (int)row;
  // final lists.  The records of a warp are packed into chunks of at most CH rows (chunk c goes
  // to stage c % S of the warp's ring): a CHUNK record precedes the first record of every chunk.
  // WAIT records go in front of the record that needs them (a wait that an earlier wait of the
  // same warp already covers is dropped: positions on one warp only grow).  Plain chain nodes
  // that follow one another inside a chunk are merged into RUN records.
  // A run may end with the TOP of its chain: a node like the plain ones, except that its contribution
  // goes to its parent's row (store / add, possibly signalled) instead of to the next record in
  // registers (Fin::tail): one record less per chain for the interpreter.
  struct Fin { int type; int pre; int cnt; int w2, pre2; bool tail = false; };  // type 2 = WAIT, 3 = RUN, 4 = CHUNK
  std::vector<std::vector<Fin>> fin(W);
  std::vector<std::vector<std::pair<uint32_t, uint32_t>>> chunks(W);  // (first row in segment, rows)
  const uint32_t S = (uint32_t)m->tape_S;
  auto x_parent_row_ok = [&](const Rec &r) {  // the parent collects contributions in a shared row
    const int x = r.node;
    return x > 0 && (erec(par[x]).flags & RF_HAS_ACC) && !erec(par[x]).tm;
  };
  for (int w = 0; w < W; ++w) {
    std::vector<int> seen(W, -1);
    uint32_t fill = CH + 1;  // rows used in the current chunk (none open yet)
    for (int i = 0; i < (int)recs[w].size(); ++i) {
      Rec &r = recs[w][i];
      bool fresh = false;
      if (fill + r.len > CH) {
        fin[w].push_back(Fin{4, (int)chunks[w].size(), 0, -1, -1});
        chunks[w].emplace_back(r.row - P.task[w].row0, 0u);
        fill = 0;
        fresh = true;
      }
      r.ring = ((uint32_t)((chunks[w].size() - 1) % S) * CH + fill) * 256u;
      fill += r.len;
      chunks[w].back().second = fill;
      int n_wait = 0;
      for (auto &d : r.deps) {
        if (seen[d.first] >= d.second) continue;
        seen[d.first] = d.second;
        fin[w].push_back(Fin{2, -1, 0, d.first, d.second});
        fresh = true;
        ++n_wait;
      }
      // a single wait in front of an elimination record travels in the record itself (one record
      // less on the warps that eliminate the upper nodes: the forward critical path)
      int emb_w = -1, emb_pre = -1;
      if (n_wait == 1 && r.type == 0 && (r.flags & ~(uint32_t)RF_FWD_IN) != RK_FWD) {
        emb_w = fin[w].back().w2;
        emb_pre = fin[w].back().pre2;
        fin[w].pop_back();
      }
      const bool plain = r.type == 0 && (r.flags & ~(uint32_t)RF_FWD_IN) == RK_FWD;
      const uint32_t kind = r.flags & RK_KIND;
      const bool chain_top = r.type == 0 && (kind == RK_STORE || kind == RK_ADD) &&
                             (r.flags & ~(uint32_t)(RK_KIND | RF_SIG_F)) == RF_FWD_IN && x_parent_row_ok(r);
      if ((plain || chain_top) && !fresh && fin[w].back().type == 3 && !fin[w].back().tail &&
          fin[w].back().cnt < 255 && (r.flags & RF_FWD_IN) && recs[w][i - 1].tm == r.tm &&
          recs[w][i - 1].srow + 1 == r.srow) {
        r.fidx = (int)fin[w].size() - 1;
        fin[w].back().cnt++;
        fin[w].back().tail = chain_top;
        continue;
      }
      r.fidx = (int)fin[w].size();
      fin[w].push_back(Fin{plain ? 3 : r.type, i, 1, emb_w, emb_pre});
    }
    if (fin[w].size() > 2047) return give_up();  // 12-bit backward positions
    HTask &Tk = P.task[w];
    Tk.nchunk = (int)chunks[w].size();
    Tk.head = 0;
    for (uint32_t c = 0; c < 4 && c < chunks[w].size(); ++c) Tk.head |= chunks[w][c].second << (8 * c);
  }
  // every signalling record arrives on an mbarrier of its own (once per group)
  P.n_bar = 0;
  for (int w = 0; w < W; ++w)
    for (Rec &r : recs[w])
      if (r.flags & RF_SIG_F) r.sig = P.n_bar++;
  // encoding (layout of the records: cn_device.cuh)
  for (int w = 0; w < W; ++w) {
    HTask &Tk = P.task[w];
    Tk.p0 = (int)P.prog.size();
    for (const Fin &F : fin[w]) {
      if (F.type == 2) {
        P.prog.push_back(make_uint4(0u, (uint32_t)RT_WAIT, (uint32_t)recs[F.w2][F.pre2].sig, 0u));
        continue;
      }
      if (F.type == 4) {  // chunk c starts: chunk c-1 is consumed, its stage takes chunk c-1+S
        const uint32_t c = (uint32_t)F.pre;
        uint32_t ex = 0, fill_stage = 0;
        if (c >= 1 && c - 1 + S < chunks[w].size()) {
          ex = chunks[w][c - 1 + S].first | chunks[w][c - 1 + S].second << 16;
          fill_stage = (c - 1) % S;
        }
        P.prog.push_back(make_uint4(ex, (uint32_t)RT_CHUNK, fill_stage | (c % S) << 16, 0u));
        continue;
      }
      const Rec &r = recs[w][F.pre];
      const int x = r.node;
      if (F.type == 3) {
        uint32_t y = (uint32_t)RT_RUN, wv = r.row;
        if (F.tail) {  // the run's last node stores / adds its contribution to its parent's row
          const Rec &t = recs[w][F.pre + F.cnt - 1];
          y |= erec(par[t.node]).srow << 16 | 1u << 26 | ((t.flags & RK_KIND) == RK_ADD ? 1u << 27 : 0u);
          if (t.flags & RF_SIG_F) wv |= (uint32_t)t.sig << 16 | 1u << 24;
        }
        P.prog.push_back(make_uint4(r.ring | (uint32_t)F.cnt << 16 |
                                        ((r.flags & RF_FWD_IN) ? 1u << 24 : 0u),
                                    y, r.srow | (r.tm ? 1u << 20 : 0u), wv));
      } else if (r.type == 1) {
        P.prog.push_back(make_uint4(r.ring, r.flags | r.row << 16, r.srow | (uint32_t)r.sig << 16,
                                    node_mask[x]));
      } else {
        const uint32_t ey = r.flags | (r.tm ? (uint32_t)RF_TMEM : 0u) | (uint32_t)r.sig << 16;
        // the parent's row is written (contribution) or read (v) only if it collects contributions
        // (RF_HAS_ACC); such a row is always in shared memory
        const uint32_t ez =
            r.srow | (uint32_t)(x && (erec(par[x]).flags & RF_HAS_ACC) ? erec(par[x]).srow : 0) << 10 |
            (uint32_t)(P.has_pp[x] ? P.pp_ord[x] : 0) << 21;
        const uint32_t ew = r.row | (uint32_t)(node_mask[x] ? P.vcopy_row[x] : 0) << 16;
        uint32_t ex = r.ring;
        if (F.w2 >= 0) ex |= (uint32_t)recs[F.w2][F.pre2].sig << 16 | 1u << 24;  // forward: wait first
        P.prog.push_back(make_uint4(ex, ey, ez, ew));
      }
    }
    Tk.p1 = (int)P.prog.size();
  }

  // ---- 5. backward program -----------------------------------------------------------------------
  // Back-substitution visits parents before children.  Its order is NOT the reverse of the
  // forward lists: per warp, the units (a RUN or a single ELIM record) whose parent is solved are
  // taken upper nodes first (every other warp waits for those), then depth-first.  A unit whose
  // last-solved node does not keep v in its system row (no RF_HAS_ACC) must be followed by its
  // only child at once (v travels in a register); every other unit reads the parent's v from the
  // parent's row (RF_BW_ROW) unless it happens to follow its parent directly.
  {
    // A forward RUN ends at the end of its chunk; the backward sweep reads no chunks, so runs
    // that continue one chain (only a CHUNK record between them, consecutive rows and slots) are
    // one backward unit: fewer records for the interpreter (~0.25 us each, whatever their length).
    struct Unit { int w; int fin_idx; int top, bottom; bool stores_v; int warp_pos = -1; int cnt = 1; };
    std::vector<Unit> units;
    for (int w = 0; w < W; ++w) {
      int fi = 0;
      int open_run = -1;  // the unit of the last RUN if only CHUNK records followed it so far
      for (const Fin &F : fin[w]) {
        if (F.type == 3 && open_run >= 0) {
          Unit &A = units[open_run];
          const Rec &first = recs[w][F.pre], &prev = recs[w][F.pre - 1];
          if ((first.flags & RF_FWD_IN) && prev.unit == open_run && prev.tm == first.tm &&
              prev.srow + 1 == first.srow && prev.row + 5 == first.row && A.cnt + F.cnt <= 255) {
            A.top = recs[w][F.pre + F.cnt - 1].node;
            A.cnt += F.cnt;
            for (int i = 0; i < F.cnt; ++i) recs[w][F.pre + i].unit = open_run;
            ++fi;
            continue;
          }
        }
        if (F.type != 4) open_run = -1;
        if (F.type == 0 || F.type == 3) {
          Unit u;
          u.w = w;
          u.fin_idx = fi;
          u.bottom = recs[w][F.pre].node;
          u.top = recs[w][F.pre + F.cnt - 1].node;
          u.stores_v = F.type == 0 && (recs[w][F.pre].flags & RF_HAS_ACC);
          u.cnt = F.cnt;
          for (int i = 0; i < F.cnt; ++i) recs[w][F.pre + i].unit = (int)units.size();
          if (F.type == 3) open_run = (int)units.size();
          units.push_back(u);
        }
        ++fi;
      }
    }
    const int nu = (int)units.size();
    std::vector<std::vector<int>> kids(nu);  // same-warp child units, the register child first
    std::vector<int> punit(nu, -1);
    std::vector<int> depth(n, 0);
    for (int x = 1; x < n; ++x) depth[x] = depth[par[x]] + 1;
    for (int u = 0; u < nu; ++u) {
      const int t = units[u].top;
      if (t == 0) continue;
      punit[u] = erec(par[t]).unit;
      if (units[punit[u]].w == units[u].w) {
        if (fwd[t]) kids[punit[u]].insert(kids[punit[u]].begin(), u);
        else kids[punit[u]].push_back(u);
      }
    }
    std::vector<std::vector<int>> blist(W);
    std::vector<uint8_t> bw_row(nu, 0);
    for (int w = 0; w < W; ++w) {
      // upper units by depth, others depth-first (a stack)
      auto upper = [&](int u) { return sw[units[u].top] > gran; };
      std::vector<int> heap, stack;
      auto push = [&](int u) { (upper(u) ? heap : stack).push_back(u); };
      for (int u = nu - 1; u >= 0; --u)
        if (units[u].w == w && (punit[u] < 0 || units[punit[u]].w != w)) push(u);
      int forced = -1, last = -1;
      while (forced >= 0 || !heap.empty() || !stack.empty()) {
        int u;
        if (forced >= 0) {
          u = forced;
        } else if (!heap.empty()) {
          auto it = std::min_element(heap.begin(), heap.end(), [&](int a, int b) {
            return depth[units[a].top] < depth[units[b].top];
          });
          u = *it;
          heap.erase(it);
        } else {
          u = stack.back();
          stack.pop_back();
        }
        // v of the parent: register if the parent unit was solved just before, else its row
        if (punit[u] >= 0 && !(last == punit[u] && fwd[units[u].top])) bw_row[u] = 1;
        units[u].warp_pos = (int)blist[w].size();
        blist[w].push_back(u);
        last = u;
        forced = -1;
        if (!units[u].stores_v) {
          if (kids[u].size() > 1 || (kids[u].size() == 1 && !fwd[units[kids[u][0]].top]))
            return fail(CN_ERR_TOPOLOGY, "internal: tape program (backward hand-over)");
          if (!kids[u].empty()) forced = kids[u][0];
        } else {
          // push so that the register child is taken first if nothing more urgent waits
          for (int i = (int)kids[u].size() - 1; i >= 0; --i) push(kids[u][i]);
        }
      }
    }
    // positions in the backward lists (a unit whose parent sits on another warp carries the wait for
    // it itself, run or single record), signals, waits, encoding
    std::vector<int> idxb(nu, 0), sigid_b(nu, -1);
    std::vector<uint8_t> sig_b(nu, 0);
    for (int w = 0; w < W; ++w) {
      int pos = 0;
      for (int u : blist[w]) {
        const bool remote = punit[u] >= 0 && units[punit[u]].w != w;
        const bool is_run = fin[w][units[u].fin_idx].type == 3;
        if (remote) sig_b[punit[u]] = 1;
        (void)is_run;  // (a run carries the wait for a remote parent itself, like a single record)
        idxb[u] = pos++;
      }
    }
    for (int u = 0; u < nu; ++u)
      if (sig_b[u]) sigid_b[u] = P.n_bar++;
    if (P.n_bar > 255) return give_up();
    for (int w = 0; w < W; ++w) {
      HTask &Tk = P.task[w];
      Tk.b0 = (int)P.prog.size();
      std::vector<int> seen(W, -1);
      for (int u : blist[w]) {
        uint4 e = P.prog[Tk.p0 + units[u].fin_idx];
        if (!((e.y & RT_MASK) == RT_RUN)) {
          e.y &= 0xFFFFu & ~(uint32_t)RF_SIG_F;  // the forward signal is not part of the backward copy
          e.x = 0;
        }
        const bool is_run = (e.y & RT_MASK) == RT_RUN;
        if (is_run) {  // (merged runs; the tail fields belong to the forward record only)
          e.x = (e.x & ~(255u << 16)) | (uint32_t)units[u].cnt << 16;
          e.y = (uint32_t)RT_RUN;
          e.w &= 0xFFFFu;
        }
        const int pu = punit[u];
        if (pu >= 0 && units[pu].w != w) {
          const int wp = units[pu].w;
          const int posb = (P.task[wp].p1 - P.task[wp].p0) + idxb[pu] + 1;
          if (posb > 4095) return give_up();
          if (is_run) {
            if (seen[wp] < posb) e.y |= (uint32_t)sigid_b[pu] << 16 | 1u << 24;
          } else if (seen[wp] < posb) {
            e.y |= RF_WAIT_B | (uint32_t)sigid_b[pu] << 16;
          }
          seen[wp] = std::max(seen[wp], posb);
        }
        if (bw_row[u]) {
          const Rec &pr = erec(par[units[u].top]);
          if (!(pr.flags & RF_HAS_ACC) || pr.tm)
            return fail(CN_ERR_TOPOLOGY, "internal: tape program (backward row of a private parent)");
          if (is_run) e.x |= 1u << 25, e.z |= pr.srow << 21;  // z bits 21..30: the parent's row
          else e.y |= RF_BW_ROW;
        }
        if (sig_b[u]) {
          if (is_run) return fail(CN_ERR_TOPOLOGY, "internal: tape program (a run cannot signal)");
          e.y |= RF_SIG_B;
          e.x = (uint32_t)sigid_b[u];
        }
        if ((int)P.prog.size() - Tk.b0 != idxb[u])
          return fail(CN_ERR_TOPOLOGY, "internal: tape program (backward positions)");
        P.prog.push_back(e);
      }
      Tk.b1 = (int)P.prog.size();
    }
  }

  // ---- dry run: the W record lists with the kernel's wait / signal rules -------------------------
  {
    std::vector<int32_t> node_of_srow((size_t)P.n_srow + 1, -1);
    std::vector<std::vector<int32_t>> node_of_slot(W);
    for (int w = 0; w < W; ++w)
      for (const Rec &r : recs[w]) {
        if (r.type != 0) continue;
        if (r.tm) {
          if (node_of_slot[w].size() <= r.srow) node_of_slot[w].resize(r.srow + 1, -1);
          node_of_slot[w][r.srow] = r.node;
        } else {
          node_of_srow[r.srow] = r.node;
        }
      }
    std::vector<int> pc(W), acc(n, 0);
    std::vector<uint8_t> bar_done((size_t)P.n_bar + 1, 0);
    std::vector<uint8_t> done_e(n, 0), done_m(n, 0);
    for (int w = 0; w < W; ++w) pc[w] = P.task[w].p0;
    bool progress = true;
    while (progress) {
      progress = false;
      for (int w = 0; w < W; ++w) {
        while (pc[w] < P.task[w].p1) {
          const uint4 e = P.prog[pc[w]];
          const uint32_t fl = e.y & 0xFFFFu;
          if ((fl & RT_MASK) == RT_CHUNK) {
          } else if ((fl & RT_MASK) == RT_WAIT) {
            if (!bar_done[e.z & 0xFFFFu]) break;
          } else if ((fl & RT_MASK) == RT_RUN) {
            const uint32_t cnt = (e.x >> 16) & 255u;
            for (uint32_t i = 0; i < cnt; ++i) {
              const int x = (e.z >> 20 & 1u) ? node_of_slot[w][(e.z & 1023u) + i]
                                             : node_of_srow[(e.z & 1023u) + i];
              const bool tail = i + 1 == cnt && (e.y >> 26 & 1u);
              if (node_mask[x] || acc[x] != 0 || (!fwd[x]) != tail || ch[x].size() > 1 ||
                  (ch[x].size() == 1 && (!done_e[ch[x][0]] || !fwd[ch[x][0]])) ||
                  (ch[x].size() == 1) != (i > 0 || (e.x >> 24 & 1u)))
                return fail(CN_ERR_TOPOLOGY, "internal: tape program (run)");
              if (tail) {
                const int p = node_of_srow[(e.y >> 16) & 1023u];
                if (x == 0 || p != par[x] || ((e.y >> 27 & 1u) == 0) != (acc[p] == 0))
                  return fail(CN_ERR_TOPOLOGY, "internal: tape program (run tail)");
                acc[p]++;
                if (e.w >> 24 & 1u) bar_done[(e.w >> 16) & 255u] = 1;
              }
              done_e[x] = 1;
            }
          } else if ((fl & RT_MASK) == RT_MECH) {
            const int x = node_of_srow[e.z & 1023u];
            if (acc[x] != 0) return fail(CN_ERR_TOPOLOGY, "internal: tape program (mech order)");
            acc[x] = 1;
            done_m[x] = 1;
          } else {
            if ((e.x >> 24 & 1u) && !bar_done[(e.x >> 16) & 255u]) break;  // (its own wait)
            const int x = (fl & RF_TMEM) ? node_of_slot[w][e.z & 1023u] : node_of_srow[e.z & 1023u];
            int want = node_mask[x] ? 1 : 0;
            for (int32_t c : ch[x]) {
              if (!done_e[c]) return fail(CN_ERR_TOPOLOGY, "internal: tape program (child order)");
              if (!fwd[c]) ++want;
            }
            if (acc[x] != want || ((fl & RF_HAS_ACC) != 0) != (want > 0))
              return fail(CN_ERR_TOPOLOGY, "internal: tape program (contributions)");
            const uint32_t kind = fl & RK_KIND;
            if (kind >= RK_STORE) {
              const int p = node_of_srow[(e.z >> 10) & 1023u];
              if (p != par[x] || (kind == RK_STORE) != (acc[p] == 0))
                return fail(CN_ERR_TOPOLOGY, "internal: tape program (store/add)");
              acc[p]++;
            }
            done_e[x] = 1;
          }
          if (fl & RF_SIG_F) bar_done[(fl & RT_MASK) == RT_MECH ? e.z >> 16 : e.y >> 16] = 1;
          ++pc[w];
          progress = true;
        }
      }
    }
    for (int w = 0; w < W; ++w)
      if (pc[w] != P.task[w].p1) return fail(CN_ERR_TOPOLOGY, "internal: tape program deadlocks");
    // backward
    std::vector<uint8_t> done_b(n, 0), stored_v(n, 0);
    for (int w = 0; w < W; ++w) pc[w] = P.task[w].b0;
    std::vector<int> lastn(W, -1);  // the node whose v is in the warp's register
    progress = true;
    while (progress) {
      progress = false;
      for (int w = 0; w < W; ++w) {
        const HTask &Tk = P.task[w];
        while (pc[w] < Tk.b1) {
          const uint4 e = P.prog[pc[w]];
          const uint32_t fl = e.y & 0xFFFFu;
          if ((fl & RT_MASK) == RT_WAIT) {
            if (!bar_done[e.z & 0xFFFFu]) break;
          } else if ((fl & RT_MASK) == RT_RUN) {
            if ((e.y >> 24 & 1u) && !bar_done[(e.y >> 16) & 255u]) break;  // (its own wait)
            for (int i = (int)((e.x >> 16) & 255u) - 1; i >= 0; --i) {
              const int x = (e.z >> 20 & 1u) ? node_of_slot[w][(e.z & 1023u) + (uint32_t)i]
                                             : node_of_srow[(e.z & 1023u) + (uint32_t)i];
              const bool from_row = i == (int)((e.x >> 16) & 255u) - 1 && (e.x >> 25 & 1u);
              if (!done_b[par[x]] || (from_row ? !stored_v[par[x]] ||
                                                     node_of_srow[(e.z >> 21) & 1023u] != par[x]
                                                : lastn[w] != par[x]))
                return fail(CN_ERR_TOPOLOGY, "internal: tape program (backward run)");
              done_b[x] = 1;
              lastn[w] = x;
            }
          } else if ((fl & RT_MASK) == RT_ELIM) {
            if ((fl & RF_WAIT_B) && !bar_done[e.y >> 16]) break;
            const int x = (fl & RF_TMEM) ? node_of_slot[w][e.z & 1023u] : node_of_srow[e.z & 1023u];
            if (x) {
              const bool from_row = fl & RF_BW_ROW;
              if (!done_b[par[x]] || (from_row ? !stored_v[par[x]] ||
                                                     node_of_srow[(e.z >> 10) & 1023u] != par[x]
                                                : lastn[w] != par[x]))
                return fail(CN_ERR_TOPOLOGY, "internal: tape program (backward order)");
            }
            done_b[x] = 1;
            lastn[w] = x;
            if (fl & RF_HAS_ACC) stored_v[x] = 1;
            if (fl & RF_SIG_B) bar_done[e.x & 0xFFFFu] = 1;
          } else {
            return fail(CN_ERR_TOPOLOGY, "internal: tape program (backward record type)");
          }
          ++pc[w];
          progress = true;
        }
      }
    }
    for (int w = 0; w < W; ++w)
      if (pc[w] != P.task[w].b1)
        return fail(CN_ERR_TOPOLOGY, "internal: tape program deadlocks (backward)");
    for (int x = 0; x < n; ++x)
      if (!done_b[x]) return fail(CN_ERR_TOPOLOGY, "internal: tape program (backward incomplete)");
  }
  return CN_OK;
}

