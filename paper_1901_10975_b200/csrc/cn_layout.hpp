// cn_layout.hpp -- build_layout(): the dt-independent part of the set-up (cn_model_create): shape
// classes, choice of kernel per class, programs of the interleaved kernel, groups, node and
// instance permutations.  Included by cn_api.cu only.
#pragma once

static inline uint64_t mix64(uint64_t h, uint64_t x) {
  h ^= x + 0x9E3779B97F4A7C15ull + (h << 6) + (h >> 2);
  h *= 0xBF58476D1CE4E5B9ull;
  return h ^ (h >> 29);
}

// dev parameter / state rows of a distributed type on the tape (same order as the table arrays)
static int tape_rows_of(const TypeInfo &ti, int type) {
  if (type == CN_PAS || type == CN_CADYN) return 0;
  return ti.n_dev_param + ti.n_state;
}

#include "cn_tape_program.hpp"

static int build_layout(cn_model *m) {
  const bool dbg = m->opt("debug") && std::atoi(m->opt("debug")) != 0;
  auto t_prev = std::chrono::steady_clock::now();
  auto lap = [&](const char *what) {
    if (!dbg) return;
    const auto t = std::chrono::steady_clock::now();
    fprintf(stderr, "[cn] build_layout %-28s %7.1f ms\n", what,
            std::chrono::duration<double, std::milli>(t - t_prev).count());
    t_prev = t;
  };
  const int32_t nc = m->n_cell;
  const int64_t N = m->N;
  const int nt = (int)m->tab.size();
  // node -> cell
  uvec<int32_t> cell_of((size_t)N);
  par_for(nc, 256, [&](int64_t c0, int64_t c1) {
    for (int64_t c = c0; c < c1; ++c)
      for (int64_t i = m->cell_first[c]; i < m->cell_first[c + 1]; ++i) cell_of[i] = (int32_t)c;
  });
  // per distributed table: CSR of instances per cell, sorted by local node
  for (int t = 0; t < nt; ++t) {
    HTable &T = m->tab[t];
    if (T.ti.point) continue;
    {  // instances ordered by node already (the usual case): the CSR is a search per cell
      std::atomic<bool> increasing{true};
      par_for(T.n, 1 << 16, [&](int64_t i0, int64_t i1) {
        for (int64_t i = std::max<int64_t>(i0, 1); i < i1; ++i)
          if (T.node[i] <= T.node[i - 1]) {
            increasing.store(false);
            return;
          }
      });
      if (increasing.load()) {
        T.cell_inst.clear();
        T.cell_first.assign((size_t)nc + 1, 0);
        par_for((int64_t)nc + 1, 1024, [&](int64_t c0, int64_t c1) {
          for (int64_t c = c0; c < c1; ++c)
            T.cell_first[c] = std::lower_bound(T.node.begin(), T.node.end(), (int32_t)m->cell_first[c]) -
                              T.node.begin();
        });
        continue;
      }
    }
    uvec<int64_t> rank;
    par_bucket(T.n, nc, [&](int64_t i) { return cell_of[T.node[i]]; }, T.cell_first, rank);
    T.cell_inst.resize((size_t)T.n);
    par_for(T.n, 1 << 16, [&](int64_t i0, int64_t i1) {
      for (int64_t i = i0; i < i1; ++i) T.cell_inst[rank[i]] = i;
    });
    FirstErr fe;
    par_for(nc, 256, [&](int64_t c0, int64_t c1) {
      for (int64_t c = c0; c < c1; ++c) {
        auto b = T.cell_inst.begin() + T.cell_first[c], e = T.cell_inst.begin() + T.cell_first[c + 1];
        if (!std::is_sorted(b, e, [&](int64_t x, int64_t y) { return T.node[x] < T.node[y]; }))
          std::sort(b, e, [&](int64_t x, int64_t y) { return T.node[x] < T.node[y]; });
        for (auto it = b; it != e && it + 1 != e; ++it)
          if (T.node[*it] == T.node[*(it + 1)])
            return fe.set(T.node[*it], CN_ERR_MECH, "table %d: two instances on node %d", t,
                          T.node[*it]);
      }
    });
    if (fe.code != CN_OK) return fail(fe.code, "%s", fe.msg);
  }
  lap("node -> cell, instance CSR");
  // shape signature per cell: topology + placement of every distributed table
  std::vector<uint64_t> sig(nc);
  par_for(nc, 4096, [&](int64_t c0, int64_t c1) {
  for (int32_t c = (int32_t)c0; c < (int32_t)c1; ++c) {
    const int64_t f = m->cell_first[c], l = m->cell_first[c + 1];
    uint64_t h = mix64(0x1234567ull, (uint64_t)(l - f));
    for (int64_t i = f + 1; i < l; ++i) h = mix64(h, (uint64_t)(m->parent[i] - f));
    for (int t = 0; t < nt; ++t) {
      const HTable &T = m->tab[t];
      if (T.ti.point) continue;
      h = mix64(h, 0xABCD0000ull + (uint64_t)t);
      for (int64_t j = T.cell_first[c]; j < T.cell_first[c + 1]; ++j)
        h = mix64(h, (uint64_t)(T.node[T.inst(j)] - f));
    }
    sig[c] = h;
  }
  });
  lap("signatures");
  auto same_shape = [&](int32_t x, int32_t y) {
    const int64_t fx = m->cell_first[x], fy = m->cell_first[y];
    const int64_t n = m->cell_first[x + 1] - fx;
    if (n != m->cell_first[y + 1] - fy) return false;
    for (int64_t i = 1; i < n; ++i)
      if (m->parent[fx + i] - fx != m->parent[fy + i] - fy) return false;
    for (int t = 0; t < nt; ++t) {
      const HTable &T = m->tab[t];
      if (T.ti.point) continue;
      const int64_t cx = T.cell_first[x + 1] - T.cell_first[x];
      if (cx != T.cell_first[y + 1] - T.cell_first[y]) return false;
      for (int64_t j = 0; j < cx; ++j)
        if (T.node[T.inst(T.cell_first[x] + j)] - fx !=
            T.node[T.inst(T.cell_first[y] + j)] - fy)
          return false;
    }
    return true;
  };
  m->cell_cls.assign(nc, -1);
  {
    // buckets of equal signature (cheap, in cell order), then the exact comparison inside every
    // bucket on all cores; classes are numbered in the order of their first cell
    std::unordered_map<uint64_t, int> bucket_of;
    bucket_of.reserve((size_t)nc / 8 + 16);
    std::vector<std::vector<int32_t>> bcells;
    for (int32_t c = 0; c < nc; ++c) {
      auto it = bucket_of.find(sig[c]);
      if (it == bucket_of.end()) {
        it = bucket_of.emplace(sig[c], (int)bcells.size()).first;
        bcells.emplace_back();
      }
      bcells[it->second].push_back(c);
    }
    std::vector<std::vector<std::vector<int32_t>>> bcls(bcells.size());
    par_for((int64_t)bcells.size(), 4, [&](int64_t b0, int64_t b1) {
      for (int64_t b = b0; b < b1; ++b)
        for (int32_t c : bcells[b]) {
          std::vector<int32_t> *hit = nullptr;
          for (auto &k : bcls[b])
            if (same_shape(k[0], c)) { hit = &k; break; }
          if (!hit) {
            bcls[b].emplace_back();
            hit = &bcls[b].back();
          }
          hit->push_back(c);
        }
    });
    std::vector<std::vector<int32_t> *> all;
    for (auto &b : bcls)
      for (auto &k : b) all.push_back(&k);
    std::sort(all.begin(), all.end(),
              [](const std::vector<int32_t> *x, const std::vector<int32_t> *y) { return (*x)[0] < (*y)[0]; });
    m->cls.reserve(all.size());
    for (auto *k : all) {
      const int id = (int)m->cls.size();
      m->cls.emplace_back();
      HClass &K = m->cls.back();
      K.rep_cell = (*k)[0];
      K.n = (int)(m->cell_first[K.rep_cell + 1] - m->cell_first[K.rep_cell]);
      K.cells.assign(k->begin(), k->end());
      for (int32_t c : *k) m->cell_cls[c] = id;
    }
  }
  // which tables need ica / cai
  bool has_cadyn = false, has_caform = false, has_sk = false;
  for (const HTable &T : m->tab) {
    if (T.type == CN_CADYN) has_cadyn = true;
    if (T.type == CN_SK) has_sk = true;
    if (T.type == CN_HHFORM && T.glob[3] != 0.0) has_caform = true;
  }
  m->any_ica = has_cadyn || has_caform;
  m->any_cai = has_cadyn || has_sk;
  if (m->any_cai) {
    m->cai0.assign((size_t)N, 1e-4);
    for (const HTable &T : m->tab)
      if (T.type == CN_CADYN)
        for (int64_t i = 0; i < T.n; ++i) m->cai0[T.node[i]] = T.glob[3];
  }

  // ---- strategy per class (north_star: interleaved one-lane-per-cell versus warp-cooperative) --
  // A class with >= 32 same-shape cells is integrated 32 cells per warp by the tape kernel when
  // the model is large enough to fill the GPU that way; everything else (small classes, small
  // models, the ragged remainder of a class) goes to the warp-cooperative kernel.
  int tape_mode = -1;  // -1 auto, 0 off, 1 on
  if (const char *e = m->opt("tape")) tape_mode = std::atoi(e);
  int64_t tape_min_cells = 8192;
  if (const char *e = m->opt("tape_min_cells")) tape_min_cells = std::atoll(e);
  int tape_min_group = 16;  // a ragged last group needs at least this many cells
  if (const char *e = m->opt("tape_min_group")) tape_min_group = std::max(1, std::atoi(e));
  // A smaller model goes to the interleaved kernel too if ALL of it fits there (then it runs in
  // window mode: one launch per min-delay window instead of three per dt) and its groups fill at
  // least a quarter of their lanes; decided after the programs are compiled (below).
  // A small model whose cells can all be RESIDENT ON CHIP AT ONCE (one CTA per cell, cn_cell.cuh)
  // goes to the on-chip window kernel instead: it then never streams from HBM inside a min-delay
  // window (config 1: 8.2 instead of 13.0 us per dt; config 2: 23 instead of 61).  Estimated here
  // for a 148-SM device; finalize() checks the real one and the delays (fallback: one launch
  // sequence per dt on the warp-cooperative kernel).
  int onchip_opt = -1;
  if (const char *e = m->opt("onchip")) onchip_opt = std::atoi(e);
  bool prefer_onchip = false;
  if (tape_mode == -1 && onchip_opt != 0 && nc > 0 && nc < tape_min_cells) {
    size_t max_bytes = 0;
    int max_n = 1;
    for (const HClass &K : m->cls) {
      size_t d = (size_t)K.n * (9 + (m->any_ica ? 1 : 0) + (m->any_cai ? 1 : 0));
      for (const HTable &T : m->tab)
        if (!T.ti.point && T.type != CN_PAS)
          d += (size_t)(T.ti.n_dev_param + T.ti.n_state) *
               (size_t)(T.cell_first[K.rep_cell + 1] - T.cell_first[K.rep_cell]);
      max_bytes = std::max(max_bytes, d * 8 + (size_t)K.n * 24);  // (+ the elimination plan)
      max_n = std::max(max_n, K.n);
    }
    const int threads = max_n <= 128 ? 64 : max_n <= 320 ? 128 : 256;
    const size_t per_sm = std::min<size_t>(std::min(32, 2048 / threads), (227 * 1024) / (max_bytes + 1024));
    prefer_onchip = max_bytes <= 220 * 1024 && (size_t)nc <= 148 * per_sm;
    for (const HTable &T : m->tab)
      if (T.type == CN_GAP && T.n > 0) prefer_onchip = false;
  }
  const bool auto_small = tape_mode == -1 && nc < tape_min_cells && nc > 0 && !prefer_onchip;
  if (auto_small && !m->opt("tape_min_group")) tape_min_group = 1;
  const bool tape_on = tape_mode == 1 || (tape_mode == -1 && nc >= tape_min_cells) || auto_small;
  // W warps per group (CTA), each with a ring of S chunks x CH rows; the whole CTA must fit the
  // 227 KB of shared memory next to the group's system (512 B per node)
  m->tape_W = 8;
  {
    // A model with fewer groups than SMs cannot fill two CTAs per SM anyway and its dt is the
    // latency of one (step, group) item: 12 warps per group shorten the item (config 3: 114 groups,
    // 60.7 -> 54.7 us per dt; 16 warps: 55.2).
    int64_t est_groups = 0;
    for (const HClass &K : m->cls) est_groups += ((int64_t)K.cells.size() + 31) / 32;
    if (est_groups > 0 && est_groups <= 148) m->tape_W = 12;
  }
  if (const char *e = m->opt("tape_w")) m->tape_W = std::min(16, std::max(1, std::atoi(e)));
  m->tape_S = 2;
  m->tape_CH = 16;
  if (const char *e = m->opt("tape_s")) m->tape_S = std::min(4, std::max(2, std::atoi(e)));
  if (const char *e = m->opt("tape_ch")) m->tape_CH = std::min(63, std::max(7, std::atoi(e)));
  if (const char *e = m->opt("tape_tmem")) m->tape_tmem = std::atoi(e) != 0;
  if (const char *e = m->opt("tape_leaf_first")) m->tape_leaf_first = std::atoi(e) != 0;
  if (const char *e = m->opt("tape_hcost")) m->tape_hcost = std::atof(e);
  if (const char *e = m->opt("tape_gran")) m->tape_gran = std::max(1.0, std::atof(e));
  if (const char *e = m->opt("tape_mcost")) m->tape_mcost_scale = std::atof(e);
  if (const char *e = m->opt("tape_bcost")) m->tape_bcost = std::atof(e);
  m->cell_tape.assign(nc, 0);
  for (HClass &K : m->cls) {
    K.count = (int64_t)K.cells.size();
    K.tp.n_groups = 0;
    K.tp.n_cells = 0;
    if (!tape_on || nt > 20) continue;
    const int64_t full = K.count / 32, rem = K.count % 32;
    K.tp.n_groups = (int)(full + (rem >= tape_min_group ? 1 : 0));
    K.tp.n_cells = std::min<int64_t>(K.count, (int64_t)K.tp.n_groups * 32);
    if (K.tp.n_groups > 0) K.tp.has_pp.assign(K.n, 0);
  }
  // a point process on any cell of the class marks its local node (two dynamic rows there)
  for (int t = 0; t < nt; ++t) {
    const HTable &T = m->tab[t];
    if (!T.ti.point) continue;
    for (int64_t i = 0; i < T.n; ++i) {
      const int32_t c = cell_of[T.node[i]];
      HTape &P = m->cls[m->cell_cls[c]].tp;
      if (P.n_groups > 0) P.has_pp[T.node[i] - m->cell_first[c]] = 1;
    }
  }
  lap("classes");
  // chunk size: the default suits plain nodes (three 5-row records); a model whose mechanism
  // records are longer gets chunks of that length (a dry pass over the classes finds out)
  int min_ch = 7;  // the longest record of any class (a chunk holds whole records)
  if (!m->opt("tape_ch")) {
    int need = 0;
    for (const HClass &K : m->cls) {
      if (K.tp.n_groups == 0) continue;
      // rows of the longest mechanism record of the class: v copy, [cai], [ica], table rows
      std::vector<int> rows(K.n, 0);
      std::vector<uint8_t> cai(K.n, 0), ica(K.n, 0);
      const int64_t f = m->cell_first[K.rep_cell];
      for (int t = 0; t < nt; ++t) {
        const HTable &T = m->tab[t];
        if (T.ti.point || T.type == CN_PAS) continue;
        for (int64_t q = T.cell_first[K.rep_cell]; q < T.cell_first[K.rep_cell + 1]; ++q) {
          const int x = (int)(T.node[T.inst(q)] - f);
          rows[x] += tape_rows_of(T.ti, T.type);
          if (T.type == CN_CADYN) cai[x] = ica[x] = 1;
          if (T.type == CN_SK) cai[x] = 1;
        }
      }
      for (int x = 0; x < K.n; ++x)
        if (rows[x] || cai[x]) need = std::max(need, 1 + cai[x] + ica[x] + rows[x]);
    }
    if (need > m->tape_CH && need <= 63) m->tape_CH = need;
    min_ch = std::max(need, 7);
  }
  lap("chunk-length pass");
  std::vector<std::pair<int, int64_t>> saved_groups;
  for (const HClass &K : m->cls) saved_groups.emplace_back(K.tp.n_groups, K.tp.n_cells);
  for (;;) {  // the classes are independent: compile their programs on all host cores
    std::vector<int> todo;
    for (int kc = 0; kc < (int)m->cls.size(); ++kc)
      if (m->cls[kc].tp.n_groups > 0) todo.push_back(kc);
    const unsigned hw = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
    const unsigned nth = (unsigned)std::min<size_t>(hw, std::max<size_t>(1, todo.size() / 8));
    std::vector<int> rcs(nth, CN_OK);
    auto work = [&](unsigned tix) {
      for (size_t j = tix; j < todo.size(); j += nth) {
        const int rc = build_tape_program(m, m->cls[todo[j]]);
        if (rc != CN_OK) rcs[tix] = rc;
      }
    };
    if (nth <= 1) {
      work(0);
    } else {
      std::vector<std::thread> pool;
      for (unsigned tix = 0; tix < nth; ++tix) pool.emplace_back(work, tix);
      for (auto &th : pool) th.join();
    }
    for (int rc : rcs)
      if (rc != CN_OK) return fail(rc, "internal: compiling a tape program failed");
    // Two CTAs per SM need 2 x (shared memory + 1 KB) <= 228 KB: if the rings are what is in the
    // way, shorter chunks (12, 10 rows = 2 plain nodes) cost less than the second CTA is worth.
    size_t sys_cap = 1, prog_cap = 1, bar_cap = 0;
    for (const HClass &K : m->cls) {
      if (K.tp.n_groups == 0) continue;
      sys_cap = std::max(sys_cap, (size_t)K.tp.n_srow);
      prog_cap = std::max(prog_cap, K.tp.prog.size());
      bar_cap = std::max(bar_cap, (size_t)K.tp.n_bar);
    }
    const size_t smem = (size_t)m->tape_W * m->tape_S * m->tape_CH * 256 + sys_cap * 512 +
                        prog_cap * 16 + ((size_t)m->tape_W * m->tape_S + 2 + bar_cap) * 8 + 16;
    int next_ch = 0;
    for (int c : {12, 10})
      if (c < m->tape_CH && c >= min_ch && next_ch == 0) next_ch = c;
    if (m->tape_W > 8 || m->opt("tape_ch") || 2 * (smem + 1024) <= 233472 || next_ch == 0 ||
        2 * (smem - (size_t)m->tape_W * m->tape_S * (m->tape_CH - 10) * 256 + 1024) > 233472)
      break;
    m->tape_CH = next_ch;
    for (size_t kc = 0; kc < m->cls.size(); ++kc) {
      m->cls[kc].tp.n_groups = saved_groups[kc].first;
      m->cls[kc].tp.n_cells = saved_groups[kc].second;
    }
  }
  int prog_total = 0;
  for (HClass &K : m->cls) {
    if (K.tp.n_groups == 0) continue;
    // the CTA must fit: rings + system + two program buffers + counters and barriers
    const size_t sys_cap = (size_t)std::max(m->tape_sys_cap, K.tp.n_srow);
    const size_t prog_cap = std::max((size_t)m->tape_prog_cap, K.tp.prog.size());
    const size_t need = (size_t)m->tape_W * m->tape_S * m->tape_CH * 256 + sys_cap * 512 +
                        prog_cap * 16 +
                        ((size_t)m->tape_W * m->tape_S + 2 + std::max(m->tape_bar_cap, K.tp.n_bar)) * 8 + 16;
    if (need > 227 * 1024) {
      K.tp.n_groups = 0;
      K.tp.n_cells = 0;
      continue;
    }
    for (int64_t q = 0; q < K.tp.n_cells; ++q) m->cell_tape[K.cells[q]] = 1;
    K.tp.prog_off = prog_total;
    prog_total += (int)K.tp.prog.size();
    m->tape_prog_cap = std::max(m->tape_prog_cap, (int)K.tp.prog.size());
    m->tape_sys_cap = std::max(m->tape_sys_cap, K.tp.n_srow);
    m->tape_bar_cap = std::max(m->tape_bar_cap, K.tp.n_bar);
  }
  if (auto_small) {
    int64_t cells = 0, groups = 0;
    bool all = true;
    for (const HClass &K : m->cls) {
      cells += K.tp.n_cells;
      groups += K.tp.n_groups;
      if (K.tp.n_cells < K.count) all = false;
    }
    for (const HTable &T : m->tab)
      if ((T.type == CN_AMPANMDA || T.type == CN_GAP) && T.n > 0)
        all = false;  // (no window mode with these)
    if (!all || cells * 4 < groups * 32) {  // back to the warp-cooperative kernel, all of it
      for (HClass &K : m->cls) {
        K.tp.n_groups = 0;
        K.tp.n_cells = 0;
      }
      std::fill(m->cell_tape.begin(), m->cell_tape.end(), 0);
      m->tape_prog_cap = m->tape_sys_cap = m->tape_bar_cap = 0;
    }
  }

  lap("tape programs");
  // ---- warp-cooperative groups: choose G per class and schedule ------------------------------
  int force_g = 0;
  if (const char *e = m->opt("force_g")) force_g = std::atoi(e);
  int max_g = 4;
  if (const char *e = m->opt("max_g")) max_g = std::max(1, std::atoi(e));
  if (onchip_opt == 1 || prefer_onchip) max_g = 1;  // the on-chip window kernel keeps one cell per CTA
  int64_t smem_cap = 24 * 1024;
  if (const char *e = m->opt("warp_smem")) smem_cap = std::atoll(e);
  const int64_t hard_cap = 200 * 1024;
  int sched_total = 0, nodeoff_total = 0;
  m->warp_smem_doubles = 0;
  int64_t coop_cells = 0;
  for (const HClass &K : m->cls) coop_cells += K.count - K.tp.n_cells;
  for (HClass &K : m->cls) {
    K.needs_ica = m->any_ica ? 1 : 0;
    const int64_t ccount = K.count - K.tp.n_cells;  // cells left for the cooperative kernel
    K.sched.clear();
    K.node_off.assign(K.n, 0);
    if (ccount == 0) {
      K.G = 1; K.lgG = 0; K.rounds = 0;
      K.sched_off = sched_total;
      K.nodeoff_off = nodeoff_total;
      nodeoff_total += K.n;
      continue;
    }
    const int arrays = 2 + K.needs_ica;
    if ((int64_t)K.n * arrays * 8 > hard_cap)
      return fail(CN_ERR_UNSUPPORTED,
                  "a cell with %d nodes does not fit the on-chip solve (limit %lld nodes)", K.n,
                  (long long)(hard_cap / (arrays * 8)));
    // several cells per warp only while that still leaves every SM its 8 warps: below that, more
    // lanes per cell (fewer rounds, fewer mechanism passes per warp) beat more cells per warp
    // (config 2, 256 cells x 601 nodes: 94.9 us per dt with G = 1, 110.7 with G = 2)
    // ... and never for cells that carry distributed mechanisms on most of their nodes (config 5:
    // Ih on every dendritic node): their mechanism loops want all 32 lanes and the occupancy that
    // the smaller system leaves (config 5 at quarter scale: step kernel 288 us per dt with one cell
    // per warp, 362 with two)
    int64_t mech_inst = 0;
    for (const HTable &T : m->tab)
      if (!T.ti.point && T.type != CN_PAS)
        mech_inst += T.cell_first[K.rep_cell + 1] - T.cell_first[K.rep_cell];
    const int class_max_g = mech_inst >= K.n ? 1 : max_g;
    int G = 1;
    while (G * 2 <= class_max_g && G * 2 <= ccount && (int64_t)K.n * arrays * 8 * G * 2 <= smem_cap &&
           coop_cells / (G * 2) >= 148 * 8)
      G *= 2;
    if (force_g > 0) {
      G = 1;
      while (G * 2 <= force_g && (int64_t)K.n * arrays * 8 * G * 2 <= hard_cap) G *= 2;
    }
    K.G = G;
    K.lgG = 0;
    while ((1 << K.lgG) < G) K.lgG++;
    std::vector<int32_t> pl(K.n);
    const int64_t f = m->cell_first[K.rep_cell];
    pl[0] = -1;
    for (int i = 1; i < K.n; ++i) pl[i] = (int32_t)(m->parent[f + i] - f);
    K.rounds = hu_schedule(K.n, pl.data(), 32 / G, K.sched);
    K.sched_off = sched_total;
    sched_total += (int)K.sched.size();
    K.node_off[0] = K.rounds * 32;
    for (int r = 0; r < K.rounds; ++r)
      for (int p = 0; p < 32 / G; ++p) {
        const uint32_t e = K.sched[(size_t)r * (32 / G) + p];
        if ((e & 0xFFFFu) != CN_IDLE) K.node_off[e & 0xFFFFu] = r * 32 + p * G;
      }
    K.nodeoff_off = nodeoff_total;
    nodeoff_total += K.n;
    m->warp_smem_doubles = std::max(m->warp_smem_doubles, K.n * G * arrays);
  }
  // groups: cooperative groups first, then tape groups
  m->cell_grp.assign(nc, -1);
  m->cell_slot.assign(nc, 0);
  m->node_pos.resize((size_t)N);
  int64_t node_base = 0, ab_base = 0;
  int32_t cell_base = 0;
  for (int kc = 0; kc < (int)m->cls.size(); ++kc) {
    HClass &K = m->cls[kc];
    for (int64_t q = K.tp.n_cells; q < K.count; q += K.G) {
      GroupInfo gi{};
      gi.cls = kc;
      gi.ncell = (int32_t)std::min<int64_t>(K.G, K.count - q);
      gi.cell_base = cell_base;
      gi.node_base = node_base;
      gi.ab_base = ab_base;
      const int gidx = (int)m->grp.size();
      for (int c = 0; c < gi.ncell; ++c) {
        const int32_t cell = K.cells[q + c];
        m->cell_grp[cell] = gidx;
        m->cell_slot[cell] = c;
      }
      m->grp.push_back(gi);
      node_base += (int64_t)K.n * K.G;
      ab_base += (int64_t)(K.rounds + 1) * 32;
      cell_base += K.G;
    }
  }
  m->n_pnode = ab_base;  // all node arrays of the cooperative kernel live in schedule order
  m->n_ab = ab_base;
  m->n_cgroup = (int)m->grp.size();
  const int ngc = m->n_cgroup;
  int64_t tape_base = 0;
  for (int kc = 0; kc < (int)m->cls.size(); ++kc) {
    HClass &K = m->cls[kc];
    for (int gq = 0; gq < K.tp.n_groups; ++gq) {
      TapeGroup tg{};
      tg.cls = kc;
      tg.tape_base = tape_base;
      tg.cell_base = cell_base;
      tg.ncell = (int32_t)std::min<int64_t>(32, K.tp.n_cells - (int64_t)gq * 32);
      tg.pp_base = m->win_stride;
      m->win_stride += (int64_t)K.tp.n_pp * 64;
      const int gidx = ngc + (int)m->tgrp.size();
      for (int c = 0; c < tg.ncell; ++c) {
        const int32_t cell = K.cells[(int64_t)gq * 32 + c];
        m->cell_grp[cell] = gidx;
        m->cell_slot[cell] = c;
      }
      m->tgrp.push_back(tg);
      tape_base += (int64_t)K.tp.n_rows * 32;
      cell_base += 32;
    }
  }
  m->n_tape = tape_base;
  if (m->n_tape >= ((int64_t)1 << 32))
    return fail(CN_ERR_UNSUPPORTED, "tape larger than 2^32 doubles");
  m->n_pcell = cell_base;
  const int ng = ngc + (int)m->tgrp.size();
  // caller node -> element of the voltage arena
  par_for(nc, 256, [&](int64_t c0, int64_t c1) {
    for (int64_t cell = c0; cell < c1; ++cell) {
      const int g = m->cell_grp[cell];
      const int c = m->cell_slot[cell];
      const int64_t f = m->cell_first[cell];
      if (g < ngc) {
        const GroupInfo &gi = m->grp[g];
        const HClass &K = m->cls[gi.cls];
        for (int i = 0; i < K.n; ++i) m->node_pos[f + i] = gi.ab_base + K.node_off[i] + c;
      } else {
        const TapeGroup &tg = m->tgrp[g - ngc];
        const HClass &K = m->cls[tg.cls];
        for (int i = 0; i < K.n; ++i)
          m->node_pos[f + i] =
              m->n_ab + tg.tape_base + ((int64_t)K.tp.row[K.tp.pos_of[i]] + 4) * 32 + c;
      }
    }
  });
  // per-table instance layout
  std::vector<int32_t> dist_nodes;
  for (int t = 0; t < nt; ++t) {
    HTable &T = m->tab[t];
    // (pas is folded into the static rows: its instances have no place of their own)
    const bool placed = T.type != CN_PAS;
    if (placed) {
      T.inst_pos.resize((size_t)T.n);
      par_for(T.n, 1 << 18, [&](int64_t i0, int64_t i1) {
        std::fill(T.inst_pos.begin() + i0, T.inst_pos.begin() + i1, (int64_t)-1);
      });
    }
    if (T.ti.point) {
      // instances ordered by group (stable); cooperative groups: slot = local node * G + cell
      // slot in shared memory; tape groups: element of the node's conductance row on the tape
      uvec<int64_t> rank;
      par_bucket(T.n, ng, [&](int64_t i) { return m->cell_grp[cell_of[T.node[i]]]; }, T.pp_first,
                 rank);
      T.pp_slot.resize((size_t)T.n);
      T.pp_wslot.resize((size_t)T.n);
      T.pp_local.resize((size_t)T.n);
      par_for(T.n, 1 << 16, [&](int64_t i0, int64_t i1) {
        for (int64_t i = i0; i < i1; ++i) {
          const int32_t cell = cell_of[T.node[i]];
          const int g = m->cell_grp[cell];
          const int64_t pos = rank[i];
          T.inst_pos[i] = pos;
          const int32_t local = (int32_t)(T.node[i] - m->cell_first[cell]);
          T.pp_local[pos] = local;
          if (g < ngc) {
            // element of the node's row pair in ppdr (schedule order, rows of 32 + 32)
            const int64_t sp = m->grp[g].ab_base + m->cls[m->grp[g].cls].node_off[local] +
                               m->cell_slot[cell];
            T.pp_slot[pos] = (int32_t)(uint32_t)((sp >> 5) * 64 + (sp & 31));
            T.pp_wslot[pos] = 0;
          } else {
            const TapeGroup &tg = m->tgrp[g - ngc];
            const int64_t el = tg.tape_base + (int64_t)m->cls[tg.cls].tp.pp_row[local] * 32 +
                               m->cell_slot[cell];
            T.pp_slot[pos] = (int32_t)(uint32_t)el;
            T.pp_wslot[pos] = (uint32_t)(tg.pp_base + (int64_t)m->cls[tg.cls].tp.pp_ord[local] * 64 +
                                         m->cell_slot[cell]);
          }
        }
      });
      T.pp_tape_begin = T.pp_first[ngc];
      T.n_dev = T.n;
    } else {
      if (placed) {
        T.tape_loc.resize((size_t)T.n);
        par_for(T.n, 1 << 18, [&](int64_t i0, int64_t i1) {
          std::fill(T.tape_loc.begin() + i0, T.tape_loc.begin() + i1, (int64_t)-1);
        });
      }
      T.cls_cnt.assign(m->cls.size(), 0);
      T.cls_nodeoff.assign(m->cls.size(), 0);
      for (int kc = 0; kc < (int)m->cls.size(); ++kc) {
        const HClass &K = m->cls[kc];
        const int32_t rc = K.rep_cell;
        T.cls_cnt[kc] = (int32_t)(T.cell_first[rc + 1] - T.cell_first[rc]);
        T.cls_nodeoff[kc] = (int32_t)dist_nodes.size();
        for (int64_t j = T.cell_first[rc]; j < T.cell_first[rc + 1]; ++j)
          dist_nodes.push_back((int32_t)(T.node[T.inst(j)] - m->cell_first[rc]));
      }
      T.grp_instbase.assign((size_t)std::max(ngc, 1), 0);
      int64_t base = 0;
      for (int g = 0; g < ngc; ++g) {
        const GroupInfo &gi = m->grp[g];
        const HClass &K = m->cls[gi.cls];
        const int cnt = T.cls_cnt[gi.cls];
        T.grp_instbase[g] = base;
        base += (int64_t)cnt * K.G;
      }
      T.n_dev = base;
      if (placed)
       par_for(nc, 256, [&](int64_t cc0, int64_t cc1) {
       for (int64_t c = cc0; c < cc1; ++c) {
        const int g = m->cell_grp[c];
        if (g < ngc) {
          const int G = m->cls[m->grp[g].cls].G;
          const int64_t b0 = T.grp_instbase[g];
          int64_t kk = 0;
          for (int64_t j = T.cell_first[c]; j < T.cell_first[c + 1]; ++j, ++kk)
            T.inst_pos[T.inst(j)] = b0 + kk * G + m->cell_slot[c];
        } else if (T.type != CN_CADYN) {
          const TapeGroup &tg = m->tgrp[g - ngc];
          const HTape &P = m->cls[tg.cls].tp;
          for (int64_t j = T.cell_first[c]; j < T.cell_first[c + 1]; ++j) {
            const int64_t i = T.inst(j);
            const int32_t local = (int32_t)(T.node[i] - m->cell_first[c]);
            T.tape_loc[i] = tg.tape_base + (int64_t)P.tab_row[t][local] * 32 + m->cell_slot[c];
          }
        }
       }
      });
    }
  }
  m->dist_nodes = std::move(dist_nodes);
  m->hm.n_group = ngc;
  m->hm.n_tgroup = (int32_t)m->tgrp.size();
  m->hm.n_class = (int32_t)m->cls.size();
  m->hm.n_table = nt;
  static_assert(sizeof(GroupInfo) == 32, "GroupInfo layout");
  static_assert(sizeof(TapeGroup) == 32, "TapeGroup layout");
  // CTA shape of the cooperative kernel: as many warps per block as fit ~100 KB, at most 8
  const int64_t wbytes = std::max<int64_t>((int64_t)m->warp_smem_doubles * 8, 8);
  int wpb = 4;  // (4 warps x 3 CTAs per SM: 170 registers per thread, no spills)
  if (const char *e = m->opt("wpb")) wpb = std::max(1, std::atoi(e));
  while (wpb > 1 && wbytes * wpb > 110 * 1024) wpb /= 2;
  m->wpb = wpb;
  lap("groups, instance layout");
  return CN_OK;
}


