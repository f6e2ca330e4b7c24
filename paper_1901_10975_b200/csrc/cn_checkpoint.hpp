// cn_checkpoint.hpp -- checkpoint / restore and cn_get_state: everything that
// moves dynamic state between the caller's order and the device layout.  Included by cn_api.cu only.
//
// A checkpoint holds the dynamic state after the last step IN THE CALLER'S ORDER: voltages, the
// states of every mechanism table, cai, the threshold flags and the spikes recorded so far.  No
// event queue: the events still in flight are regenerated from the spikes and the NetCon delays
// (L156: in-flight events collapse to their originating spikes).  Nothing of the internal layout
// (tapes, permutations, launch mode) is in the file, and no parameter: it loads into any model
// with the same STRUCTURE (cells, topology, mechanism tables and their nodes), whatever its
// stimuli (IClamp parameters, scripted sources), weights or options -- the paper's "launch
// multiple simulations with different stimuli" (L156).
#pragma once

struct CkHeader {
  uint64_t magic;       // "CNCKPT02"
  int64_t k, n_sp, n_node, n_cell, n_state_doubles, has_cai, total_bytes;
  double dt;
  uint64_t structure;   // hash of cell_first, parent, and (type, n, node[]) of every table
};
static const uint64_t kCkMagic = 0x434E434B50543032ull;

static uint64_t ck_structure_hash(cn_model *m) {
  if (m->ck_hash_done) return m->ck_hash;
  // per-range hashes on all cores, combined in order
  auto hash_range = [&](const void *p, size_t bytes) {
    const unsigned P = std::max(1u, par_threads((int64_t)(bytes / 8), 1 << 18));
    std::vector<uint64_t> part(P, 0);
    const uint64_t *w = static_cast<const uint64_t *>(p);
    const int64_t nw = (int64_t)(bytes / 8);
    par_run(P, [&](unsigned t) {
      uint64_t h = 0x5EEDull + t;
      for (int64_t i = nw * t / P, e = nw * (t + 1) / P; i < e; ++i) h = mix64(h, w[i]);
      part[t] = h;
    });
    uint64_t h = mix64(0xABCDEFull, (uint64_t)bytes);
    for (uint64_t x : part) h = mix64(h, x);
    const unsigned char *tail = static_cast<const unsigned char *>(p) + nw * 8;
    for (size_t i = 0; i < bytes % 8; ++i) h = mix64(h, tail[i]);
    return h;
  };
  uint64_t h = mix64(0xC0FFEEull, (uint64_t)m->N);
  h = mix64(h, (uint64_t)m->n_cell);
  h = mix64(h, hash_range(m->cell_first.data(), m->cell_first.size() * sizeof(int64_t)));
  h = mix64(h, hash_range(m->parent.data(), (size_t)m->N * sizeof(int32_t)));
  for (const HTable &T : m->tab) {
    h = mix64(h, (uint64_t)T.type * 1000003u + (uint64_t)T.n);
    h = mix64(h, hash_range(T.node.data(), (size_t)T.n * sizeof(int32_t)));
  }
  m->ck_hash = h;
  m->ck_hash_done = true;
  return h;
}

static int64_t ck_state_doubles(const cn_model *m) {
  int64_t n = 0;
  for (const HTable &T : m->tab) n += (int64_t)T.ti.n_state * T.n;
  return n;
}

static size_t pad8(size_t b) { return (b + 7) & ~(size_t)7; }

static size_t ck_total_bytes(const cn_model *m, int64_t n_sp) {
  return sizeof(CkHeader) + (size_t)m->N * 8 + (size_t)ck_state_doubles(m) * 8 +
         (m->any_cai ? (size_t)m->N * 8 : 0) + pad8((size_t)m->n_cell) + pad8((size_t)n_sp * 4) +
         (size_t)n_sp * 8;
}

static int ck_spike_count(const cn_model *m, int64_t *n_sp) {
  unsigned long long ns = 0;
  CU(cudaStreamSynchronize(m->stream));
  CU(cudaMemcpy(&ns, m->d_nsp, sizeof(ns), cudaMemcpyDeviceToHost));
  *n_sp = (int64_t)std::min<unsigned long long>(ns, (unsigned long long)m->sp_cap);
  return CN_OK;
}

// device scratch of the model, grown on demand (checkpoints, cn_get_state)
static int ensure_scratch(cn_model *m, size_t bytes) {
  if (bytes <= m->scratch_bytes) return CN_OK;
  if (m->d_scratch) cudaFree(m->d_scratch);
  m->d_scratch = nullptr;
  m->scratch_bytes = 0;
  CU(cudaMalloc(&m->d_scratch, bytes));
  m->scratch_bytes = bytes;
  return CN_OK;
}

// where state s of caller instance i of table T lives: >= 0 element of T.d_state[s], < 0 element
// -(loc + 1) of the tape
static inline int64_t state_loc(const HTable &T, int64_t i, int s) {
  const bool on_tape = !T.ti.point && T.tape_loc[i] >= 0;
  return on_tape ? -(T.tape_loc[i] + (int64_t)(T.ti.n_dev_param + s) * 32 + 1) : T.inst_pos[i];
}

// cai of caller node i: >= 0 element of d_cai, < 0 element -(loc + 1) of the tape, INT64_MIN: the
// node keeps no cai (a tape cell's node without SK / cai dynamics)
static int64_t cai_loc(const cn_model *m, int64_t i, int32_t cell) {
  if (!m->cell_tape[cell]) return m->node_pos[i];
  const TapeGroup &tg = m->tgrp[m->cell_grp[cell] - m->n_cgroup];
  const int32_t r = m->cls[tg.cls].tp.cai_row[i - m->cell_first[cell]];
  if (r < 0) return INT64_MIN;
  return -(tg.tape_base + (int64_t)r * 32 + m->cell_slot[cell] + 1);
}

static const int64_t kCkChunk = (int64_t)1 << 22;  // instances per gather / scatter pass

// out[i0, i1) <-> device, through loc computed by `locf(i)`; to_dev: scatter, else gather
template <class LocF>
static int ck_move(cn_model *m, int64_t n, double *host, const double *alt_c, bool to_dev, LocF &&locf) {
  double *alt = const_cast<double *>(alt_c);
  std::vector<int64_t> loc;
  for (int64_t i0 = 0; i0 < n; i0 += kCkChunk) {
    const int64_t c = std::min(kCkChunk, n - i0);
    loc.resize((size_t)c);
    par_for(c, 1 << 16, [&](int64_t a, int64_t b) {
      for (int64_t i = a; i < b; ++i) loc[i] = locf(i0 + i);
    });
    int rc = ensure_scratch(m, (size_t)kCkChunk * 16);
    if (rc != CN_OK) return rc;
    int64_t *d_loc = static_cast<int64_t *>(m->d_scratch);
    double *d_val = reinterpret_cast<double *>(d_loc + kCkChunk);
    CU(cudaMemcpyAsync(d_loc, loc.data(), (size_t)c * 8, cudaMemcpyHostToDevice, m->stream));
    if (to_dev) {
      CU(cudaMemcpyAsync(d_val, host + i0, (size_t)c * 8, cudaMemcpyHostToDevice, m->stream));
      scatter_state_kernel<<<(unsigned)((c + 255) / 256), 256, 0, m->stream>>>(m->hm.tape, alt, d_loc, c, d_val);
    } else {
      gather_state_kernel<<<(unsigned)((c + 255) / 256), 256, 0, m->stream>>>(m->hm.tape, alt, d_loc, c, 0, d_val);
      CU(cudaMemcpyAsync(host + i0, d_val, (size_t)c * 8, cudaMemcpyDeviceToHost, m->stream));
    }
    m->launches++;
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(m->stream));
  }
  return CN_OK;
}

// nrn_state of the last step is applied at the start of the next one on the interleaved kernel:
// apply it now, so that the states on the tape are the states after the last step
static int flush_pending_state(cn_model *m) {
  if (!m->state_pending || m->hm.n_tgroup == 0) return CN_OK;
  cudaError_t e = launch_tape(m, m->k, TM_ADVANCE | TM_FLUSH);
  if (e != cudaSuccess) return fail(CN_ERR_CUDA, "state flush failed: %s", cudaGetErrorString(e));
  m->launches++;
  m->state_pending = false;
  return CN_OK;
}

static std::vector<int32_t> node_cells(const cn_model *m) {
  std::vector<int32_t> cell_of((size_t)m->N);
  par_for(m->n_cell, 256, [&](int64_t c0, int64_t c1) {
    for (int64_t c = c0; c < c1; ++c)
      for (int64_t i = m->cell_first[c]; i < m->cell_first[c + 1]; ++i) cell_of[i] = (int32_t)c;
  });
  return cell_of;
}

static inline int32_t pcell_of(const cn_model *m, int32_t c) {
  const int g = m->cell_grp[c];
  return (g < m->n_cgroup ? m->grp[g].cell_base : m->tgrp[g - m->n_cgroup].cell_base) + m->cell_slot[c];
}

extern "C" int cn_checkpoint_size(const cn_model *m, int64_t *bytes_out) {
  if (!m || !bytes_out) return fail(CN_ERR_ARG, "NULL argument");
  if (!m->uploaded) return fail(CN_ERR_ARG, "nothing to checkpoint before the first cn_run");
  int64_t n_sp = 0;
  int rc = ck_spike_count(m, &n_sp);
  if (rc != CN_OK) return rc;
  *bytes_out = (int64_t)ck_total_bytes(m, n_sp);
  return CN_OK;
}

extern "C" int cn_checkpoint_save(const cn_model *cm, void *buf, int64_t bytes) {
  cn_model *m = const_cast<cn_model *>(cm);
  if (!m || !buf) return fail(CN_ERR_ARG, "NULL argument");
  if (!m->uploaded) return fail(CN_ERR_ARG, "nothing to checkpoint before the first cn_run");
  int64_t n_sp = 0;
  int rc = ck_spike_count(m, &n_sp);
  if (rc != CN_OK) return rc;
  const size_t tot = ck_total_bytes(m, n_sp);
  if (bytes < 0 || (size_t)bytes < tot) return fail(CN_ERR_ARG, "checkpoint buffer too small (%zu needed)", tot);
  if ((rc = flush_pending_state(m)) != CN_OK) return rc;
  char *p = static_cast<char *>(buf);
  CkHeader h{};
  h.magic = kCkMagic;
  h.k = m->k;
  h.n_sp = n_sp;
  h.n_node = m->N;
  h.n_cell = m->n_cell;
  h.n_state_doubles = ck_state_doubles(m);
  h.has_cai = m->any_cai ? 1 : 0;
  h.total_bytes = (int64_t)tot;
  h.dt = m->dt;
  h.structure = ck_structure_hash(m);
  memcpy(p, &h, sizeof(h));
  p += sizeof(h);
  // voltages
  if (m->N > 0) {
    gather_kernel<<<(unsigned)((m->N + 255) / 256), 256, 0, m->stream>>>(m->d_v, m->d_node_pos, m->N, m->d_gather);
    m->launches++;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(p, m->d_gather, (size_t)m->N * 8, cudaMemcpyDeviceToHost, m->stream));
    CU(cudaStreamSynchronize(m->stream));
  }
  p += (size_t)m->N * 8;
  // mechanism states, table after table, state after state
  for (const HTable &T : m->tab)
    for (int s = 0; s < T.ti.n_state; ++s) {
      rc = ck_move(m, T.n, reinterpret_cast<double *>(p), T.d_state[s], false,
                   [&](int64_t i) { return state_loc(T, i, s); });
      if (rc != CN_OK) return rc;
      p += (size_t)T.n * 8;
    }
  if (m->any_cai) {
    const std::vector<int32_t> cell_of = node_cells(m);
    double *out = reinterpret_cast<double *>(p);
    rc = ck_move(m, m->N, out, m->d_cai, false, [&](int64_t i) {
      const int64_t l = cai_loc(m, i, cell_of[i]);
      return l == INT64_MIN ? (int64_t)0 : l;  // (no storage: read anything, replaced below)
    });
    if (rc != CN_OK) return rc;
    par_for(m->N, 1 << 16, [&](int64_t a, int64_t b) {  // nodes without storage keep their constant
      for (int64_t i = a; i < b; ++i)
        if (cai_loc(m, i, cell_of[i]) == INT64_MIN) out[i] = m->cai0[i];
    });
    p += (size_t)m->N * 8;
  }
  {  // threshold flags, caller cell order
    std::vector<unsigned char> fl((size_t)std::max(m->n_pcell, 1));
    if (m->n_pcell > 0)
      CU(cudaMemcpy(fl.data(), m->hm.flag, (size_t)m->n_pcell, cudaMemcpyDeviceToHost));
    memset(p, 0, pad8((size_t)m->n_cell));
    for (int32_t c = 0; c < m->n_cell; ++c) p[c] = (char)fl[pcell_of(m, c)];
    p += pad8((size_t)m->n_cell);
  }
  {  // spikes sorted by (step, gid)
    std::vector<int32_t> g((size_t)n_sp);
    std::vector<int64_t> s((size_t)n_sp);
    if (n_sp > 0) {
      CU(cudaMemcpy(g.data(), m->d_sp_gid, (size_t)n_sp * 4, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(s.data(), m->d_sp_step, (size_t)n_sp * 8, cudaMemcpyDeviceToHost));
    }
    std::vector<int64_t> ord((size_t)n_sp);
    std::iota(ord.begin(), ord.end(), 0);
    std::sort(ord.begin(), ord.end(), [&](int64_t x, int64_t y) {
      return s[x] != s[y] ? s[x] < s[y] : g[x] < g[y];
    });
    memset(p, 0, pad8((size_t)n_sp * 4));
    int32_t *pg = reinterpret_cast<int32_t *>(p);
    for (int64_t i = 0; i < n_sp; ++i) pg[i] = g[ord[i]];
    p += pad8((size_t)n_sp * 4);
    int64_t *ps = reinterpret_cast<int64_t *>(p);
    for (int64_t i = 0; i < n_sp; ++i) ps[i] = s[ord[i]];
    p += (size_t)n_sp * 8;
  }
  return CN_OK;
}

extern "C" int cn_checkpoint_load(cn_model *m, const void *buf, int64_t bytes) {
  if (!m || !buf) return fail(CN_ERR_ARG, "NULL argument");
  if (bytes < 0 || (size_t)bytes < sizeof(CkHeader)) return fail(CN_ERR_ARG, "not a checkpoint");
  CkHeader h;
  memcpy(&h, buf, sizeof(h));
  // ---- every check comes before the first write to the model -----------------------------------
  if (h.magic != kCkMagic) return fail(CN_ERR_ARG, "not a checkpoint (or one of another library version)");
  if (!std::isfinite(h.dt) || !(h.dt > 0.0)) return fail(CN_ERR_ARG, "checkpoint corrupt: dt");
  if (h.k < 0 || h.n_sp < 0) return fail(CN_ERR_ARG, "checkpoint corrupt: negative count");
  if (h.n_node != m->N || h.n_cell != m->n_cell || h.n_state_doubles != ck_state_doubles(m) ||
      (h.has_cai != 0) != m->any_cai || h.structure != ck_structure_hash(m))
    return fail(CN_ERR_ARG, "checkpoint of a model with a different structure (cells, topology or "
                            "mechanism tables)");
  if (h.n_sp > m->sp_cap) return fail(CN_ERR_OVERFLOW, "checkpoint holds more spikes than the buffer");
  if (h.total_bytes != (int64_t)ck_total_bytes(m, h.n_sp) || bytes < h.total_bytes)
    return fail(CN_ERR_ARG, "checkpoint truncated or corrupt (%lld bytes expected)",
                (long long)ck_total_bytes(m, h.n_sp));
  if (m->uploaded && h.dt != m->dt)
    return fail(CN_ERR_DT, "checkpoint was taken with dt = %.17g, the model runs with %.17g", h.dt, m->dt);
  const char *p = static_cast<const char *>(buf) + sizeof(CkHeader);
  const double *pv = reinterpret_cast<const double *>(p);
  const double *pstate = pv + m->N;
  const double *pcai = pstate + h.n_state_doubles;
  const char *pflag = reinterpret_cast<const char *>(pcai + (m->any_cai ? m->N : 0));
  const int32_t *pgid = reinterpret_cast<const int32_t *>(pflag + pad8((size_t)m->n_cell));
  const int64_t *pstep = reinterpret_cast<const int64_t *>(reinterpret_cast<const char *>(pgid) + pad8((size_t)h.n_sp * 4));
  for (int64_t i = 0; i < h.n_sp; ++i) {
    if (pgid[i] < 0 || pgid[i] >= m->n_cell || pstep[i] < 0 || pstep[i] > h.k ||
        (i > 0 && pstep[i] < pstep[i - 1]))
      return fail(CN_ERR_ARG, "checkpoint corrupt: spike list");
  }
  if (!m->uploaded) {
    int rc = finalize(m, h.dt);
    if (rc != CN_OK) return rc;
  }
  CU(cudaStreamSynchronize(m->stream));
  int rc;
  // ---- voltages (and their copies at the head of the mechanism records of the tapes) ------------
  if (m->N > 0) {
    CU(cudaMemcpyAsync(m->d_gather, pv, (size_t)m->N * 8, cudaMemcpyHostToDevice, m->stream));
    scatter_kernel<<<(unsigned)((m->N + 255) / 256), 256, 0, m->stream>>>(m->d_v, m->d_node_pos, m->N, m->d_gather);
    m->launches++;
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(m->stream));
    if (m->hm.n_tgroup > 0) {
      const std::vector<int32_t> cell_of = node_cells(m);
      uvec<int64_t> idx;
      std::vector<double> val;
      for (int64_t i = 0; i < m->N; ++i) {
        const int32_t c = cell_of[i];
        if (!m->cell_tape[c]) continue;
        const TapeGroup &tg = m->tgrp[m->cell_grp[c] - m->n_cgroup];
        const int32_t r = m->cls[tg.cls].tp.vcopy_row[i - m->cell_first[c]];
        if (r < 0) continue;
        idx.push_back(-(tg.tape_base + (int64_t)r * 32 + m->cell_slot[c] + 1));
        val.push_back(pv[i]);
      }
      rc = ck_move(m, (int64_t)idx.size(), val.data(), nullptr, true, [&](int64_t j) { return idx[j]; });
      if (rc != CN_OK) return rc;
    }
  }
  // ---- mechanism states ----------------------------------------------------------------------------
  {
    const double *q = pstate;
    for (const HTable &T : m->tab)
      for (int s = 0; s < T.ti.n_state; ++s) {
        rc = ck_move(m, T.n, const_cast<double *>(q), T.d_state[s], true,
                     [&](int64_t i) { return state_loc(T, i, s); });
        if (rc != CN_OK) return rc;
        q += T.n;
      }
  }
  if (m->any_cai) {
    const std::vector<int32_t> cell_of = node_cells(m);
    // nodes without storage are skipped: compact the rest
    uvec<int64_t> idx;
    std::vector<double> val;
    idx.reserve((size_t)m->N);
    val.reserve((size_t)m->N);
    for (int64_t i = 0; i < m->N; ++i) {
      const int64_t l = cai_loc(m, i, cell_of[i]);
      if (l == INT64_MIN) continue;
      idx.push_back(l);
      val.push_back(pcai[i]);
    }
    rc = ck_move(m, (int64_t)idx.size(), val.data(), m->d_cai, true, [&](int64_t j) { return idx[j]; });
    if (rc != CN_OK) return rc;
  }
  {  // threshold flags
    std::vector<unsigned char> fl((size_t)std::max(m->n_pcell, 1), 0);
    for (int32_t c = 0; c < m->n_cell; ++c) fl[pcell_of(m, c)] = (unsigned char)(pflag[c] != 0);
    if (m->n_pcell > 0)
      CU(cudaMemcpy(const_cast<unsigned char *>(m->hm.flag), fl.data(), (size_t)m->n_pcell, cudaMemcpyHostToDevice));
  }
  // ---- spikes, and what event delivery derives from them --------------------------------------------
  {
    const DModel &H = m->hm;
    if (h.n_sp > 0) {
      CU(cudaMemcpy(m->d_sp_gid, pgid, (size_t)h.n_sp * 4, cudaMemcpyHostToDevice));
      CU(cudaMemcpy(m->d_sp_step, pstep, (size_t)h.n_sp * 8, cudaMemcpyHostToDevice));
    }
    const unsigned long long ns = (unsigned long long)h.n_sp;
    CU(cudaMemcpy(m->d_nsp, &ns, sizeof(ns), cudaMemcpyHostToDevice));
    CU(cudaMemset(m->d_overflow, 0, sizeof(int32_t)));
    // per-step delivery: sp_end[s % wr] = number of spikes with step <= s, for the steps the next
    // maxd deliveries look back at
    std::vector<int64_t> ring((size_t)H.wr, 0);
    for (int64_t s = std::max<int64_t>(0, h.k - H.wr + 1); s <= h.k; ++s)
      ring[(size_t)(s % H.wr)] = std::upper_bound(pstep, pstep + h.n_sp, s) - pstep;
    CU(cudaMemcpy(H.sp_end, ring.data(), (size_t)H.wr * 8, cudaMemcpyHostToDevice));
    m->win_idx = 0;
    if (m->window || m->cwindow) {
      // window delivery: one mark that stands for all the windows before the restart -- every spike
      // that can still deliver (step >= k - maxd) lies behind it
      const int64_t lo_step = std::max<int64_t>(0, h.k - H.maxd);
      const int64_t lo = std::lower_bound(pstep, pstep + h.n_sp, lo_step) - pstep;
      CU(cudaMemcpy(H.win_mark_step, &lo_step, 8, cudaMemcpyHostToDevice));
      CU(cudaMemcpy(H.win_mark_nsp, &lo, 8, cudaMemcpyHostToDevice));
      m->win_idx = 1;
    }
  }
  CU(cudaDeviceSynchronize());  // (the model's stream may not wait for the legacy default stream)
  m->k = h.k;
  m->state_pending = false;
  m->probe_rows = 0;
  return CN_OK;
}

extern "C" int cn_get_state(const cn_model *cm, int32_t t, int32_t s, double *out, int64_t n) {
  cn_model *m = const_cast<cn_model *>(cm);
  if (!m || !out) return fail(CN_ERR_ARG, "NULL argument");
  if (t < 0 || t >= (int)m->tab.size()) return fail(CN_ERR_MECH, "table out of range");
  HTable &T = m->tab[t];
  if (s < 0 || s >= T.ti.n_state || n != T.n) return fail(CN_ERR_MECH, "state / size mismatch");
  if (!m->uploaded) return fail(CN_ERR_ARG, "states exist after the first cn_run");
  if (n == 0) return CN_OK;
  if (!T.ti.point) {  // the interleaved kernel applies nrn_state of a step at the start of the next
    int rc = flush_pending_state(m);
    if (rc != CN_OK) return rc;
  }
  // instances live in the table arrays (cooperative groups) or on a tape (interleaved groups)
  return ck_move(m, n, out, T.d_state[s], false, [&](int64_t i) { return state_loc(T, i, s); });
}
