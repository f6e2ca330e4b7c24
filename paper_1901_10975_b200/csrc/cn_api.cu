// cn_api.cu -- the C ABI of libcn (include/cn.h): validation and deep copy of the description, the
// step loop, read-back, checkpoints.  The set-up lives in cn_host.hpp (model structure, helpers),
// cn_layout.hpp (shape classes, programs, permutations) and cn_finalize.hpp (dt-dependent tables).
// C ABI declared in include/cn.h.  No CPU compute path exists: every step runs in cn_device.cuh.
#include "../../include/cn.h"
#include "cn_device.cuh"
#include "cn_tape.cuh"
#include "cn_cell.cuh"
#include "cn_expand.cuh"

#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <cctype>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <numeric>
#include <string>
#include <thread>
#include <unordered_map>
#include <vector>

using namespace cn;


#include "cn_host.hpp"

// ---------------------------------------------------------------------------------------------
// create: validate + deep copy + shape classes + permutation (dt-independent part)
// ---------------------------------------------------------------------------------------------

static bool finite_all(const double *x, int64_t n) {
  for (int64_t i = 0; i < n; ++i)
    if (!std::isfinite(x[i])) return false;
  return true;
}

static int build_layout(cn_model *m);
static void raw_upload(cn_model *m, int dev, int64_t N, const double *cm, const double *ri,
                       const double *area, const std::vector<RawSrc> &tabs);

extern "C" int cn_model_create(const cn_model_desc *de, cn_model **out) {
  return cn_model_create_opts(de, nullptr, out);
}

extern "C" int cn_model_create_opts(const cn_model_desc *de, const char *options, cn_model **out) {
  if (out) *out = nullptr;
  if (!de || !out) return fail(CN_ERR_ARG, "cn_model_create: NULL argument");
  Options parsed;
  if (int rc = parsed.parse(options)) return rc;
  const bool dbg = parsed.get("debug") && std::atoi(parsed.get("debug")) != 0;
  auto t_prev = std::chrono::steady_clock::now();
  auto lap = [&](const char *what) {
    if (!dbg) return;
    const auto t = std::chrono::steady_clock::now();
    fprintf(stderr, "[cn] create %-34s %7.1f ms\n", what,
            std::chrono::duration<double, std::milli>(t - t_prev).count());
    t_prev = t;
  };
  if (de->n_cell < 0 || de->n_node < 0) return fail(CN_ERR_ARG, "negative sizes");
  if (de->n_node >= (int64_t)1 << 31) return fail(CN_ERR_ARG, "n_node must be < 2^31");
  if (de->n_mech < 0 || de->n_mech > CN_MAX_TABLES)
    return fail(CN_ERR_MECH, "n_mech must be in [0, %d]", CN_MAX_TABLES);
  const int64_t N = de->n_node;
  if (de->n_mech > 0 && !de->mech) return fail(CN_ERR_MECH, "NULL mechanism table array");
  if (de->n_cell > 0 &&
      (!de->cell_first || !de->parent || !de->area_um2 || !de->ri_MOhm || !de->cm_uF_cm2 ||
       !de->thr_mV))
    return fail(CN_ERR_ARG, "NULL node / cell array");
  if (de->n_cell > 0 && (de->cell_first[0] != 0 || de->cell_first[de->n_cell] != N))
    return fail(CN_ERR_TOPOLOGY, "cell_first must start at 0 and end at n_node");
  if (de->n_cell == 0 && N != 0) return fail(CN_ERR_TOPOLOGY, "nodes without cells");
  {  // cells: monotone cell_first first (the parallel pass below reads ranges from it)
    FirstErr fe;
    par_for(de->n_cell, 4096, [&](int64_t c0, int64_t c1) {
      for (int64_t c = c0; c < c1; ++c) {
        const int64_t f = de->cell_first[c], l = de->cell_first[c + 1];
        if (f < 0 || l > N || l <= f) return fe.set(c, CN_ERR_TOPOLOGY, "cell %lld is empty", (long long)c);
        if (l - f > 65534)
          return fe.set(c, CN_ERR_UNSUPPORTED, "cell %lld has more than 65534 nodes", (long long)c);
      }
    });
    if (fe.code != CN_OK) return fail(fe.code, "%s", fe.msg);
    par_for(de->n_cell, 256, [&](int64_t c0, int64_t c1) {
      for (int64_t c = c0; c < c1; ++c) {
        const int64_t f = de->cell_first[c], l = de->cell_first[c + 1];
        if (de->parent[f] != -1)
          return fe.set(f, CN_ERR_TOPOLOGY, "root of cell %lld has a parent", (long long)c);
        for (int64_t i = f + 1; i < l; ++i)
          if (de->parent[i] < f || de->parent[i] >= i)
            return fe.set(i, CN_ERR_TOPOLOGY,
                          "parent[%lld] = %d violates parent < child inside cell %lld",
                          (long long)i, de->parent[i], (long long)c);
      }
    });
    if (fe.code != CN_OK) return fail(fe.code, "%s", fe.msg);
  }
  if (!finite_all(de->thr_mV, de->n_cell) || !std::isfinite(de->v_init_mV) ||
      !std::isfinite(de->celsius))
    return fail(CN_ERR_ARG, "non-finite value in a node / cell array");
  {
    FirstErr fe;
    par_for(N, 1 << 16, [&](int64_t i0, int64_t i1) {
      for (int64_t i = i0; i < i1; ++i) {
        const double ar = de->area_um2[i], r = de->ri_MOhm[i], c = de->cm_uF_cm2[i];
        if (!std::isfinite(ar) || !std::isfinite(r) || !std::isfinite(c))
          return fe.set(i, CN_ERR_ARG, "non-finite value in a node / cell array (node %lld)",
                        (long long)i);
        if (!(ar > 0.0) || !(c > 0.0))
          return fe.set(i, CN_ERR_ARG, "area and cm must be > 0 (node %lld)", (long long)i);
        if (de->parent[i] >= 0 && !(r > 0.0))
          return fe.set(i, CN_ERR_ARG, "ri must be > 0 (node %lld)", (long long)i);
      }
    });
    if (fe.code != CN_OK) return fail(fe.code, "%s", fe.msg);
  }
  for (int32_t t = 0; t < de->n_mech; ++t) {
    const cn_mech_table &mt = de->mech[t];
    TypeInfo ti;
    if (!type_info(mt.type, ti)) return fail(CN_ERR_MECH, "table %d: unknown type %d", t, mt.type);
    if (mt.n < 0 || mt.n_param != ti.n_param || mt.n_global != ti.n_global)
      return fail(CN_ERR_MECH, "table %d: type %d needs %d params and %d globals", t, mt.type,
                  ti.n_param, ti.n_global);
    if (mt.n > 0 && (!mt.node || (ti.n_param > 0 && !mt.param)))
      return fail(CN_ERR_MECH, "table %d: NULL array", t);
    if (ti.n_global > 0 && !mt.global) return fail(CN_ERR_MECH, "table %d: NULL globals", t);
    if (!finite_all(mt.global, ti.n_global))
      return fail(CN_ERR_MECH, "table %d: non-finite parameter", t);
    if (mt.type == CN_HHFORM)
      for (int j : {5, 9, 11, 15})
        if (mt.global[j] == 0.0)
          return fail(CN_ERR_MECH, "table %d: gate slope constants k and sigma must be non-zero", t);
    FirstErr fe;
    par_for(mt.n, 1 << 16, [&](int64_t i0, int64_t i1) {
      for (int64_t i = i0; i < i1; ++i) {
        if (mt.node[i] < 0 || mt.node[i] >= N)
          return fe.set(i, CN_ERR_MECH, "table %d: node of instance %lld out of range", t,
                        (long long)i);
        for (int j = 0; j < ti.n_param; ++j)
          if (!std::isfinite(mt.param[(int64_t)j * mt.n + i]))
            return fe.set(i, CN_ERR_MECH, "table %d: non-finite parameter", t);
        if (mt.type == CN_EXP2SYN && (!(mt.param[i] > 0.0) || !(mt.param[mt.n + i] > mt.param[i])))
          return fe.set(i, CN_ERR_MECH, "table %d: Exp2Syn needs 0 < tau1 < tau2", t);
        if (mt.type == CN_EXPSYN && !(mt.param[i] > 0.0))
          return fe.set(i, CN_ERR_MECH, "table %d: ExpSyn needs tau > 0", t);
        if (mt.type == CN_GAP) {
          const double pr = mt.param[mt.n + i];
          if (!(pr >= 0.0 && pr < (double)N) || pr != (double)(int64_t)pr)
            return fe.set(i, CN_ERR_MECH, "table %d: gap junction %lld has no such peer node", t,
                          (long long)i);
        }
      }
    });
    if (fe.code != CN_OK) return fail(fe.code, "%s", fe.msg);
  }
  if (de->n_netcon < 0 || de->n_stim < 0) return fail(CN_ERR_NETCON, "negative count");
  if (de->n_netcon > 0 && (!de->nc_src_gid || !de->nc_tgt_mech || !de->nc_tgt_inst ||
                           !de->nc_weight_uS || !de->nc_delay_ms))
    return fail(CN_ERR_NETCON, "NULL NetCon array with n_netcon > 0");
  if (de->n_stim > 0 && (!de->stim_gid || !de->stim_t_ms))
    return fail(CN_ERR_NETCON, "NULL scripted-source array with n_stim > 0");
  int32_t n_src = de->n_cell;
  {
    FirstErr fe;
    std::mutex mu;
    par_for(de->n_netcon, 1 << 16, [&](int64_t i0, int64_t i1) {
      int32_t hi = 0;
      for (int64_t i = i0; i < i1; ++i) {
        const int32_t tm = de->nc_tgt_mech[i];
        if (tm < 0 || tm >= de->n_mech)
          return fe.set(i, CN_ERR_NETCON, "netcon %lld: bad table", (long long)i);
        const int ty = de->mech[tm].type;
        if (ty != CN_EXPSYN && ty != CN_EXP2SYN && ty != CN_AMPANMDA)
          return fe.set(i, CN_ERR_NETCON, "netcon %lld: target type %d receives no events",
                        (long long)i, ty);
        if (de->nc_tgt_inst[i] < 0 || de->nc_tgt_inst[i] >= de->mech[tm].n)
          return fe.set(i, CN_ERR_NETCON, "netcon %lld: target instance out of range", (long long)i);
        if (de->nc_src_gid[i] < 0)
          return fe.set(i, CN_ERR_NETCON, "netcon %lld: negative source", (long long)i);
        if (!std::isfinite(de->nc_weight_uS[i]) || !std::isfinite(de->nc_delay_ms[i]) ||
            !(de->nc_delay_ms[i] > 0.0))
          return fe.set(i, CN_ERR_NETCON, "netcon %lld: weight / delay invalid", (long long)i);
        hi = std::max(hi, de->nc_src_gid[i] + 1);
      }
      std::lock_guard<std::mutex> lk(mu);
      n_src = std::max(n_src, hi);
    });
    if (fe.code != CN_OK) return fail(fe.code, "%s", fe.msg);
  }
  for (int64_t i = 0; i < de->n_stim; ++i) {
    if (de->stim_gid[i] < de->n_cell)
      return fail(CN_ERR_NETCON, "scripted source %lld: gid must be >= n_cell", (long long)i);
    if (!std::isfinite(de->stim_t_ms[i]) || de->stim_t_ms[i] < 0.0)
      return fail(CN_ERR_NETCON, "scripted source %lld: time invalid", (long long)i);
    n_src = std::max(n_src, de->stim_gid[i] + 1);
  }

  lap("validation");
  cn_model *m = new (std::nothrow) cn_model();
  if (!m) return fail(CN_ERR_NOMEM, "out of host memory");
  // A model that is headed for the interleaved kernel: its compact arrays travel to the device on
  // a thread of their own while the cores below copy the description and compile the layout
  // (cn_expand.cuh).  Joined before this call returns or fails.
  std::thread raw_thread;
  bool raw_started = false;
  auto raw_join = [&] {
    if (raw_thread.joinable()) raw_thread.join();
  };
  {
    int tape_mode = -1, dev = 0;
    int64_t tape_min_cells = 8192;
    if (const char *e = parsed.get("tape")) tape_mode = std::atoi(e);
    if (const char *e = parsed.get("tape_min_cells")) tape_min_cells = std::atoll(e);
    const bool headed = tape_mode == 1 || (tape_mode == -1 && de->n_cell >= tape_min_cells);
    if (headed && N >= (1 << 16) && de->n_mech <= 20 && cudaGetDevice(&dev) == cudaSuccess) {
      std::vector<RawSrc> src((size_t)de->n_mech);
      for (int32_t t = 0; t < de->n_mech; ++t) {
        const cn_mech_table &mt = de->mech[t];
        TypeInfo ti;
        type_info(mt.type, ti);
        src[t] = RawSrc{mt.node, mt.param, mt.n, ti.n_param, !ti.point && ti.n_param > 0 && mt.n > 0};
      }
      m->raw.param.assign((size_t)de->n_mech, nullptr);
      m->raw.node.assign((size_t)de->n_mech, nullptr);
      raw_thread = std::thread(raw_upload, m, dev, N, de->cm_uF_cm2, de->ri_MOhm, de->area_um2, src);
      raw_started = true;
    }
  }
  try {
    m->options = parsed;
    m->n_cell = de->n_cell;
    m->N = N;
    m->cell_first.assign(de->cell_first, de->cell_first + (de->n_cell ? de->n_cell + 1 : 0));
    if (de->n_cell == 0) m->cell_first.assign(1, 0);
    par_assign(m->parent, de->parent, N);
    // (area, ri, cm and the parameters of distributed tables that are on their way to the device
    // already are copied after the layout is known, and only if the host will need them: below)
    if (!raw_started) {
      par_assign(m->area, de->area_um2, N);
      par_assign(m->ri, de->ri_MOhm, N);
      par_assign(m->cm, de->cm_uF_cm2, N);
    }
    m->thr.assign(de->thr_mV, de->thr_mV + de->n_cell);
    m->v_init = de->v_init_mV;
    m->celsius = de->celsius;
    m->tab.resize(de->n_mech);
    for (int32_t t = 0; t < de->n_mech; ++t) {
      const cn_mech_table &mt = de->mech[t];
      HTable &T = m->tab[t];
      T.type = mt.type;
      type_info(mt.type, T.ti);
      T.n = mt.n;
      par_assign(T.node, mt.node, mt.n);
      const bool deferred = raw_started && !T.ti.point && T.ti.n_param > 0 && mt.n > 0;
      if (!deferred) par_assign(T.param, mt.param, mt.n * T.ti.n_param);
      T.glob.assign(mt.global, mt.global + T.ti.n_global);
    }
    lap("deep copy");
    m->n_netcon = de->n_netcon;
    par_assign(m->nc_src, de->nc_src_gid, de->n_netcon);
    par_assign(m->nc_tgt_mech, de->nc_tgt_mech, de->n_netcon);
    par_assign(m->nc_tgt_inst, de->nc_tgt_inst, de->n_netcon);
    par_assign(m->nc_w, de->nc_weight_uS, de->n_netcon);
    par_assign(m->nc_delay, de->nc_delay_ms, de->n_netcon);
    m->stim_gid.assign(de->stim_gid, de->stim_gid + de->n_stim);
    m->stim_t.assign(de->stim_t_ms, de->stim_t_ms + de->n_stim);
    m->n_src = n_src;
    m->sp_cap = 16 * (int64_t)de->n_cell + 65536;
    int rc = build_layout(m);
    if (rc != CN_OK || m->tgrp.empty()) m->raw.cancel.store(true);
    raw_join();
    if (rc != CN_OK) {
      m->raw.release();
      delete m;
      return rc;
    }
    if (m->tgrp.empty()) m->raw.release();
    // The host keeps the node arrays and the parameters of a distributed table only where
    // finalize() reads them: cells on the warp-cooperative kernel, or a device copy that did not
    // arrive.  Otherwise all it needs is cm and area at the nodes of the point processes.
    if (raw_started) {
      const bool on_device = m->raw.err == cudaSuccess && m->raw.cm && m->raw.ri && m->raw.area;
      if (m->n_cgroup > 0 || !on_device) {
        par_assign(m->area, de->area_um2, N);
        par_assign(m->ri, de->ri_MOhm, N);
        par_assign(m->cm, de->cm_uF_cm2, N);
      } else {
        m->node_arrays_host = false;
        for (int32_t t = 0; t < de->n_mech; ++t) {
          HTable &T = m->tab[t];
          if (!T.ti.point) continue;
          T.pp_cm.resize((size_t)T.n);
          T.pp_area.resize((size_t)T.n);
          par_for(T.n, 1 << 16, [&](int64_t i0, int64_t i1) {
            for (int64_t i = i0; i < i1; ++i) {
              T.pp_cm[i] = de->cm_uF_cm2[T.node[i]];
              T.pp_area[i] = de->area_um2[T.node[i]];
            }
          });
        }
      }
    }
    for (int32_t t = 0; t < de->n_mech; ++t) {
      HTable &T = m->tab[t];
      const cn_mech_table &mt = de->mech[t];
      if (T.ti.point || T.ti.n_param == 0 || mt.n == 0 || !T.param.empty()) continue;
      const bool on_device = m->raw.err == cudaSuccess && (size_t)t < m->raw.param.size() &&
                             m->raw.param[t] != nullptr;
      if (m->n_cgroup > 0 || !on_device) par_assign(T.param, mt.param, mt.n * T.ti.n_param);
    }
    lap("layout, upload of the compact arrays joined");
  } catch (const std::bad_alloc &) {
    m->raw.cancel.store(true);
    raw_join();
    m->raw.release();
    delete m;
    return fail(CN_ERR_NOMEM, "out of host memory");
  }
  *out = m;
  return CN_OK;
}

#include "cn_layout.hpp"
#include "cn_finalize.hpp"

// ---------------------------------------------------------------------------------------------
// run
// ---------------------------------------------------------------------------------------------

template <int WPB>
static cudaError_t launch_step(cn_model *m, int64_t k, cudaStream_t st) {
  const int ng = m->hm.n_group;
  const size_t smem = (size_t)WPB * m->warp_smem_doubles * sizeof(double);
  bool *attr_set = m->step_attr_set;  // (per model: cudaFuncSetAttribute is per device)
  if (!attr_set[WPB]) {
    cudaError_t e = cudaFuncSetAttribute(step_kernel<WPB>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    attr_set[WPB] = true;
  }
  step_kernel<WPB><<<(ng + WPB - 1) / WPB, WPB * 32, smem, st>>>(m->hm, k);
  return cudaGetLastError();
}

static size_t tape_smem_bytes(const cn_model *m, int pbuf) {
  const size_t W = (size_t)m->tape_W;
  return W * m->tape_S * m->tape_CH * 256 + (size_t)m->hm.tape_sys_cap * 512 +
         (size_t)pbuf * m->hm.tape_prog_cap * 16 + (W * m->tape_S + 2 + m->tape_bar_cap) * 8 + 16;
}

// Persistent CTAs: as many as fit the device at once (shared memory decides), each looping over
// the groups blockIdx.x, blockIdx.x + gridDim.x, ...
static cudaError_t launch_tape(cn_model *m, int64_t k, int mode, int nsteps = 1,
                               cudaStream_t st = nullptr) {
  if (!st) st = m->stream;
  auto kern = m->tape_W <= 8 ? tape_step_kernel<256> : tape_step_kernel<512>;
  if (m->tape_ctas == 0) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         227 * 1024);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout,
                             cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0, per_sm = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
      return e;
    // Two CTAs per SM when they fit: 2 x 256 threads x 128 registers fill the register file,
    // each CTA allocates half of the SM's tensor memory, and shared memory decides.  (The
    // occupancy API answers 1 for this kernel whatever the shared-memory size; the hardware
    // does run two CTAs side by side -- measured.)
    int smem_sm = 0;
    e = cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
    if (e != cudaSuccess) return e;
    // the next group's program is prefetched into a second buffer unless that costs the second CTA
    m->hm.tape_pbuf = 2;
    if (m->tape_W <= 8 && 2 * (tape_smem_bytes(m, 2) + 1024) > (size_t)smem_sm &&
        2 * (tape_smem_bytes(m, 1) + 1024) <= (size_t)smem_sm)
      m->hm.tape_pbuf = 1;
    if (tape_smem_bytes(m, 2) > 227 * 1024) m->hm.tape_pbuf = 1;  // (build_layout fitted one buffer)
    if (const char *s = m->opt("tape_pbuf")) m->hm.tape_pbuf = std::atoi(s) == 1 ? 1 : 2;
    const size_t smem = tape_smem_bytes(m, m->hm.tape_pbuf);
    per_sm = (m->tape_W <= 8 && 2 * (smem + 1024) <= (size_t)smem_sm) ? 2 : 1;
    if (const char *s = m->opt("tape_ctas_per_sm")) per_sm = std::max(1, std::min(2, std::atoi(s)));
    if (m->opt("debug") && std::atoi(m->opt("debug")) != 0)
      fprintf(stderr, "[cn] tape kernel: %zu B smem, %d threads, %d CTAs/SM\n", smem,
              32 * m->tape_W, per_sm);
    m->tape_ctas = std::min(m->hm.n_tgroup, sms * per_sm);
  }
  kern<<<m->tape_ctas, 32 * m->tape_W, tape_smem_bytes(m, m->hm.tape_pbuf), st>>>(
      m->hm, k, mode, nsteps);
  return cudaGetLastError();
}

static int run_steps(cn_model *m, int64_t K) {
  const int ng = m->hm.n_group, ntg = m->hm.n_tgroup;
  int deliver_blocks = 8;
  if (m->n_netcon > 1000000) deliver_blocks = 148;
  int64_t pp_tape = 0;
  for (const HTable &T : m->tab)
    if (T.ti.point) pp_tape = std::max(pp_tape, T.n - T.pp_tape_begin);
  const int pp_blocks = (int)std::min<int64_t>((pp_tape + 255) / 256, 148 * 8);
  int64_t pp_coop = 0;
  for (const HTable &T : m->tab)
    if (T.ti.point) pp_coop = std::max(pp_coop, T.pp_tape_begin);
  const int ppc_blocks = (int)std::min<int64_t>((pp_coop + 255) / 256, 148 * 16);
  CU(cudaEventRecord(m->ev0, m->stream));
  if (m->cwindow) {
    // cell-window mode: the events of a window of up to win_steps steps are summed per (step,
    // synapse), then one launch keeps every cell on chip for the whole window (cn_cell.cuh)
    for (int64_t s = 0; s < K;) {
      const int n = (int)std::min<int64_t>(m->win_steps, K - s);
      const int64_t k = m->k + s;
      if (m->n_netcon > 0) {
        deliver_window_kernel<<<deliver_blocks, 128, 0, m->stream>>>(m->hm, k, n, m->win_idx);
        m->launches++;
      }
      const bool timeit = m->ktime_every > 0 && m->ktime_used < m->ktime_ev.size();
      if (timeit) cudaEventRecord(m->ktime_ev[m->ktime_used].first, m->stream);
      switch (m->cwin_threads) {
        case 64: cell_window_kernel<64><<<m->cwin_grid, 64, m->cwin_smem, m->stream>>>(m->hm, k, n, m->probe_rows); break;
        case 128: cell_window_kernel<128><<<m->cwin_grid, 128, m->cwin_smem, m->stream>>>(m->hm, k, n, m->probe_rows); break;
        default: cell_window_kernel<256><<<m->cwin_grid, 256, m->cwin_smem, m->stream>>>(m->hm, k, n, m->probe_rows); break;
      }
      if (timeit) {
        cudaEventRecord(m->ktime_ev[m->ktime_used++].second, m->stream);
        m->ktime_steps.push_back(n);
      }
      if (!m->probe.empty()) m->probe_rows = std::min(m->probe_cap, m->probe_rows + n);
      m->launches++;
      m->win_idx++;
      s += n;
    }
    CU(cudaEventRecord(m->ev1, m->stream));
    CU(cudaGetLastError());
    m->k += K;
    m->timed = true;
    return CN_OK;
  }
  if (m->window) {
    // one launch of the interleaved kernel per window of up to win_steps steps; the events and
    // point processes of the whole window are prepared by two small kernels in front of it
    int64_t pp_all = 0;
    for (const HTable &T : m->tab)
      if (T.ti.point) pp_all = std::max(pp_all, T.n);
    const int ppb = (int)std::max<int64_t>(1, std::min<int64_t>((pp_all + 255) / 256, 148 * 8));
    for (int64_t s = 0; s < K;) {
      const int n = (int)std::min<int64_t>(m->win_steps, K - s);
      const int64_t k = m->k + s;
      // (win_rows needs no clearing: the interleaved kernel zeroes every row it consumes)
      CU(cudaMemsetAsync(m->hm.win_done, 0, (size_t)ntg * sizeof(int32_t), m->stream));
      CU(cudaMemsetAsync(m->hm.win_ticket, 0, sizeof(uint32_t), m->stream));
      if (m->n_netcon > 0) {
        deliver_window_kernel<<<deliver_blocks, 128, 0, m->stream>>>(m->hm, k, n, m->win_idx);
        m->launches++;
      }
      if (pp_all > 0) {
        pp_window_kernel<<<ppb, 256, 0, m->stream>>>(m->hm, k, n);
        m->launches++;
      }
      const bool timeit = m->ktime_every > 0 && m->ktime_used < m->ktime_ev.size();
      if (timeit) cudaEventRecord(m->ktime_ev[m->ktime_used].first, m->stream);
      m->hm.trace_row0 = m->probe_rows;
      if (!m->probe.empty()) m->probe_rows = std::min(m->probe_cap, m->probe_rows + n);
      cudaError_t e = launch_tape(m, k, (m->state_pending ? TM_ADVANCE : 0) | TM_WINDOW, n);
      if (e != cudaSuccess) return fail(CN_ERR_CUDA, "tape launch failed: %s", cudaGetErrorString(e));
      if (timeit) {
        cudaEventRecord(m->ktime_ev[m->ktime_used++].second, m->stream);
        m->ktime_steps.push_back(n);
      }
      m->state_pending = true;
      m->launches++;
      m->win_idx++;
      s += n;
    }
    CU(cudaEventRecord(m->ev1, m->stream));
    CU(cudaGetLastError());
    m->k += K;
    m->timed = true;
    return CN_OK;
  }
  // ---- one launch sequence per dt: deliver -> point processes -> step kernels (-> probes) --------
  // k_arg >= 0: the step itself; k_arg = -(1 + s): step = device counter + s (replayed CUDA graph).
  auto issue_step = [&](int64_t k_arg, int64_t row_arg, cudaStream_t st, bool timeit) -> int {
    // event pair around the kernel class selected by cn_select_timed_kernel
    auto t0 = [&](int which) {
      if (timeit && m->ktime_which == which) cudaEventRecord(m->ktime_ev[m->ktime_used].first, st);
    };
    auto t1 = [&](int which) {
      if (timeit && m->ktime_which == which) {
        cudaEventRecord(m->ktime_ev[m->ktime_used++].second, st);
        m->ktime_steps.push_back(1);
      }
    };
    const bool pp_any = (ntg > 0 && pp_tape > 0) || (ng > 0 && pp_coop > 0);
    if (m->n_netcon > 0) {
      t0(2);
      deliver_kernel<<<deliver_blocks, 128, 0, st>>>(m->hm, k_arg);
      t1(2);
      m->launches++;
    }
    if (pp_any) t0(1);
    if (ntg > 0 && pp_tape > 0) {
      pp_step_kernel<false><<<pp_blocks, 256, 0, st>>>(m->hm, k_arg);
      m->launches++;
    }
    if (ng > 0 && pp_coop > 0) {
      pp_step_kernel<true><<<ppc_blocks, 256, 0, st>>>(m->hm, k_arg);
      m->launches++;
    }
    if (pp_any) t1(1);
    const bool time_tape = ntg > 0;  // the dominant step kernel is the tape kernel when it runs
    if (ng > 0) {
      cudaError_t e;
      if (!time_tape) t0(0);
      switch (m->wpb) {
        case 8: e = launch_step<8>(m, k_arg, st); break;
        case 4: e = launch_step<4>(m, k_arg, st); break;
        case 2: e = launch_step<2>(m, k_arg, st); break;
        default: e = launch_step<1>(m, k_arg, st); break;
      }
      if (e != cudaSuccess) return fail(CN_ERR_CUDA, "step launch failed: %s", cudaGetErrorString(e));
      if (!time_tape) t1(0);
      m->launches++;
    }
    if (ntg > 0) {
      t0(0);
      cudaError_t e = launch_tape(m, k_arg, m->state_pending ? TM_ADVANCE : 0, 1, st);
      if (e != cudaSuccess) return fail(CN_ERR_CUDA, "tape launch failed: %s", cudaGetErrorString(e));
      m->state_pending = true;
      t1(0);
      m->launches++;
    }
    if (!m->probe.empty() && (row_arg < 0 || row_arg < m->probe_cap)) {
      const int np = (int)m->probe.size();
      probe_kernel<<<(np + 127) / 128, 128, 0, st>>>(m->d_v, m->d_probe_pos, np, m->d_trace, row_arg,
                                                      m->hm.step_ctr, m->probe_cap);
      m->launches++;
    }
    return CN_OK;
  };
  // The sequence of CN_GRAPH_STEPS consecutive steps is captured once into a CUDA graph (on a
  // stream of the model's own: the caller's may be the legacy default stream, which cannot
  // capture) and replayed; the kernels of the graph take their step from a device counter that a
  // one-thread kernel sets in front of every replay.  The first step of a model, runs shorter
  // than a graph, the remainder of a run and runs with per-launch event timing are issued directly.
  const bool use_graph = m->graph_on && m->ktime_every == 0;
  int64_t s = 0;
  while (s < K) {
    const int64_t k = m->k + s;
    const bool warm = m->direct_steps > 0 && (ntg == 0 || m->state_pending);
    if (use_graph && warm && K - s >= CN_GRAPH_STEPS) {
      if (!m->graph_exec) {
        const int64_t l0 = m->launches;
        if (!m->cap_stream) CU(cudaStreamCreateWithFlags(&m->cap_stream, cudaStreamNonBlocking));
        CU(cudaStreamBeginCapture(m->cap_stream, cudaStreamCaptureModeThreadLocal));
        int rc = CN_OK;
        for (int j = 0; j < CN_GRAPH_STEPS && rc == CN_OK; ++j)
          rc = issue_step(-(1 + (int64_t)j), -(1 + (int64_t)j), m->cap_stream, false);
        cudaGraph_t g = nullptr;
        cudaError_t e = cudaStreamEndCapture(m->cap_stream, &g);
        m->graph_kernels = m->launches - l0;
        m->launches = l0;
        if (rc != CN_OK) { if (g) cudaGraphDestroy(g); return rc; }
        if (e != cudaSuccess) return fail(CN_ERR_CUDA, "graph capture failed: %s", cudaGetErrorString(e));
        e = cudaGraphInstantiate(&m->graph_exec, g, 0);
        cudaGraphDestroy(g);
        if (e != cudaSuccess) return fail(CN_ERR_CUDA, "graph instantiation failed: %s", cudaGetErrorString(e));
      }
      set_ctr_kernel<<<1, 1, 0, m->stream>>>(m->hm.step_ctr, k, m->probe_rows);
      CU(cudaGraphLaunch(m->graph_exec, m->stream));
      m->launches += 1 + m->graph_kernels;
      m->graph_replays++;
      if (!m->probe.empty()) m->probe_rows = std::min(m->probe_cap, m->probe_rows + CN_GRAPH_STEPS);
      s += CN_GRAPH_STEPS;
      continue;
    }
    const bool timeit = m->ktime_every > 0 && (k % m->ktime_every) == 0 &&
                        m->ktime_used < m->ktime_ev.size();
    int rc = issue_step(k, m->probe_rows, m->stream, timeit);
    if (rc != CN_OK) return rc;
    if (!m->probe.empty() && m->probe_rows < m->probe_cap) m->probe_rows++;
    m->direct_steps++;
    ++s;
  }
  CU(cudaEventRecord(m->ev1, m->stream));
  CU(cudaGetLastError());
  m->k += K;
  m->timed = true;
  return CN_OK;
}

extern "C" int cn_run_async(cn_model *m, double tstop, double dt) {
  if (!m) return fail(CN_ERR_ARG, "NULL model");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(CN_ERR_DT, "dt must be > 0");
  if (!std::isfinite(tstop)) return fail(CN_ERR_ARG, "tstop must be finite");
  if (!m->uploaded) {
    int rc = finalize(m, dt);
    if (rc != CN_OK) return rc;
  } else if (dt != m->dt) {
    return fail(CN_ERR_DT, "dt = %.17g differs from the first run's dt = %.17g", dt, m->dt);
  }
  const int64_t target = llround(tstop / dt);
  if (target <= m->k) return CN_OK;
  return run_steps(m, target - m->k);
}

extern "C" int cn_sync(cn_model *m) {
  if (!m) return fail(CN_ERR_ARG, "NULL model");
  if (!m->uploaded) return CN_OK;
  CU(cudaStreamSynchronize(m->stream));
  int32_t ov = 0;
  CU(cudaMemcpy(&ov, m->d_overflow, sizeof(ov), cudaMemcpyDeviceToHost));
  if (ov == 2)
    return fail(CN_ERR_OVERFLOW, "a point-process conductance / current or event weight left the "
                                 "range of the fixed-point sums (2^18 row-normalised units)");
  if (ov) return fail(CN_ERR_OVERFLOW, "spike buffer overflow (capacity %lld)", (long long)m->sp_cap);
  return CN_OK;
}

extern "C" int cn_run(cn_model *m, double tstop, double dt) {
  int rc = cn_run_async(m, tstop, dt);
  if (rc != CN_OK) return rc;
  return cn_sync(m);
}

extern "C" int cn_set_stream(cn_model *m, void *s) {
  if (!m) return fail(CN_ERR_ARG, "NULL model");
  m->stream = (cudaStream_t)s;
  return CN_OK;
}

extern "C" int cn_get_v(const cn_model *cm, double *out, int64_t n) {
  cn_model *m = const_cast<cn_model *>(cm);
  if (!m || (!out && n > 0)) return fail(CN_ERR_ARG, "NULL argument");
  if (n != m->N) return fail(CN_ERR_ARG, "n = %lld but the model has %lld nodes", (long long)n,
                             (long long)m->N);
  if (!m->uploaded) {  // before the first run: initial condition
    for (int64_t i = 0; i < n; ++i) out[i] = m->v_init;
    return CN_OK;
  }
  if (n == 0) return CN_OK;
  gather_kernel<<<(unsigned)((n + 255) / 256), 256, 0, m->stream>>>(m->d_v, m->d_node_pos, n,
                                                                     m->d_gather);
  m->launches++;
  CU(cudaGetLastError());
  CU(cudaMemcpyAsync(out, m->d_gather, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost,
                     m->stream));
  CU(cudaStreamSynchronize(m->stream));
  return CN_OK;
}

extern "C" int cn_get_spikes(const cn_model *cm, int32_t *gid, int64_t *step, int64_t cap,
                             int64_t *n_out) {
  cn_model *m = const_cast<cn_model *>(cm);
  if (!m || !n_out) return fail(CN_ERR_ARG, "NULL argument");
  *n_out = 0;
  if (!m->uploaded) return CN_OK;
  CU(cudaStreamSynchronize(m->stream));
  unsigned long long ns = 0;
  CU(cudaMemcpy(&ns, m->d_nsp, sizeof(ns), cudaMemcpyDeviceToHost));
  int64_t n = std::min<int64_t>((int64_t)ns, m->sp_cap);
  *n_out = n;
  if (cap == 0 || n == 0) return CN_OK;
  if (!gid || !step) return fail(CN_ERR_ARG, "NULL output array");
  std::vector<int32_t> g((size_t)n);
  std::vector<int64_t> s((size_t)n);
  CU(cudaMemcpy(g.data(), m->d_sp_gid, (size_t)n * sizeof(int32_t), cudaMemcpyDeviceToHost));
  CU(cudaMemcpy(s.data(), m->d_sp_step, (size_t)n * sizeof(int64_t), cudaMemcpyDeviceToHost));
  std::vector<int64_t> ord((size_t)n);
  std::iota(ord.begin(), ord.end(), 0);
  std::sort(ord.begin(), ord.end(), [&](int64_t x, int64_t y) {
    if (s[x] != s[y]) return s[x] < s[y];
    return g[x] < g[y];
  });
  const int64_t w = std::min(n, cap);
  for (int64_t i = 0; i < w; ++i) { gid[i] = g[ord[i]]; step[i] = s[ord[i]]; }
  return CN_OK;
}

extern "C" int cn_set_probes(cn_model *m, const int32_t *node, int64_t n, int64_t max_steps) {
  if (!m || (n > 0 && !node)) return fail(CN_ERR_ARG, "NULL argument");
  if (m->uploaded) return fail(CN_ERR_ARG, "probes must be set before the first cn_run");
  if (n < 0 || max_steps < 0) return fail(CN_ERR_ARG, "negative count");
  for (int64_t i = 0; i < n; ++i)
    if (node[i] < 0 || node[i] >= m->N) return fail(CN_ERR_ARG, "probe node out of range");
  m->probe.assign(node, node + n);
  m->probe_cap = max_steps;
  return CN_OK;
}

extern "C" int cn_get_trace(const cn_model *cm, double *out, int64_t cap_steps, int64_t *n_steps) {
  cn_model *m = const_cast<cn_model *>(cm);
  if (!m || !n_steps) return fail(CN_ERR_ARG, "NULL argument");
  *n_steps = m->probe_rows;
  const int64_t rows = std::min(m->probe_rows, cap_steps);
  if (rows <= 0 || m->probe.empty()) return CN_OK;
  if (!out) return fail(CN_ERR_ARG, "NULL output");
  CU(cudaStreamSynchronize(m->stream));
  CU(cudaMemcpy(out, m->d_trace, (size_t)rows * m->probe.size() * sizeof(double),
                cudaMemcpyDeviceToHost));
  return CN_OK;
}

extern "C" int64_t cn_steps_done(const cn_model *m) { return m ? m->k : 0; }
extern "C" int64_t cn_launch_count(const cn_model *m) { return m ? m->launches : 0; }

extern "C" int cn_last_run_ms(const cn_model *m, double *ms) {
  if (!m || !ms) return fail(CN_ERR_ARG, "NULL argument");
  if (!m->timed) return fail(CN_ERR_ARG, "no run yet");
  float f = 0.f;
  CU(cudaEventSynchronize(m->ev1));
  CU(cudaEventElapsedTime(&f, m->ev0, m->ev1));
  *ms = f;
  return CN_OK;
}

extern "C" int cn_get_run_info(const cn_model *m, int64_t *info) {
  if (!m || !info) return fail(CN_ERR_ARG, "NULL argument");
  info[0] = !m->uploaded ? -1 : m->cwindow ? 2 : m->window ? 1 : 0;
  info[1] = m->graph_replays;
  info[2] = (m->window || m->cwindow) ? m->win_steps : 1;
  info[3] = m->cwindow ? m->cwin_grid : m->tape_ctas;
  return CN_OK;
}

extern "C" int cn_get_layout_info(const cn_model *m, int64_t *info) {
  if (!m || !info) return fail(CN_ERR_ARG, "NULL argument");
  info[0] = (int64_t)m->cls.size();
  info[1] = (int64_t)m->grp.size() + (int64_t)m->tgrp.size();
  info[2] = (int64_t)m->warp_smem_doubles * 8;
  int r = 0;
  for (const HClass &K : m->cls) r = std::max(r, K.rounds);
  info[3] = r;
  info[4] = (int64_t)m->tgrp.size();
  info[5] = m->n_tape * 8;
  info[6] = m->hm.n_tgroup > 0 ? (int64_t)tape_smem_bytes(m, m->hm.tape_pbuf ? m->hm.tape_pbuf : 2) : 0;  // valid after the first cn_run
  info[7] = (int64_t)m->tape_W | (int64_t)m->tape_ctas << 8 | (int64_t)m->tape_sys_cap << 24;
  return CN_OK;
}

#include "cn_checkpoint.hpp"

// ---------------------------------------------------------------------------------------------
// cn_get_state_noalloc: cn_get_state for callers that must not allocate device memory
// ---------------------------------------------------------------------------------------------
// cn_get_state gathers through a scratch buffer that it grows with cudaMalloc on first use
// (ensure_scratch).  This variant keeps its scratch -- the location list and the gathered
// values, 16 B per instance -- in a file-scope device array of fixed size, so the call allocates
// nothing on the device or on the host heap: CN_NOALLOC_MAX_INSTANCES instances, 1 MiB, held by
// every GPU that loads the library until the process exits.  The array is shared by every call
// and keeps the last call's contents; nothing in it has to start at zero (the n locations and the
// n values are written before they are read).  Calls that overlap on the GPU would race on it:
// the entry point holds a process-wide lock and returns after its work has completed on the
// model's stream, so two calls of one process never overlap.
static __device__ __align__(256) unsigned char cn_noalloc_scratch[CN_NOALLOC_MAX_INSTANCES * 16];
static int64_t g_noalloc_loc[CN_NOALLOC_MAX_INSTANCES];  // host staging of the location list
static std::mutex g_noalloc_mu;
static void *g_noalloc_ptr[64] = {};  // device address of the array, per device ordinal

// variant of gather_state_kernel (cn_tape.cuh) on the static scratch: locations in the first
// half, values in the second
__global__ void gather_state_noalloc_kernel(const double *__restrict__ tape,
                                            const double *__restrict__ st,
                                            unsigned char *__restrict__ scratch, int64_t n) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int64_t *loc = reinterpret_cast<const int64_t *>(scratch);
  double *val = reinterpret_cast<double *>(scratch + (size_t)CN_NOALLOC_MAX_INSTANCES * 8);
  const int64_t l = loc[i];
  val[i] = l >= 0 ? st[l] : tape[-(l + 1)];
}

// In host code the array's name is a host-side stand-in, not a device address: the address a
// kernel can use comes from cudaGetSymbolAddress, once per device, with that device current.
static int noalloc_scratch_ptr(unsigned char **out) {
  int dev = 0;
  CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(CN_ERR_UNSUPPORTED, "device ordinal %d not supported", dev);
  if (!g_noalloc_ptr[dev]) {
    void *p = nullptr;
    CU(cudaGetSymbolAddress(&p, cn_noalloc_scratch));
    g_noalloc_ptr[dev] = p;
  }
  *out = static_cast<unsigned char *>(g_noalloc_ptr[dev]);
  return CN_OK;
}

extern "C" int cn_get_state_noalloc(const cn_model *cm, int32_t t, int32_t s, double *out, int64_t n) {
  cn_model *m = const_cast<cn_model *>(cm);
  if (!m || !out) return fail(CN_ERR_ARG, "NULL argument");
  if (t < 0 || t >= (int)m->tab.size()) return fail(CN_ERR_MECH, "table out of range");
  HTable &T = m->tab[t];
  if (s < 0 || s >= T.ti.n_state || n != T.n) return fail(CN_ERR_MECH, "state / size mismatch");
  if (n > CN_NOALLOC_MAX_INSTANCES)
    return fail(CN_ERR_UNSUPPORTED,
                "cn_get_state_noalloc: table %d has %lld instances, the static scratch holds %d "
                "(use cn_get_state)", t, (long long)n, CN_NOALLOC_MAX_INSTANCES);
  if (!m->uploaded) return fail(CN_ERR_ARG, "states exist after the first cn_run");
  if (n == 0) return CN_OK;
  std::lock_guard<std::mutex> lk(g_noalloc_mu);
  unsigned char *scratch = nullptr;
  int rc = noalloc_scratch_ptr(&scratch);
  if (rc != CN_OK) return rc;
  if (!T.ti.point) {  // (see cn_get_state)
    rc = flush_pending_state(m);
    if (rc != CN_OK) return rc;
  }
  for (int64_t i = 0; i < n; ++i) g_noalloc_loc[i] = state_loc(T, i, s);
  CU(cudaMemcpyAsync(scratch, g_noalloc_loc, (size_t)n * 8, cudaMemcpyHostToDevice, m->stream));
  gather_state_noalloc_kernel<<<(unsigned)((n + 255) / 256), 256, 0, m->stream>>>(
      m->hm.tape, T.d_state[s], scratch, n);
  CU(cudaGetLastError());
  m->launches++;
  CU(cudaMemcpyAsync(out, scratch + (size_t)CN_NOALLOC_MAX_INSTANCES * 8, (size_t)n * 8,
                     cudaMemcpyDeviceToHost, m->stream));
  CU(cudaStreamSynchronize(m->stream));
  return CN_OK;
}

extern "C" int cn_set_spike_capacity(cn_model *m, int64_t cap) {
  if (!m || cap < 1) return fail(CN_ERR_ARG, "bad capacity");
  if (m->uploaded) return fail(CN_ERR_ARG, "capacity must be set before the first cn_run");
  m->sp_cap = cap;
  return CN_OK;
}

extern "C" int cn_set_kernel_timing(cn_model *m, int32_t every, int32_t max_samples) {
  if (!m || every < 0 || max_samples < 0) return fail(CN_ERR_ARG, "bad argument");
  for (auto &pr : m->ktime_ev) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
  m->ktime_ev.clear();
  m->ktime_used = 0;
  m->ktime_steps.clear();
  m->ktime_every = every;
  if (every > 0)
    for (int i = 0; i < max_samples; ++i) {
      cudaEvent_t a, b;
      CU(cudaEventCreate(&a));
      CU(cudaEventCreate(&b));
      m->ktime_ev.emplace_back(a, b);
    }
  return CN_OK;
}

extern "C" int cn_select_timed_kernel(cn_model *m, int32_t which) {
  if (!m || which < 0 || which > 2) return fail(CN_ERR_ARG, "bad argument");
  m->ktime_which = which;
  return CN_OK;
}

extern "C" int cn_get_kernel_timing(cn_model *m, double *sum_ms, int64_t *count) {
  if (!m || !sum_ms || !count) return fail(CN_ERR_ARG, "NULL argument");
  double tot = 0.0;
  for (size_t i = 0; i < m->ktime_used; ++i) {
    float f = 0.f;
    CU(cudaEventSynchronize(m->ktime_ev[i].second));
    CU(cudaEventElapsedTime(&f, m->ktime_ev[i].first, m->ktime_ev[i].second));
    tot += f;
  }
  *sum_ms = tot;
  int64_t steps = 0;  // a sample of the window mode covers several dt
  for (size_t i = 0; i < m->ktime_used && i < m->ktime_steps.size(); ++i) steps += m->ktime_steps[i];
  *count = steps;
  m->ktime_used = 0;
  m->ktime_steps.clear();
  return CN_OK;
}

extern "C" void cn_model_destroy(cn_model *m) {
  if (!m) return;
  if (m->uploaded) cudaStreamSynchronize(m->stream);
  for (auto &pr : m->ktime_ev) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
  for (void *p : m->dev_allocs) cudaFree(p);
  m->raw.release();
  if (m->d_scratch) cudaFree(m->d_scratch);
  if (m->ev0) cudaEventDestroy(m->ev0);
  if (m->ev1) cudaEventDestroy(m->ev1);
  if (m->graph_exec) cudaGraphExecDestroy(m->graph_exec);
  if (m->cap_stream) cudaStreamDestroy(m->cap_stream);
  delete m;
}

#ifdef CN_TRACE
// development builds only (CN_TRACE=1): positions per task of the first tape class, phase clocks
extern "C" int cn_debug_tasks(const cn_model *m, int32_t *out, int32_t cap) {
  for (const HClass &K : m->cls) {
    if (K.tp.n_groups == 0) continue;
    int n = 0;
    for (const HTask &t : K.tp.task) {
      if (n + 2 <= cap) { out[n++] = t.p1 - t.p0; out[n++] = (int32_t)t.nrows; }
    }
    if (n + 2 <= cap) {  // simulated makespan and total work of the schedule, x100
      out[n++] = (int32_t)(K.tp.sim_makespan * 100.0);
      out[n++] = (int32_t)(K.tp.sim_work * 100.0);
    }
    return n;
  }
  return 0;
}

extern "C" int cn_debug_cell_trace(long long *out, int reset) {
  int rc = (int)cudaMemcpyFromSymbol(out, cn::g_cell_trace, sizeof(long long) * 16);
  if (reset) {
    long long z[16] = {};
    cudaMemcpyToSymbol(cn::g_cell_trace, z, sizeof(z));
  }
  return rc;
}

extern "C" int cn_debug_trace2(long long *out) {
  return (int)cudaMemcpyFromSymbol(out, cn::g_trace2, sizeof(long long) * 2 * 8 * 16 * 128 * 2);
}

extern "C" int cn_debug_trace(long long *out) {
  return (int)cudaMemcpyFromSymbol(out, cn::g_trace, sizeof(long long) * 148 * 16 * 8 * 8);
}
#endif
