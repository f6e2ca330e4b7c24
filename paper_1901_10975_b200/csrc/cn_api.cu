// cn_api.cu -- the C ABI of libcn (include/cn.h): validation and deep copy of the description, the
// step loop, read-back, checkpoints.  The set-up lives in cn_host.hpp (model structure, helpers),
// cn_layout.hpp (shape classes, programs, permutations) and cn_finalize.hpp (dt-dependent tables).
// C ABI declared in include/cn.h.  No CPU compute path exists: every step runs in cn_device.cuh.
#include "../../include/cn.h"
#include "cn_device.cuh"
#include "cn_tape.cuh"

#include <algorithm>
#include <chrono>
#include <cmath>
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

extern "C" int cn_model_create(const cn_model_desc *de, cn_model **out) {
  if (out) *out = nullptr;
  if (!de || !out) return fail(CN_ERR_ARG, "cn_model_create: NULL argument");
  if (de->n_cell < 0 || de->n_node < 0) return fail(CN_ERR_ARG, "negative sizes");
  if (de->n_node >= (int64_t)1 << 31) return fail(CN_ERR_ARG, "n_node must be < 2^31");
  if (de->n_mech < 0 || de->n_mech > CN_MAX_TABLES)
    return fail(CN_ERR_MECH, "n_mech must be in [0, %d]", CN_MAX_TABLES);
  const int64_t N = de->n_node;
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

  cn_model *m = new (std::nothrow) cn_model();
  if (!m) return fail(CN_ERR_NOMEM, "out of host memory");
  try {
    m->n_cell = de->n_cell;
    m->N = N;
    m->cell_first.assign(de->cell_first, de->cell_first + (de->n_cell ? de->n_cell + 1 : 0));
    if (de->n_cell == 0) m->cell_first.assign(1, 0);
    par_assign(m->parent, de->parent, N);
    par_assign(m->area, de->area_um2, N);
    par_assign(m->ri, de->ri_MOhm, N);
    par_assign(m->cm, de->cm_uF_cm2, N);
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
      par_assign(T.param, mt.param, mt.n * T.ti.n_param);
      T.glob.assign(mt.global, mt.global + T.ti.n_global);
    }
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
    if (rc != CN_OK) {
      delete m;
      return rc;
    }
  } catch (const std::bad_alloc &) {
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
static cudaError_t launch_step(cn_model *m, int64_t k) {
  const int ng = m->hm.n_group;
  const size_t smem = (size_t)WPB * m->warp_smem_doubles * sizeof(double);
  static bool attr_set[16] = {};
  if (!attr_set[WPB]) {
    cudaError_t e = cudaFuncSetAttribute(step_kernel<WPB>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    attr_set[WPB] = true;
  }
  step_kernel<WPB><<<(ng + WPB - 1) / WPB, WPB * 32, smem, m->stream>>>(m->hm, k);
  return cudaGetLastError();
}

static size_t tape_smem_bytes(const cn_model *m, int pbuf) {
  const size_t W = (size_t)m->tape_W;
  return W * m->tape_S * m->tape_CH * 256 + (size_t)m->hm.tape_sys_cap * 512 +
         (size_t)pbuf * m->hm.tape_prog_cap * 16 + (W * m->tape_S + 2 + m->tape_bar_cap) * 8 + 16;
}

// Persistent CTAs: as many as fit the device at once (shared memory decides), each looping over
// the groups blockIdx.x, blockIdx.x + gridDim.x, ...
static cudaError_t launch_tape(cn_model *m, int64_t k, int mode, int nsteps = 1) {
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
    if (const char *s = std::getenv("CN_TAPE_PBUF")) m->hm.tape_pbuf = std::atoi(s) == 1 ? 1 : 2;
    const size_t smem = tape_smem_bytes(m, m->hm.tape_pbuf);
    per_sm = (m->tape_W <= 8 && 2 * (smem + 1024) <= (size_t)smem_sm) ? 2 : 1;
    if (const char *s = std::getenv("CN_TAPE_CTAS_PER_SM")) per_sm = std::max(1, std::min(2, std::atoi(s)));
    if (std::getenv("CN_DEBUG"))
      fprintf(stderr, "[cn] tape kernel: %zu B smem, %d threads, %d CTAs/SM\n", smem,
              32 * m->tape_W, per_sm);
    m->tape_ctas = std::min(m->hm.n_tgroup, sms * per_sm);
  }
  kern<<<m->tape_ctas, 32 * m->tape_W, tape_smem_bytes(m, m->hm.tape_pbuf), m->stream>>>(
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
      if (m->win_stride > 0)
        CU(cudaMemsetAsync(m->hm.win_rows, 0, (size_t)m->win_stride * n * sizeof(double), m->stream));
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
  for (int64_t s = 0; s < K; ++s) {
    const int64_t k = m->k + s;
    if (m->n_netcon > 0) {
      deliver_kernel<<<deliver_blocks, 128, 0, m->stream>>>(m->hm, k);
      m->launches++;
    }
    if (ntg > 0 && pp_tape > 0) {
      pp_step_kernel<false><<<pp_blocks, 256, 0, m->stream>>>(m->hm, k);
      m->launches++;
    }
    if (ng > 0 && pp_coop > 0) {
      pp_step_kernel<true><<<ppc_blocks, 256, 0, m->stream>>>(m->hm, k);
      m->launches++;
    }
    const bool timeit = m->ktime_every > 0 && (k % m->ktime_every) == 0 &&
                        m->ktime_used < m->ktime_ev.size();
    const bool time_tape = ntg > 0;  // the dominant kernel is the tape kernel when it runs
    if (ng > 0) {
      cudaError_t e;
      if (timeit && !time_tape) cudaEventRecord(m->ktime_ev[m->ktime_used].first, m->stream);
      switch (m->wpb) {
        case 8: e = launch_step<8>(m, k); break;
        case 4: e = launch_step<4>(m, k); break;
        case 2: e = launch_step<2>(m, k); break;
        default: e = launch_step<1>(m, k); break;
      }
      if (e != cudaSuccess) return fail(CN_ERR_CUDA, "step launch failed: %s", cudaGetErrorString(e));
      if (timeit && !time_tape) {
        cudaEventRecord(m->ktime_ev[m->ktime_used++].second, m->stream);
        m->ktime_steps.push_back(1);
      }
      m->launches++;
    }
    if (ntg > 0) {
      if (timeit) cudaEventRecord(m->ktime_ev[m->ktime_used].first, m->stream);
      cudaError_t e = launch_tape(m, k, m->state_pending ? TM_ADVANCE : 0);
      if (e != cudaSuccess) return fail(CN_ERR_CUDA, "tape launch failed: %s", cudaGetErrorString(e));
      m->state_pending = true;
      if (timeit) {
        cudaEventRecord(m->ktime_ev[m->ktime_used++].second, m->stream);
        m->ktime_steps.push_back(1);
      }
      m->launches++;
    }
    if (!m->probe.empty() && m->probe_rows < m->probe_cap) {
      const int np = (int)m->probe.size();
      probe_kernel<<<(np + 127) / 128, 128, 0, m->stream>>>(m->d_v, m->d_probe_pos, np,
                                                              m->d_trace, m->probe_rows);
      m->probe_rows++;
      m->launches++;
    }
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

extern "C" int cn_get_state(const cn_model *cm, int32_t t, int32_t s, double *out, int64_t n) {
  cn_model *m = const_cast<cn_model *>(cm);
  if (!m || !out) return fail(CN_ERR_ARG, "NULL argument");
  if (t < 0 || t >= (int)m->tab.size()) return fail(CN_ERR_MECH, "table out of range");
  HTable &T = m->tab[t];
  if (s < 0 || s >= T.ti.n_state || n != T.n) return fail(CN_ERR_MECH, "state / size mismatch");
  if (!m->uploaded) return fail(CN_ERR_ARG, "states exist after the first cn_run");
  if (n == 0) return CN_OK;
  if (m->state_pending && !T.ti.point && m->hm.n_tgroup > 0) {
    // the interleaved kernel applies nrn_state of a step at the start of the next one: do it now
    cudaError_t e = launch_tape(m, m->k, TM_ADVANCE | TM_FLUSH);
    if (e != cudaSuccess) return fail(CN_ERR_CUDA, "state flush failed: %s", cudaGetErrorString(e));
    m->launches++;
    m->state_pending = false;
  }
  // instances live in the table arrays (cooperative groups) or on a tape (interleaved groups)
  std::vector<int64_t> loc((size_t)n);
  for (int64_t i = 0; i < n; ++i) {
    const bool on_tape = !T.ti.point && T.tape_loc[i] >= 0;
    loc[i] = on_tape ? -(T.tape_loc[i] + (int64_t)T.ti.n_dev_param * 32 + 1) : T.inst_pos[i];
  }
  int64_t *d_loc = nullptr;
  double *d_out = nullptr;
  CU(cudaMalloc(&d_loc, (size_t)n * sizeof(int64_t)));
  if (cudaMalloc(&d_out, (size_t)n * sizeof(double)) != cudaSuccess) {
    cudaFree(d_loc);
    return fail(CN_ERR_NOMEM, "out of device memory");
  }
  cudaMemcpyAsync(d_loc, loc.data(), (size_t)n * sizeof(int64_t), cudaMemcpyHostToDevice, m->stream);
  gather_state_kernel<<<(unsigned)((n + 255) / 256), 256, 0, m->stream>>>(
      m->hm.tape, T.d_state[s], d_loc, n, s, d_out);
  m->launches++;
  cudaMemcpyAsync(out, d_out, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, m->stream);
  cudaError_t e = cudaStreamSynchronize(m->stream);
  cudaFree(d_loc);
  cudaFree(d_out);
  if (e != cudaSuccess) return fail(CN_ERR_CUDA, "cn_get_state: %s", cudaGetErrorString(e));
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

// ---------------------------------------------------------------------------------------------
// checkpoint / restore (L134-156)
// ---------------------------------------------------------------------------------------------

struct CkHeader {
  uint64_t magic;
  int64_t k, n_sp, win_idx, n_blob;
  double dt;
  int32_t state_pending, window;
  uint64_t layout;  // hash of everything the raw dump depends on
};

static uint64_t ck_layout_hash(const cn_model *m) {
  uint64_t h = mix64(0xC0FFEEull, (uint64_t)m->N);
  h = mix64(h, (uint64_t)m->n_cell);
  h = mix64(h, (uint64_t)m->n_ab);
  h = mix64(h, (uint64_t)m->n_tape);
  h = mix64(h, (uint64_t)m->n_pcell);
  h = mix64(h, (uint64_t)m->tape_W * 1000003u + (uint64_t)m->tape_CH * 1009u + (uint64_t)m->tape_S);
  h = mix64(h, (uint64_t)m->cls.size());
  for (const HTable &T : m->tab) h = mix64(h, (uint64_t)T.n_dev * 31u + (uint64_t)T.type);
  for (const TapeGroup &tg : m->tgrp) h = mix64(h, (uint64_t)tg.tape_base + (uint64_t)tg.cls);
  return h;
}

// every device array that changes during cn_run and is live at a step boundary
static std::vector<std::pair<void *, size_t>> ck_blobs(const cn_model *m, int64_t n_sp) {
  std::vector<std::pair<void *, size_t>> b;
  const DModel &H = m->hm;
  b.emplace_back(m->d_v, (size_t)(m->n_ab + m->n_tape) * sizeof(double));
  for (const HTable &T : m->tab)
    for (int j = 0; j < T.ti.n_state; ++j)
      if (T.d_state[j]) b.emplace_back(T.d_state[j], (size_t)std::max<int64_t>(T.n_dev, 1) * sizeof(double));
  if (m->d_cai) b.emplace_back(m->d_cai, (size_t)m->n_pnode * sizeof(double));
  b.emplace_back(H.flag, (size_t)m->n_pcell);
  b.emplace_back(m->d_sp_gid, (size_t)n_sp * sizeof(int32_t));
  b.emplace_back(m->d_sp_step, (size_t)n_sp * sizeof(int64_t));
  b.emplace_back(m->d_nsp, sizeof(unsigned long long));
  b.emplace_back(H.sp_end, (size_t)H.wr * sizeof(int64_t));
  if (m->window) {
    b.emplace_back(H.win_mark_step, (size_t)H.win_mark_cap * sizeof(int64_t));
    b.emplace_back(H.win_mark_nsp, (size_t)H.win_mark_cap * sizeof(int64_t));
  }
  return b;
}

static int ck_spike_count(const cn_model *m, int64_t *n_sp) {
  unsigned long long ns = 0;
  CU(cudaStreamSynchronize(m->stream));
  CU(cudaMemcpy(&ns, m->d_nsp, sizeof(ns), cudaMemcpyDeviceToHost));
  *n_sp = (int64_t)std::min<unsigned long long>(ns, (unsigned long long)m->sp_cap);
  return CN_OK;
}

extern "C" int cn_checkpoint_size(const cn_model *m, int64_t *bytes_out) {
  if (!m || !bytes_out) return fail(CN_ERR_ARG, "NULL argument");
  if (!m->uploaded) return fail(CN_ERR_ARG, "nothing to checkpoint before the first cn_run");
  int64_t n_sp = 0;
  int rc = ck_spike_count(m, &n_sp);
  if (rc != CN_OK) return rc;
  size_t tot = sizeof(CkHeader);
  for (auto &b : ck_blobs(m, n_sp)) tot += sizeof(uint64_t) + ((b.second + 7) & ~(size_t)7);
  *bytes_out = (int64_t)tot;
  return CN_OK;
}

extern "C" int cn_checkpoint_save(const cn_model *m, void *buf, int64_t bytes) {
  if (!m || !buf) return fail(CN_ERR_ARG, "NULL argument");
  if (!m->uploaded) return fail(CN_ERR_ARG, "nothing to checkpoint before the first cn_run");
  int64_t n_sp = 0;
  int rc = ck_spike_count(m, &n_sp);
  if (rc != CN_OK) return rc;
  const auto blobs = ck_blobs(m, n_sp);
  size_t tot = sizeof(CkHeader);
  for (auto &b : blobs) tot += sizeof(uint64_t) + ((b.second + 7) & ~(size_t)7);
  if ((size_t)bytes < tot) return fail(CN_ERR_ARG, "checkpoint buffer too small (%zu needed)", tot);
  char *p = static_cast<char *>(buf);
  CkHeader h{};
  h.magic = 0x434E434B50543031ull;  // "CNCKPT01"
  h.k = m->k;
  h.n_sp = n_sp;
  h.win_idx = m->win_idx;
  h.n_blob = (int64_t)blobs.size();
  h.dt = m->dt;
  h.state_pending = m->state_pending ? 1 : 0;
  h.window = m->window ? 1 : 0;
  h.layout = ck_layout_hash(m);
  memcpy(p, &h, sizeof(h));
  p += sizeof(h);
  for (auto &b : blobs) {
    const uint64_t sz = b.second;
    memcpy(p, &sz, sizeof(sz));
    p += sizeof(sz);
    if (sz) CU(cudaMemcpy(p, b.first, sz, cudaMemcpyDeviceToHost));
    p += (sz + 7) & ~(size_t)7;
  }
  return CN_OK;
}

extern "C" int cn_checkpoint_load(cn_model *m, const void *buf, int64_t bytes) {
  if (!m || !buf) return fail(CN_ERR_ARG, "NULL argument");
  if ((size_t)bytes < sizeof(CkHeader)) return fail(CN_ERR_ARG, "not a checkpoint");
  const char *p = static_cast<const char *>(buf);
  CkHeader h;
  memcpy(&h, p, sizeof(h));
  p += sizeof(h);
  if (h.magic != 0x434E434B50543031ull) return fail(CN_ERR_ARG, "not a checkpoint");
  if (!m->uploaded) {
    int rc = finalize(m, h.dt);
    if (rc != CN_OK) return rc;
  } else if (h.dt != m->dt) {
    return fail(CN_ERR_DT, "checkpoint was taken with dt = %.17g, the model runs with %.17g", h.dt, m->dt);
  }
  if (h.layout != ck_layout_hash(m) || (h.window != 0) != m->window)
    return fail(CN_ERR_ARG, "checkpoint of a different model, library build or launch mode");
  if (h.n_sp > m->sp_cap) return fail(CN_ERR_OVERFLOW, "checkpoint holds more spikes than the buffer");
  const auto blobs = ck_blobs(m, h.n_sp);
  if ((int64_t)blobs.size() != h.n_blob) return fail(CN_ERR_ARG, "checkpoint layout mismatch");
  CU(cudaStreamSynchronize(m->stream));
  const char *end = static_cast<const char *>(buf) + bytes;
  for (auto &b : blobs) {
    uint64_t sz;
    if (p + sizeof(sz) > end) return fail(CN_ERR_ARG, "checkpoint truncated");
    memcpy(&sz, p, sizeof(sz));
    p += sizeof(sz);
    if (sz != b.second || p + sz > end) return fail(CN_ERR_ARG, "checkpoint layout mismatch");
    if (sz) CU(cudaMemcpy(b.first, p, sz, cudaMemcpyHostToDevice));
    p += (sz + 7) & ~(size_t)7;
  }
  CU(cudaDeviceSynchronize());  // (the model's stream may not wait for the legacy default stream)
  m->k = h.k;
  m->win_idx = h.win_idx;
  m->state_pending = h.state_pending != 0;
  m->probe_rows = 0;
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
  if (m->ev0) cudaEventDestroy(m->ev0);
  if (m->ev1) cudaEventDestroy(m->ev1);
  delete m;
}

// debugging aid for DESIGN/bench: positions per task of the first tape class
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

#ifdef CN_TRACE
extern "C" int cn_debug_trace(long long *out) {
  return (int)cudaMemcpyFromSymbol(out, cn::g_trace, sizeof(long long) * 148 * 16 * 8 * 8);
}
#endif
