// cn_api.cu -- host side of libcn: validation, shape classes, permutation, upload, step loop.
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


// ---------------------------------------------------------------------------------------------
// errors
// ---------------------------------------------------------------------------------------------

static thread_local char g_err[512] = "";

static int fail(int code, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

#define CU(call)                                                                         \
  do {                                                                                   \
    cudaError_t e_ = (call);                                                             \
    if (e_ != cudaSuccess)                                                               \
      return fail(e_ == cudaErrorMemoryAllocation ? CN_ERR_NOMEM : CN_ERR_CUDA,          \
                  "%s failed: %s", #call, cudaGetErrorString(e_));                       \
  } while (0)

extern "C" const char *cn_last_error(void) { return g_err; }

// ---------------------------------------------------------------------------------------------
// mechanism metadata
// ---------------------------------------------------------------------------------------------

struct TypeInfo { int n_param, n_state, n_global, point, n_dev_param; };

static bool type_info(int type, TypeInfo &ti) {
  switch (type) {
    case CN_PAS: ti = {2, 0, 0, 0, 0}; return true;       // folded into the static arrays
    case CN_HH: ti = {4, 3, 2, 0, 5}; return true;        // + invc
    case CN_EXPSYN: ti = {2, 1, 0, 1, 3}; return true;    // + scale
    case CN_EXP2SYN: ti = {3, 2, 0, 1, 5}; return true;   // + scale, factor
    case CN_ICLAMP: ti = {3, 0, 0, 1, 4}; return true;    // + scale
    case CN_HHFORM: ti = {1, 2, 16, 0, 2}; return true;   // + invc
    case CN_SK: ti = {1, 1, 4, 0, 2}; return true;        // + invc
    case CN_CADYN: ti = {0, 0, 4, 0, 0}; return true;
    case CN_AMPANMDA: ti = {0, 4, 7, 1, 1}; return true;  // scale
    case CN_GAP: ti = {2, 0, 0, 1, 2}; return true;       // g * scale, peer's position
  }
  return false;
}

static double h_vtrap(double x, double y) {
  double u = x / y;
  if (std::fabs(u) < 1e-6) return y * (1.0 - u / 2.0);
  return x / (std::exp(u) - 1.0);
}

static double h_exp2_factor(double t1, double t2) {
  double tp = (t1 * t2) / (t2 - t1) * std::log(t2 / t1);
  return 1.0 / (std::exp(-tp / t2) - std::exp(-tp / t1));
}

// std::vector that does not value-initialise (large set-up arrays are filled by all host cores)
template <class T>
struct NoInitAlloc {
  using value_type = T;
  NoInitAlloc() = default;
  template <class U> NoInitAlloc(const NoInitAlloc<U> &) {}
  T *allocate(size_t n) { return static_cast<T *>(::operator new(n * sizeof(T))); }
  void deallocate(T *p, size_t) { ::operator delete(p); }
  template <class U, class... A> void construct(U *p, A &&...a) {
    if constexpr (sizeof...(A) == 0) ::new ((void *)p) U; else ::new ((void *)p) U(std::forward<A>(a)...);
  }
  template <class U> bool operator==(const NoInitAlloc<U> &) const { return true; }
  template <class U> bool operator!=(const NoInitAlloc<U> &) const { return false; }
};
template <class T> using uvec = std::vector<T, NoInitAlloc<T>>;

// body(begin, end) over [0, n_items) on all host cores (create / first-run set-up only)
template <class F>
static void par_for(int64_t n_items, int64_t grain, F &&body) {
  const unsigned hw = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
  const unsigned nth = (unsigned)std::min<int64_t>(hw, std::max<int64_t>(1, n_items / grain));
  if (nth <= 1) {
    body((int64_t)0, n_items);
    return;
  }
  std::vector<std::thread> pool;
  for (unsigned t = 0; t < nth; ++t)
    pool.emplace_back([&body, n_items, nth, t] { body(n_items * t / nth, n_items * (t + 1) / nth); });
  for (auto &th : pool) th.join();
}

static unsigned par_threads(int64_t n_items, int64_t grain) {
  const unsigned hw = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
  return (unsigned)std::min<int64_t>(hw, std::max<int64_t>(1, n_items / grain));
}

// body(t) for t in [0, P) on P threads
template <class F>
static void par_run(unsigned P, F &&body) {
  if (P <= 1) {
    body(0u);
    return;
  }
  std::vector<std::thread> pool;
  for (unsigned t = 0; t < P; ++t) pool.emplace_back([&body, t] { body(t); });
  for (auto &th : pool) th.join();
}

// Stable counting sort of the items [0, n) by key(i) in [0, nb) on all cores: first[b] = number
// of items with a smaller key, rank[i] = position of item i in the sorted order.
template <class KeyF>
static void par_bucket(int64_t n, int64_t nb, KeyF &&key, std::vector<int64_t> &first,
                       uvec<int64_t> &rank) {
  unsigned P = par_threads(n, 1 << 16);
  while (P > 1 && (int64_t)P * nb > ((int64_t)32 << 20)) P /= 2;
  std::vector<std::vector<int64_t>> cnt(P);
  par_run(P, [&](unsigned t) {
    cnt[t].assign((size_t)nb, 0);
    for (int64_t i = n * t / P, e = n * (t + 1) / P; i < e; ++i) cnt[t][key(i)]++;
  });
  first.assign((size_t)nb + 1, 0);
  int64_t run = 0;
  for (int64_t b = 0; b < nb; ++b) {
    first[b] = run;
    for (unsigned t = 0; t < P; ++t) {
      const int64_t c = cnt[t][b];
      cnt[t][b] = run;
      run += c;
    }
  }
  first[nb] = run;
  rank.resize((size_t)n);
  par_run(P, [&](unsigned t) {
    for (int64_t i = n * t / P, e = n * (t + 1) / P; i < e; ++i) rank[i] = cnt[t][key(i)]++;
  });
}

// dst = src[0, n) copied by all cores (first touch of the fresh pages included)
template <class T>
static void par_assign(uvec<T> &dst, const T *src, int64_t n) {
  dst.resize((size_t)n);
  par_for(n, 1 << 18, [&](int64_t i0, int64_t i1) {
    if (i1 > i0) memcpy(dst.data() + i0, src + i0, (size_t)(i1 - i0) * sizeof(T));
  });
}

// validation passes run on all cores; the failure with the smallest index is the one reported
struct FirstErr {
  std::mutex mu;
  int64_t key = INT64_MAX;
  int code = CN_OK;
  char msg[256] = "";
  void set(int64_t k, int c, const char *fmt, ...) {
    char buf[256];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    std::lock_guard<std::mutex> lk(mu);
    if (k < key) {
      key = k;
      code = c;
      memcpy(msg, buf, sizeof(msg));
    }
  }
};

// ---------------------------------------------------------------------------------------------
// model
// ---------------------------------------------------------------------------------------------

struct HTable {
  int type = 0;
  TypeInfo ti{};
  int64_t n = 0;
  uvec<int32_t> node;
  uvec<double> param;  // [n_param][n]
  std::vector<double> glob;
  // layout
  int64_t n_dev = 0;               // padded device instance count
  uvec<int64_t> inst_pos;   // caller instance -> device instance (table arrays)
  uvec<int64_t> tape_loc;   // distributed: tape element of the first PARAMETER row of an
                                   // instance on a tape cell, else -1
  int64_t pp_tape_begin = 0;       // point: instances [pp_tape_begin, n) sit on tape cells
  // device
  double *d_param[CN_MAX_PARAM] = {};
  double *d_state[CN_MAX_STATE] = {};
  int64_t *d_pp_first = nullptr;
  int32_t *d_pp_slot = nullptr;
  int32_t *d_cls_cnt = nullptr, *d_cls_nodeoff = nullptr;
  int64_t *d_grp_instbase = nullptr;
  // host layout tables
  std::vector<int64_t> pp_first;
  uvec<int32_t> pp_slot;
  uvec<uint32_t> pp_wslot;  // window mode: element in one step's block of win_rows
  uint32_t *d_pp_wslot = nullptr;
  std::vector<int32_t> cls_cnt, cls_nodeoff;
  std::vector<int64_t> grp_instbase;
  // per-cell CSR of distributed instances sorted by local node
  std::vector<int64_t> cell_first;
  uvec<int64_t> cell_inst;
};

struct HTask {
  int p0 = 0, p1 = 0, b0 = 0, b1 = 0;  // forward / backward records in the class's program
  int nchunk = 0, tm_base = 0, pp0 = 0;  // pp0: ordinal of the warp's first point-process node
  uint32_t row0 = 0, nrows = 0, head = 0;
};

struct HTape {  // per class: the program of the interleaved kernel (cn_tape.cuh)
  std::vector<HTask> task;                   // one per warp
  std::vector<uint4> prog;                   // records of all warps, warp after warp
  int n_groups = 0;
  int64_t n_cells = 0;                       // the first n_cells of HClass::cells are tape cells
  std::vector<int32_t> order, pos_of;        // system row -> local node, local node -> system row
  std::vector<uint32_t> row;                 // per system row: first tape row of the node's record
  std::vector<uint8_t> has_pp;               // per local node
  std::vector<std::vector<int32_t>> tab_row; // [table][local node]: first row of its block or -1
  std::vector<int32_t> cai_row, ica_row, pp_row, vcopy_row;  // per local node or -1
  std::vector<int32_t> pp_ord;               // ordinal of a node among the class's has_pp nodes
  int n_pp = 0;
  int n_rows = 0, prog_off = 0;
  int n_srow = 0;                            // rows of the shared-memory system (the rest: TMEM)
  int n_bar = 0;                             // signal mbarriers (one per signalling record)
  double sim_makespan = 0.0, sim_work = 0.0; // schedule quality (cn_debug_tasks)
};

struct HClass {
  HTape tp;
  int n = 0, G = 1, lgG = 0, rounds = 0, needs_ica = 0;
  int rep_cell = -1;
  int64_t count = 0;
  int sched_off = 0;
  std::vector<int32_t> cells;
  std::vector<uint32_t> sched;
  std::vector<int32_t> node_off;  // local node -> slot offset round*32 + p*G (root: rounds*32)
  int nodeoff_off = 0;
};

struct cn_model {
  // description (deep copy)
  int32_t n_cell = 0;
  int64_t N = 0;
  std::vector<int64_t> cell_first;
  uvec<int32_t> parent;
  uvec<double> area, ri, cm;
  std::vector<double> thr;
  double v_init = -65.0, celsius = 6.3;
  std::vector<HTable> tab;
  int64_t n_netcon = 0;
  uvec<int32_t> nc_src, nc_tgt_mech;
  uvec<int64_t> nc_tgt_inst;
  uvec<double> nc_w, nc_delay;
  std::vector<int32_t> stim_gid;
  std::vector<double> stim_t;
  int32_t n_src = 0;
  // layout
  std::vector<HClass> cls;
  std::vector<GroupInfo> grp;
  std::vector<int32_t> cell_cls, cell_grp, cell_slot;
  uvec<int64_t> node_pos;  // caller node -> device node
  std::vector<int32_t> dist_nodes;  // per class and distributed table: local node lists
  int64_t n_pnode = 0, n_ab = 0;
  int32_t n_pcell = 0;
  // interleaved (tape) groups
  std::vector<TapeGroup> tgrp;
  std::vector<uint8_t> cell_tape;   // per caller cell
  int64_t n_tape = 0;               // doubles
  int64_t win_stride = 0, win_ninst = 0;  // window mode: doubles per step in win_rows / win_deliv
  int tape_prog_cap = 0, tape_sys_cap = 0, tape_bar_cap = 0;
  int tape_W = 8, tape_S = 4, tape_CH = 8;  // warps per group, ring stages, rows per chunk
  double tape_hcost = 0.0;  // hand-over between warps, in chain nodes
  double tape_gran = 4.0;  // whole subtrees are cut to at most 1 / (tape_gran * W) of a cell's work
  double tape_mcost_scale = 0.5, tape_bcost = 1.0;  // cost model of the schedule (units: chain nodes;
                                                    // swept on config 4, see profiles/r01_README.md)
  bool tape_leaf_first = false;     // scheduling variant: all whole subtrees before any upper node
  bool tape_tmem = true;            // plain chain nodes keep their system rows in tensor memory
  int tape_ctas = 0;                // persistent CTAs of the interleaved kernel (0: not yet known)
  bool window = false;              // window mode: one launch of the interleaved kernel per
  int win_steps = 0;                //   up to win_steps steps (cn_tape.cuh)
  int64_t win_idx = 0;
  std::vector<int> ktime_steps;     // steps covered by each kernel-timing sample
  bool state_pending = false;       // nrn_state of the last step has not been applied yet
  int n_cgroup = 0;                 // warp-cooperative groups come first in the group numbering
  std::vector<double> cai0;         // initial cai per caller node (when any table needs it)
  int warp_smem_doubles = 0, wpb = 4;
  bool any_ica = false, any_cai = false;
  // run state
  double dt = 0.0;
  int64_t k = 0;
  bool uploaded = false;
  int64_t launches = 0;
  int64_t sp_cap = 0;
  cudaStream_t stream = 0;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  bool timed = false;
  int ktime_every = 0;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ktime_ev;
  size_t ktime_used = 0;
  // probes
  std::vector<int32_t> probe;
  int64_t probe_cap = 0, probe_rows = 0;
  // device
  std::vector<void *> dev_allocs;
  DModel hm{};
  DModel *d_m = nullptr;
  double *d_v = nullptr, *d_cai = nullptr, *d_trace = nullptr, *d_gather = nullptr;
  int64_t *d_node_pos = nullptr, *d_probe_pos = nullptr;
  int32_t *d_overflow = nullptr;
  unsigned long long *d_nsp = nullptr;
  int32_t *d_sp_gid = nullptr;
  int64_t *d_sp_step = nullptr;
};


template <class T, class A>
static int dev_upload(cn_model *m, const std::vector<T, A> &h, T **out, size_t min_elems = 1) {
  size_t n = std::max(h.size(), min_elems);
  void *p = nullptr;
  CU(cudaMalloc(&p, n * sizeof(T)));
  m->dev_allocs.push_back(p);
  if (!h.empty()) CU(cudaMemcpy(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
  if (h.size() < n)
    CU(cudaMemset((char *)p + h.size() * sizeof(T), 0, (n - h.size()) * sizeof(T)));
  *out = (T *)p;
  return CN_OK;
}

template <class T>
static int dev_alloc(cn_model *m, size_t n, T **out, bool zero = true) {
  void *p = nullptr;
  if (n == 0) n = 1;
  CU(cudaMalloc(&p, n * sizeof(T)));
  m->dev_allocs.push_back(p);
  if (zero) CU(cudaMemset(p, 0, n * sizeof(T)));
  *out = (T *)p;
  return CN_OK;
}

// ---------------------------------------------------------------------------------------------
// list scheduling of the elimination (Hu's level algorithm for in-trees, P nodes per round,
// at most one child of a parent per round so that the parent updates never collide)
// ---------------------------------------------------------------------------------------------

static int hu_schedule(int n, const int32_t *par, int P, std::vector<uint32_t> &out) {
  out.clear();
  if (n <= 1) return 0;
  std::vector<int> depth(n, 0), left(n, 0), used(n, -1);
  int maxd = 0;
  for (int i = 1; i < n; ++i) {
    depth[i] = depth[par[i]] + 1;
    left[par[i]]++;
    maxd = std::max(maxd, depth[i]);
  }
  std::vector<std::vector<int>> bucket(maxd + 1);
  for (int i = 1; i < n; ++i)
    if (left[i] == 0) bucket[depth[i]].push_back(i);
  int remaining = n - 1, round = 0;
  std::vector<int> picked;
  while (remaining > 0) {
    picked.clear();
    for (int dl = maxd; dl >= 1 && (int)picked.size() < P; --dl) {
      auto &bk = bucket[dl];
      for (size_t j = 0; j < bk.size() && (int)picked.size() < P;) {
        int i = bk[j];
        if (used[par[i]] != round) {
          used[par[i]] = round;
          picked.push_back(i);
          bk[j] = bk.back();
          bk.pop_back();
        } else {
          ++j;
        }
      }
    }
    for (int i : picked) {
      out.push_back((uint32_t)i | ((uint32_t)par[i] << 16));
      --remaining;
      int p = par[i];
      if (--left[p] == 0 && p != 0) bucket[depth[p]].push_back(p);
    }
    for (int j = (int)picked.size(); j < P; ++j) out.push_back(CN_IDLE | (CN_IDLE << 16));
    ++round;
  }
  return round;
}

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
  const bool dbg = std::getenv("CN_DEBUG") != nullptr;
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
        h = mix64(h, (uint64_t)(T.node[T.cell_inst[j]] - f));
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
        if (T.node[T.cell_inst[T.cell_first[x] + j]] - fx !=
            T.node[T.cell_inst[T.cell_first[y] + j]] - fy)
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
  if (const char *e = std::getenv("CN_TAPE")) tape_mode = std::atoi(e);
  int64_t tape_min_cells = 8192;
  if (const char *e = std::getenv("CN_TAPE_MIN_CELLS")) tape_min_cells = std::atoll(e);
  int tape_min_group = 16;  // a ragged last group needs at least this many cells
  if (const char *e = std::getenv("CN_TAPE_MIN_GROUP")) tape_min_group = std::max(1, std::atoi(e));
  // A smaller model goes to the interleaved kernel too if ALL of it fits there (then it runs in
  // window mode: one launch per min-delay window instead of three per dt) and its groups fill at
  // least a quarter of their lanes; decided after the programs are compiled (below).
  const bool auto_small = tape_mode == -1 && nc < tape_min_cells && nc > 0;
  if (auto_small && !std::getenv("CN_TAPE_MIN_GROUP")) tape_min_group = 1;
  const bool tape_on = tape_mode == 1 || (tape_mode == -1 && nc >= tape_min_cells) || auto_small;
  // W warps per group (CTA), each with a ring of S chunks x CH rows; the whole CTA must fit the
  // 227 KB of shared memory next to the group's system (512 B per node)
  m->tape_W = 8;
  if (const char *e = std::getenv("CN_TAPE_W")) m->tape_W = std::min(16, std::max(1, std::atoi(e)));
  m->tape_S = 2;
  m->tape_CH = 16;
  if (const char *e = std::getenv("CN_TAPE_S")) m->tape_S = std::min(4, std::max(2, std::atoi(e)));
  if (const char *e = std::getenv("CN_TAPE_CH")) m->tape_CH = std::min(63, std::max(7, std::atoi(e)));
  if (const char *e = std::getenv("CN_TAPE_TMEM")) m->tape_tmem = std::atoi(e) != 0;
  if (const char *e = std::getenv("CN_TAPE_LEAF_FIRST")) m->tape_leaf_first = std::atoi(e) != 0;
  if (const char *e = std::getenv("CN_TAPE_HCOST")) m->tape_hcost = std::atof(e);
  if (const char *e = std::getenv("CN_TAPE_GRAN")) m->tape_gran = std::max(1.0, std::atof(e));
  if (const char *e = std::getenv("CN_TAPE_MCOST")) m->tape_mcost_scale = std::atof(e);
  if (const char *e = std::getenv("CN_TAPE_BCOST")) m->tape_bcost = std::atof(e);
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
  if (!std::getenv("CN_TAPE_CH")) {
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
          const int x = (int)(T.node[T.cell_inst[q]] - f);
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
    if (m->tape_W > 8 || std::getenv("CN_TAPE_CH") || 2 * (smem + 1024) <= 233472 || next_ch == 0 ||
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
  if (const char *e = std::getenv("CN_FORCE_G")) force_g = std::atoi(e);
  int max_g = 4;
  if (const char *e = std::getenv("CN_MAX_G")) max_g = std::max(1, std::atoi(e));
  int64_t smem_cap = 24 * 1024;
  if (const char *e = std::getenv("CN_WARP_SMEM")) smem_cap = std::atoll(e);
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
    int G = 1;
    while (G * 2 <= max_g && G * 2 <= ccount && (int64_t)K.n * arrays * 8 * G * 2 <= smem_cap &&
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
    T.inst_pos.resize((size_t)T.n);
    par_for(T.n, 1 << 18, [&](int64_t i0, int64_t i1) {
      std::fill(T.inst_pos.begin() + i0, T.inst_pos.begin() + i1, (int64_t)-1);
    });
    if (T.ti.point) {
      // instances ordered by group (stable); cooperative groups: slot = local node * G + cell
      // slot in shared memory; tape groups: element of the node's conductance row on the tape
      uvec<int64_t> rank;
      par_bucket(T.n, ng, [&](int64_t i) { return m->cell_grp[cell_of[T.node[i]]]; }, T.pp_first,
                 rank);
      T.pp_slot.resize((size_t)T.n);
      T.pp_wslot.resize((size_t)T.n);
      par_for(T.n, 1 << 16, [&](int64_t i0, int64_t i1) {
        for (int64_t i = i0; i < i1; ++i) {
          const int32_t cell = cell_of[T.node[i]];
          const int g = m->cell_grp[cell];
          const int64_t pos = rank[i];
          T.inst_pos[i] = pos;
          const int32_t local = (int32_t)(T.node[i] - m->cell_first[cell]);
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
      T.tape_loc.resize((size_t)T.n);
      par_for(T.n, 1 << 18, [&](int64_t i0, int64_t i1) {
        std::fill(T.tape_loc.begin() + i0, T.tape_loc.begin() + i1, (int64_t)-1);
      });
      T.cls_cnt.assign(m->cls.size(), 0);
      T.cls_nodeoff.assign(m->cls.size(), 0);
      for (int kc = 0; kc < (int)m->cls.size(); ++kc) {
        const HClass &K = m->cls[kc];
        const int32_t rc = K.rep_cell;
        T.cls_cnt[kc] = (int32_t)(T.cell_first[rc + 1] - T.cell_first[rc]);
        T.cls_nodeoff[kc] = (int32_t)dist_nodes.size();
        for (int64_t j = T.cell_first[rc]; j < T.cell_first[rc + 1]; ++j)
          dist_nodes.push_back((int32_t)(T.node[T.cell_inst[j]] - m->cell_first[rc]));
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
      par_for(nc, 256, [&](int64_t cc0, int64_t cc1) {
       for (int64_t c = cc0; c < cc1; ++c) {
        const int g = m->cell_grp[c];
        if (g < ngc) {
          const int G = m->cls[m->grp[g].cls].G;
          const int64_t b0 = T.grp_instbase[g];
          int64_t kk = 0;
          for (int64_t j = T.cell_first[c]; j < T.cell_first[c + 1]; ++j, ++kk)
            T.inst_pos[T.cell_inst[j]] = b0 + kk * G + m->cell_slot[c];
        } else if (T.type != CN_PAS && T.type != CN_CADYN) {
          const TapeGroup &tg = m->tgrp[g - ngc];
          const HTape &P = m->cls[tg.cls].tp;
          for (int64_t j = T.cell_first[c]; j < T.cell_first[c + 1]; ++j) {
            const int64_t i = T.cell_inst[j];
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
  if (const char *e = std::getenv("CN_WPB")) wpb = std::max(1, std::atoi(e));
  while (wpb > 1 && wbytes * wpb > 110 * 1024) wpb /= 2;
  m->wpb = wpb;
  lap("groups, instance layout");
  return CN_OK;
}


// ---------------------------------------------------------------------------------------------
// first cn_run: dt-dependent constants (row-normalised system), initial states, upload
// ---------------------------------------------------------------------------------------------

static int finalize(cn_model *m, double dt) {
  const bool dbg = std::getenv("CN_DEBUG") != nullptr;
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
  // row-normalised static arrays:  c_i = 1e-3 cm_i/dt,  b' = b/c_i,  a' = a/c_parent,
  // dstat = (c - b - sum_children a + sum static g)/c,  rstat = (sum static g*e)/c
  uvec<double> invc((size_t)N), bn((size_t)N), an((size_t)N);
  std::vector<double> dstat((size_t)m->n_pnode, 1.0), rstat((size_t)m->n_pnode, 0.0);
  // one arena: [schedule-ordered v of the cooperative groups | tapes of the interleaved groups]
  uvec<double> v0((size_t)(m->n_ab + m->n_tape));
  double *tape = v0.data() + m->n_ab;
  uvec<double> dsum((size_t)N), rsum((size_t)N);
  uvec<int32_t> cell_of_node((size_t)N);
  par_for((int64_t)v0.size(), 1 << 20, [&](int64_t i0, int64_t i1) {
    std::fill(v0.begin() + i0, v0.begin() + i1, 0.0);
  });
  par_for(N, 1 << 20, [&](int64_t i0, int64_t i1) {
    std::fill(bn.begin() + i0, bn.begin() + i1, 0.0);
    std::fill(an.begin() + i0, an.begin() + i1, 0.0);
    std::fill(rsum.begin() + i0, rsum.begin() + i1, 0.0);
  });
  // cells are independent (a parent sits in the same cell): all host cores
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
  for (const HTable &T : m->tab)
    if (T.type == CN_PAS)  // (at most one instance of a table per node: no two threads meet)
      par_for(T.n, 65536, [&](int64_t q0, int64_t q1) {
        for (int64_t i = q0; i < q1; ++i) {
          const double g = T.param[i], e = T.param[T.n + i];
          dsum[T.node[i]] += g;
          rsum[T.node[i]] += g * e;
        }
      });
  // inverse map: (group, slot) -> caller cell
  std::vector<int32_t> cell_of_pcell((size_t)m->n_pcell, -1);
  for (int32_t c = 0; c < m->n_cell; ++c) {
    const int g = m->cell_grp[c];
    const int32_t cb = g < m->n_cgroup ? m->grp[g].cell_base : m->tgrp[g - m->n_cgroup].cell_base;
    cell_of_pcell[cb + m->cell_slot[c]] = c;
  }
  // interleaved groups: whole rows of 32 lanes at a time (contiguous writes; the 32 cells are
  // read as 32 sequential streams); a, b, d, r precede the node's v row
  par_for((int64_t)m->tgrp.size(), 1, [&](int64_t g0, int64_t g1) {
    for (int64_t g = g0; g < g1; ++g) {
      const TapeGroup &tg = m->tgrp[g];
      const HClass &K = m->cls[tg.cls];
      int64_t f[32];
      for (int l = 0; l < tg.ncell; ++l) f[l] = m->cell_first[cell_of_pcell[tg.cell_base + l]];
      for (int j = 0; j < K.n; ++j) {
        double *rec = tape + tg.tape_base + ((int64_t)K.tp.row[K.tp.pos_of[j]] + 4) * 32;
        for (int l = 0; l < tg.ncell; ++l) {
          const int64_t i = f[l] + j;
          rec[-4 * 32 + l] = an[i];
          rec[-3 * 32 + l] = bn[i];
          rec[-2 * 32 + l] = dsum[i] * invc[i];
          rec[-1 * 32 + l] = rsum[i] * invc[i];
          rec[l] = m->v_init;
        }
      }
    }
  });
  if (m->n_cgroup > 0)
    par_for(N, 65536, [&](int64_t i0, int64_t i1) {
      for (int64_t i = i0; i < i1; ++i) {
        if (m->cell_tape[cell_of_node[i]]) continue;
        const int64_t q = m->node_pos[i];
        dstat[q] = dsum[i] * invc[i];
        rstat[q] = rsum[i] * invc[i];
        v0[q] = m->v_init;
      }
    });
  lap("static rows");
  // idle lanes of a ragged tape group: unit diagonal, everything else zero; cai rows
  for (const TapeGroup &tg : m->tgrp) {
    const HTape &P = m->cls[tg.cls].tp;
    for (int j = 0; j < m->cls[tg.cls].n; ++j)
      for (int l = tg.ncell; l < 32; ++l) tape[tg.tape_base + ((int64_t)P.row[j] + 2) * 32 + l] = 1.0;
  }
  for (const TapeGroup &tg : m->tgrp) {  // the copy of v at the head of every mechanism record
    const HTape &P = m->cls[tg.cls].tp;
    for (int i = 0; i < m->cls[tg.cls].n; ++i)
      if (P.vcopy_row[i] >= 0)
        for (int l = 0; l < 32; ++l)
          tape[tg.tape_base + (int64_t)P.vcopy_row[i] * 32 + l] = m->v_init;
  }
  if (m->any_cai)
    for (int32_t c = 0; c < m->n_cell; ++c) {
      if (!m->cell_tape[c]) continue;
      const TapeGroup &tg = m->tgrp[m->cell_grp[c] - m->n_cgroup];
      const HTape &P = m->cls[tg.cls].tp;
      const int64_t f = m->cell_first[c];
      for (int i = 0; i < m->cls[tg.cls].n; ++i)
        if (P.cai_row[i] >= 0)
          tape[tg.tape_base + (int64_t)P.cai_row[i] * 32 + m->cell_slot[c]] = m->cai0[f + i];
    }
  lap("idle lanes, v copies, cai");
  // schedule-ordered off-diagonals
  std::vector<double> a_s((size_t)m->n_ab, 0.0), b_s((size_t)m->n_ab, 0.0);
  std::vector<uint32_t> sched_all;
  std::vector<int32_t> nodeoff_all;
  std::vector<ClassInfo> cinfo(m->cls.size());
  for (size_t kc = 0; kc < m->cls.size(); ++kc) {
    const HClass &K = m->cls[kc];
    cinfo[kc] = ClassInfo{K.n, K.G, K.lgG, K.rounds, K.sched_off, K.needs_ica, K.nodeoff_off, 0};
    sched_all.insert(sched_all.end(), K.sched.begin(), K.sched.end());
    nodeoff_all.insert(nodeoff_all.end(), K.node_off.begin(), K.node_off.end());
  }
  for (int g = 0; g < ng; ++g) {
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
  lap("coop schedule arrays");
  // thresholds, flags, gids per permuted cell
  std::vector<double> thr((size_t)m->n_pcell, 0.0);
  std::vector<unsigned char> flag((size_t)m->n_pcell, 0);
  std::vector<int32_t> gid_of((size_t)m->n_pcell, -1);
  for (int32_t pc = 0; pc < m->n_pcell; ++pc) {
    const int32_t c = cell_of_pcell[pc];
    if (c < 0) continue;
    thr[pc] = m->thr[c];
    flag[pc] = m->v_init > m->thr[c];
    gid_of[pc] = c;
  }
  // cai per node of the cooperative groups
  std::vector<double> cai;
  if (m->any_cai) {
    cai.assign((size_t)m->n_pnode, 1e-4);
    for (int64_t i = 0; i < N; ++i)
      if (!m->cell_tape[cell_of_node[i]]) cai[m->node_pos[i]] = m->cai0[i];
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
    for (const HTable &T : m->tab)
      if (T.ti.point)
        for (int64_t i = 0; i < T.n; ++i)
          if (!m->cell_tape[cell_of_node[T.node[i]]]) {
            double &d = dstat[m->node_pos[T.node[i]]];
            d = -std::fabs(d);
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
    // instances are independent (each writes its own elements): all host cores
    par_for(T.n, 4096, [&](int64_t ii0, int64_t ii1) {
     for (int64_t i = ii0; i < ii1; ++i) {
      const int32_t nd_i = T.node[i];
      double P[CN_MAX_PARAM] = {0.0}, S[CN_MAX_STATE] = {0.0};
      for (int j = 0; j < T.ti.n_param; ++j) P[j] = T.param[(size_t)j * T.n + i];
      const double scale = 100.0 / m->area[nd_i] * invc[nd_i];
      const double v = m->v_init;
      switch (T.type) {
        case CN_HH: {
          P[4] = invc[nd_i];
          double al, be;
          al = 0.1 * h_vtrap(-(v + 40.0), 10.0); be = 4.0 * std::exp(-(v + 65.0) / 18.0);
          S[0] = al / (al + be);
          al = 0.07 * std::exp(-(v + 65.0) / 20.0); be = 1.0 / (std::exp(-(v + 35.0) / 10.0) + 1.0);
          S[1] = al / (al + be);
          al = 0.01 * h_vtrap(-(v + 55.0), 10.0); be = 0.125 * std::exp(-(v + 65.0) / 80.0);
          S[2] = al / (al + be);
          break;
        }
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
          P[1] = invc[nd_i];
          S[0] = 1.0 / (1.0 + std::exp((T.glob[4] - v) / T.glob[5]));
          S[1] = 1.0 / (1.0 + std::exp((T.glob[10] - v) / T.glob[11]));
          break;
        case CN_SK: {
          P[1] = invc[nd_i];
          double ca = m->any_cai ? m->cai0[nd_i] : 1e-4;
          if (ca < 1e-9) ca = 1e-9;
          S[0] = 1.0 / (1.0 + std::pow(T.glob[1] / ca, T.glob[2]));
          break;
        }
        case CN_AMPANMDA: P[0] = scale; break;
        case CN_GAP:  // positions in the voltage arena (exact in a double: < 2^53)
          P[0] *= scale;
          P[1] = (double)m->node_pos[(int64_t)P[1]];
          break;
        default: break;
      }
      if (!T.ti.point && T.tape_loc[i] >= 0) {  // the instance lives on a tape
        double *rec = tape + T.tape_loc[i];
        for (int j = 0; j < T.ti.n_dev_param; ++j) rec[(size_t)j * 32] = P[j];
        for (int j = 0; j < T.ti.n_state; ++j) rec[(size_t)(T.ti.n_dev_param + j) * 32] = S[j];
      } else if (T.inst_pos[i] >= 0) {
        const int64_t q = T.inst_pos[i];
        for (int j = 0; j < T.ti.n_dev_param; ++j) par[j][q] = P[j];
        for (int j = 0; j < T.ti.n_state; ++j) st[j][q] = S[j];
      }
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
  // the arena (filled above, including the mechanism rows of the tapes) and the programs
  {
    UP(v0, m->d_v);
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
    H.tape_W = m->tape_W;
    H.tape_S = m->tape_S;
    H.tape_CH = m->tape_CH;
    H.tape_prog_cap = std::max(m->tape_prog_cap, 1);
    H.tape_sys_cap = std::max(m->tape_sys_cap, 1);
    H.tape_bar_cap = m->tape_bar_cap;
    H.tape_pf = 0;  // measured on config 4: prefetching ahead of the ring only costs (0: off)
    if (const char *e = std::getenv("CN_TAPE_PF")) H.tape_pf = std::max(0, std::min(4096, std::atoi(e)));
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
  lap("arena + programs upload");
  // NetCons: CSR by source gid, sorted by delay steps (stable in caller order)
  {
    std::vector<int64_t> order((size_t)m->n_netcon);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int64_t x, int64_t y) {
      if (m->nc_src[x] != m->nc_src[y]) return m->nc_src[x] < m->nc_src[y];
      return dsteps[x] < dsteps[y];
    });
    std::vector<int64_t> src_first((size_t)m->n_src + 1, 0);
    for (int64_t i = 0; i < m->n_netcon; ++i) src_first[m->nc_src[i] + 1]++;
    for (int32_t s = 0; s < m->n_src; ++s) src_first[s + 1] += src_first[s];
    std::vector<int32_t> nd((size_t)m->n_netcon), ntab((size_t)m->n_netcon);
    std::vector<int64_t> ninst((size_t)m->n_netcon);
    std::vector<double> nw((size_t)m->n_netcon);
    for (int64_t j = 0; j < m->n_netcon; ++j) {
      const int64_t i = order[j];
      nd[j] = dsteps[i];
      ntab[j] = m->nc_tgt_mech[i];
      ninst[j] = m->tab[m->nc_tgt_mech[i]].inst_pos[m->nc_tgt_inst[i]];
      nw[j] = m->nc_w[i];
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
    if (const char *e = std::getenv("CN_TAPE_WINDOW")) ok = ok && std::atoi(e) != 0;
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
      rc = dev_alloc(m, (size_t)m->hm.n_tgroup, &H.win_done); if (rc != CN_OK) return rc;
      rc = dev_alloc(m, 1, &H.win_ticket); if (rc != CN_OK) return rc;
      H.win_mark_cap = H.maxd + 64;
      rc = dev_alloc(m, (size_t)H.win_mark_cap, &H.win_mark_step); if (rc != CN_OK) return rc;
      rc = dev_alloc(m, (size_t)H.win_mark_cap, &H.win_mark_nsp); if (rc != CN_OK) return rc;
    }
  }
  // spikes
  rc = dev_alloc(m, (size_t)m->sp_cap, &m->d_sp_gid, false); if (rc) return rc;
  rc = dev_alloc(m, (size_t)m->sp_cap, &m->d_sp_step, false); if (rc) return rc;
  rc = dev_alloc(m, 1, &m->d_nsp); if (rc) return rc;
  rc = dev_alloc(m, 1, &m->d_overflow); if (rc) return rc;
  H.sp_gid = m->d_sp_gid; H.sp_step = m->d_sp_step; H.n_sp = m->d_nsp; H.sp_cap = m->sp_cap;
  H.overflow = m->d_overflow;
  lap("window buffers, spikes");
  // caller-order lookup for cn_get_v, probes
  UP(m->node_pos, m->d_node_pos);
  rc = dev_alloc(m, (size_t)std::max<int64_t>(N, 1), &m->d_gather, false); if (rc) return rc;
  if (!m->probe.empty()) {
    std::vector<int64_t> pp(m->probe.size());
    for (size_t j = 0; j < pp.size(); ++j) pp[j] = m->node_pos[m->probe[j]];
    UP(pp, m->d_probe_pos);
    rc = dev_alloc(m, (size_t)(m->probe_cap * (int64_t)m->probe.size()), &m->d_trace, false);
    if (rc) return rc;
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
  CU(cudaEventCreate(&m->ev0));
  CU(cudaEventCreate(&m->ev1));
  m->dt = dt;
  m->uploaded = true;
  return CN_OK;
}

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
