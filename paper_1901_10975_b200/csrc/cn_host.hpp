// cn_host.hpp -- host side of libcn: error reporting, mechanism metadata, helpers that spread the
// set-up over the host cores, the model structure (description, layout, device pointers) and the
// list scheduler of the warp-cooperative kernel.  Included by cn_api.cu only (one translation unit).
#pragma once

// ---------------------------------------------------------------------------------------------
// errors
// ---------------------------------------------------------------------------------------------

#define CN_GRAPH_STEPS 20  // per-dt launch sequences per CUDA graph

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
  uvec<int32_t> pp_local;   // local node of the instance in its cell (cell-window mode)
  int32_t *d_pp_local = nullptr;
  uint32_t *d_pp_wslot = nullptr;
  std::vector<int32_t> cls_cnt, cls_nodeoff;
  std::vector<int64_t> grp_instbase;
  // per-cell CSR of distributed instances sorted by local node
  std::vector<int64_t> cell_first;
  uvec<int64_t> cell_inst;  // empty: the caller's instances are ordered by node already (identity)
  int64_t inst(int64_t j) const { return cell_inst.empty() ? j : cell_inst[j]; }
  // point tables of a model whose node arrays stayed off the host (cn_model::node_arrays_host):
  // cm and area at the node of every instance
  uvec<double> pp_cm, pp_area;
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

// Options of one model, fixed at cn_model_create_opts ("key=value;key=value"; include/cn.h lists
// them).  The library reads no environment variable and has no global flag.
static const char *const kOptionKeys[] = {
    "tape", "tape_min_cells", "tape_min_group", "tape_w", "tape_s", "tape_ch", "tape_tmem",
    "tape_leaf_first", "tape_hcost", "tape_gran", "tape_mcost", "tape_bcost", "tape_pf",
    "tape_window", "tape_pbuf", "tape_ctas_per_sm", "force_g", "max_g", "warp_smem", "wpb",
    "graph", "onchip", "debug"};

struct Options {
  std::vector<std::pair<std::string, std::string>> kv;
  const char *get(const char *key) const {
    for (const auto &p : kv)
      if (p.first == key) return p.second.c_str();
    return nullptr;
  }
  // "k=v;k=v" (';', ',' or white space between the pairs); CN_OK or CN_ERR_ARG with a message
  int parse(const char *str) {
    kv.clear();
    if (!str) return CN_OK;
    std::string s(str);
    size_t i = 0;
    while (i < s.size()) {
      while (i < s.size() && (s[i] == ';' || s[i] == ',' || std::isspace((unsigned char)s[i]))) ++i;
      size_t j = i;
      while (j < s.size() && s[j] != ';' && s[j] != ',' && !std::isspace((unsigned char)s[j])) ++j;
      if (j == i) break;
      const std::string item = s.substr(i, j - i);
      i = j;
      const size_t eq = item.find('=');
      if (eq == std::string::npos || eq == 0 || eq + 1 == item.size())
        return fail(CN_ERR_ARG, "option '%s' is not key=value", item.c_str());
      const std::string key = item.substr(0, eq), val = item.substr(eq + 1);
      bool known = false;
      for (const char *k : kOptionKeys) known = known || key == k;
      if (!known) return fail(CN_ERR_ARG, "unknown option '%s'", key.c_str());
      char *end = nullptr;
      (void)std::strtod(val.c_str(), &end);
      if (!end || *end != '\0') return fail(CN_ERR_ARG, "option '%s': '%s' is not a number", key.c_str(), val.c_str());
      kv.emplace_back(key, val);
    }
    return CN_OK;
  }
};

// The caller's compact arrays on the device, from which the tapes of the interleaved groups are
// expanded (cn_expand.cuh).  A thread of cn_model_create uploads them while the host compiles the
// layout (joined before create returns: the caller's arrays are not read afterwards); finalize()
// uploads what is missing from the model's copies and releases everything once the tapes stand.
struct RawDev {
  double *cm = nullptr, *ri = nullptr, *area = nullptr;
  std::vector<double *> param;   // per table: [n_param][n] as given, NULL = not on the device
  std::vector<int32_t *> node;   // per table
  std::vector<void *> tmp;       // layout tables of the expansion kernels
  std::atomic<bool> cancel{false};  // the layout found no use for the rest
  cudaError_t err = cudaSuccess;
  void release() {
    for (double **p : {&cm, &ri, &area})
      if (*p) { cudaFree(*p); *p = nullptr; }
    for (double *&p : param)
      if (p) { cudaFree(p); p = nullptr; }
    for (int32_t *&p : node)
      if (p) { cudaFree(p); p = nullptr; }
    for (void *p : tmp) cudaFree(p);
    tmp.clear();
  }
};

struct RawSrc {  // one table of the description, wherever it lives on the host
  const int32_t *node;
  const double *param;
  int64_t n;
  int n_param;
  bool want;  // distributed with parameters (the tables a tape can hold or fold)
};

struct cn_model {
  Options options;
  RawDev raw;
  const char *opt(const char *key) const { return options.get(key); }
  // description (deep copy)
  int32_t n_cell = 0;
  int64_t N = 0;
  std::vector<int64_t> cell_first;
  uvec<int32_t> parent;
  uvec<double> area, ri, cm;
  bool node_arrays_host = true;  // false: area / ri / cm live on the device only (RawDev), see cn_model_create_opts
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
  bool cwindow = false;             // cell-window mode (cn_cell.cuh): one CTA keeps one cell on chip
  int cwin_grid = 0, cwin_threads = 256;  //   for a window of up to win_steps steps
  size_t cwin_smem = 0;
  std::vector<std::vector<uint16_t>> cwin_perm;  // per class: local node -> plan position
  bool window = false;              // window mode: one launch of the interleaved kernel per
  int win_steps = 0;                //   up to win_steps steps (cn_tape.cuh)
  int64_t win_idx = 0;
  std::vector<int> ktime_steps;     // steps covered by each kernel-timing sample
  bool state_pending = false;       // nrn_state of the last step has not been applied yet
  int n_cgroup = 0;                 // warp-cooperative groups come first in the group numbering
  std::vector<double> cai0;         // initial cai per caller node (when any table needs it)
  int warp_smem_doubles = 0, wpb = 4;
  bool step_attr_set[16] = {};      // shared-memory opt-in of step_kernel<WPB> done on this model's device
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
  int ktime_every = 0, ktime_which = 0;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ktime_ev;
  size_t ktime_used = 0;
  // CUDA graph of CN_GRAPH_STEPS per-dt launch sequences (cn_api.cu run_steps)
  bool graph_on = true;
  cudaGraphExec_t graph_exec = nullptr;
  cudaStream_t cap_stream = nullptr;
  int64_t graph_kernels = 0, graph_replays = 0, direct_steps = 0;
  // checkpoints / state read-back
  uint64_t ck_hash = 0;
  bool ck_hash_done = false;
  void *d_scratch = nullptr;
  size_t scratch_bytes = 0;
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

