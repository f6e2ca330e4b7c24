// cn_device.cuh -- device-side data model and kernels of libcn (sm_100a, fp64).
//
// One warp integrates one GROUP = G cells of one shape class (same topology and same placement
// of distributed mechanisms) for one dt, with P = 32/G lanes per cell:
//   cur    : per mechanism table, D += g, R += g*E into a zeroed shared-memory system
//            (nrn_cur; conductance form L160)
//   solve  : Hines elimination in shared memory, list-scheduled in rounds of P independent nodes
//            (L62, L66, L196).  EVERY per-node array (v, static diagonal / rhs, off-diagonals) is
//            stored in schedule order [round][lane], so each round is one coalesced 256 B load per
//            array, prefetched several rounds ahead in registers; a node's static terms and old v
//            are added when the node is eliminated, and v_new is stored from the back-substitution
//            round (L66).  There is no separate load or store pass over the nodes.
//   state  : per mechanism table, cnexp / implicit updates with the new v (L67, L278)
//   detect : warp-ballot threshold detection on the root nodes, spike append (L68)
// The linear system is the paper's backward-Euler system written for v_new instead of delta-v and
// with every row divided by c_i = 1e-3 cm_i/dt.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define CN_MAX_TABLES 24
#define CN_MAX_PARAM 8
#define CN_MAX_STATE 4
#define CN_MAX_GLOBAL 16
#define CN_IDLE 0xFFFFu

namespace cn {

enum { T_PAS = 1, T_HH = 2, T_EXPSYN = 3, T_EXP2SYN = 4, T_ICLAMP = 5, T_HHFORM = 6, T_SK = 7,
       T_CADYN = 8, T_AMPANMDA = 9, T_GAP = 10 };

struct DTable {
  int type, is_point, n_param, n_state;
  int64_t pp_tape_begin, pp_tape_end;  // point tables: instance range that sits on tape groups
  double *param[CN_MAX_PARAM];   // permuted SoA, incl. derived per-instance constants (see host)
  double *state[CN_MAX_STATE];
  double glob[CN_MAX_GLOBAL];
  const uint32_t *pp_wslot;      // point tables, window mode: element of the node's conductance row
                                 // in one step's block of win_rows
  int64_t pp_goff;               // point tables, window mode: first column of the table in win_deliv
  const int64_t *pp_first;       // point tables: [n_group+1] instance range of each group
  const int32_t *pp_slot;        // point tables: [n] shared-memory slot (node*G + cell) in its group
  const int32_t *pp_local;       // point tables, cell-window mode: [n] local node of the instance
  const int32_t *cls_cnt;        // distributed: [n_class] instances per cell
  const int32_t *cls_nodeoff;    // distributed: [n_class] offset into dist_nodes
  const int64_t *grp_instbase;   // distributed: [n_group] first instance of the group
};

struct GroupInfo {
  int32_t cls, ncell;
  int32_t cell_base;   // first permuted cell index of the group
  int32_t pad;
  int64_t node_base;   // unused (kept for layout stability)
  int64_t ab_base;     // first slot of the group's schedule-ordered node arrays ((rounds+1)*32)
};

struct ClassInfo {
  int32_t n, G, lgG, rounds;
  int32_t sched_off, needs_ica, nodeoff_off, pad1;
};

// ---- interleaved ("tape") groups: 32 same-shape cells, one lane per cell (cn_tape.cuh) ----------
struct TapeGroup {
  int64_t tape_base;     // first element of the group's tape (multiple of 32 doubles)
  int32_t cls, cell_base, ncell, pad0;
  int64_t pp_base;       // window mode: first element of the group's rows in a step's block of win_rows
};

struct TapeClass {
  int32_t n, prog_off, prog_len, n_bar;  // n_bar: signal mbarriers the class's program uses
};

// the part of a class's program that one warp runs: forward records [p0, p1), backward records
// [b0, b1) and its segment of the group's tape, which is cut into chunks of whole records (at
// most tape_CH rows each); head holds the row counts of the first four chunks (8 bits each),
// which are requested before the program starts
struct TapeTask {
  int32_t p0, p1, b0, b1;
  int32_t nchunk, tm_base;  // tm_base: first tensor-memory slot of the warp
  uint32_t row0, head;
  uint32_t nrows, pp0;      // rows of the segment; ordinal of the warp's first point-process node
};

// Program record (uint4) of the interleaved kernel: one per run of plain chain nodes (RUN), per
// other node elimination (ELIM), per node with distributed mechanisms (MECH), per chunk of the
// warp's tape segment (CHUNK) and per cross-warp dependency (WAIT).
//   RUN   x = ring byte offset of the first node's record (16) | nodes in the run (8) | first
//             node takes a contribution in registers (bit 24) | backward: v of the run's parent
//             comes from the parent's system row, z bits 21..30 (bit 25)
//         y = RT_RUN | backward: wait for mbarrier bits 16..23 first (bit 24) | forward: the run's
//             last node is the top of its chain (bit 26) and stores /
//             adds (bit 27) its contribution to its parent's system row (bits 16..25)
//         z = system row of the first node (10), or, with bit 20 set, its slot in the warp's share
//             of tensor memory     w = first tape row of the first node's record (16) | forward,
//             chain top: it arrives on mbarrier bits 16..23 (bit 24)
//   ELIM  x = ring byte offset (16) | forward: wait for mbarrier bits 16..23 first (bit 24)
//         y = flags (16) | forward: mbarrier the record arrives on (RF_SIG_F); backward copy:
//             mbarrier to wait for (RF_WAIT_B); the backward copy arrives on mbarrier x (RF_SIG_B)
//         z = own system row (10) | parent's system row (10)
//         w = first tape row of the record (16) | tape row of the v copy in the node's mechanism
//             record (16)
//   MECH  x = ring byte offset (16)
//         y = flags (16) | first tape row of the record (16)
//         z = system row of the node (10) | mbarrier the record arrives on (16, RF_SIG_F)
//         w = mask of the distributed tables on the node
//   CHUNK the records that follow sit in the next chunk: the stage of the chunk before it is free
//         x = first row (relative to the warp's segment) of the chunk to request into that stage
//             (16) | its rows (8; 0: nothing left to request)
//         y = RT_CHUNK   z = stage to fill (16) | stage to wait for (16)
//   WAIT  y = RT_WAIT    z = mbarrier to wait for
enum { RK_ROOT = 0, RK_FWD = 1, RK_STORE = 2, RK_ADD = 3, RK_KIND = 3,
       RF_FWD_IN = 4,     // the previous record of this warp handed its contribution in registers
       RF_HAS_ACC = 8,    // contributions (mechanisms, children) wait in the node's own system row
       RF_HAS_PP = 16,    // two dynamic rows (conductance, current of point processes)
       RF_MECHV = 32,     // the node has a mechanism record: v is also stored to its v copy
       RF_SIG_F = 64,     // publish this warp's position after the record, forward / backward
       RF_SIG_B = 128,
       RF_WAIT_B = 256,   // backward: wait for the parent's warp first
       RF_TMEM = 512,     // the node's own row is a tensor-memory slot of the warp (z, low 10 bits)
       RF_BW_ROW = 1024,  // backward: v of the parent comes from the parent's row, not a register
       RM_HAS_CAI = 1, RM_NEED_ICA = 2,
       RT_ELIM = 0, RT_MECH = 1 << 13, RT_WAIT = 2 << 13, RT_RUN = 3 << 13, RT_CHUNK = 4 << 13,
       RT_MASK = 7 << 13 };

// cell-window mode (cn_cell.cuh): where the copies of a class's mechanism tables sit in the CTA's
// shared memory (doubles from the start of the mechanism block), and the size of the whole block
struct CellClass {
  int32_t mech_off[CN_MAX_TABLES];  // doubles from the start of the mechanism block
  int32_t dist_off[CN_MAX_TABLES];  // first entry of the table's node positions in the plan's dist list
  int32_t mech_doubles;
  // Elimination plan (cn_finalize.hpp build_cell_plan).  Every per-node array in shared memory is
  // in PLAN ORDER: the nodes of a chain side by side in elimination order, chains sorted by level,
  // the root last.  plan_noff[noff_off + p] = where node p lives in the schedule-ordered arrays
  // in HBM.  Segments [seg_off, seg_off + n_seg); lvl[lvl_off + L] = first segment of level L
  // (n_lev + 1 entries, relative); child positions from child_off (n_child entries, the root's
  // children last: root_child_off relative to child_off); dist positions from dist_base (n_dist).
  int32_t seg_off, n_seg, n_lev, lvl_off, child_off, n_child, root_child_off, root_nchild;
  int32_t noff_off, dist_base, n_dist, pad;
};

// one unbranched chain of a cell in plan order: nodes first .. first + len - 1 (distal to
// proximal), the positions of the children of its first node (each the last node of an earlier
// chain; child_off relative to the class's child list), and the position of the parent of its
// last node
struct CellSeg {
  uint16_t first, len, nchild, par;
  uint32_t child_off, pad;
};

struct DModel {
  int32_t n_group, n_class, n_table, warp_smem_doubles;
  int32_t n_tgroup, tape_prog_cap, tape_sys_cap, tape_W;
  int32_t tape_pf, pad_pf;      // rows a warp's L2 prefetch runs ahead of its ring
  int32_t tape_S, tape_CH, tape_pbuf, tape_bar_cap;  // ring of a warp: S stages of CH rows; program buffers
  const TapeGroup *tgrp;
  const TapeClass *tcls;
  const TapeTask *ttask;        // [n_class][tape_W]
  const uint4 *prog;
  double *tape;                 // == v + n_ab: one arena, so node positions index both
  const GroupInfo *grp;
  const ClassInfo *cls;
  const uint32_t *sched;        // per class: rounds * P entries, node | parent << 16
  const int32_t *dist_nodes;    // local node lists of distributed tables per class
  const int32_t *node_off;      // per class: slot offset (round*32 + p*G) of every local node
  double *v;                    // [n_slot] schedule order, padded
  const double *dstat, *rstat;  // static diagonal / rhs parts (row-normalised), schedule order
  double *ppdr;                 // point-process conductance / current of this dt, schedule order,
                                // rows of 32 + 32 doubles: slot s -> (s/32)*64 + s%32 (+32: current)
  const double *a_s, *b_s;      // off-diagonals, schedule order
  double *cai;                  // per node (only when a table needs it) else null
  const double *thr;            // [n_pcell]
  unsigned char *flag;          // [n_pcell]
  const int32_t *gid_of_pcell;  // [n_pcell]
  // spikes
  int32_t *sp_gid;
  int64_t *sp_step;
  unsigned long long *n_sp;
  int64_t sp_cap;
  int32_t *overflow;
  // delivery
  int64_t *sp_end;              // ring [wr]: number of spikes with step <= s
  int32_t wr, mind, maxd, pad2;
  const int64_t *src_first;     // [n_src+1] netcons by source gid, sorted by delay steps
  const int32_t *nc_d;          // delay in steps
  const int32_t *nc_tab;
  const int64_t *nc_inst;       // permuted instance
  const double *nc_w;
  int64_t n_stim;
  const int32_t *stim_gid;      // sorted by step
  const int64_t *stim_step;
  // window mode (interleaved kernel only): one launch integrates up to `mind` steps
  double *win_rows;             // [steps][win_stride]: point-process conductance / current rows
  double *win_deliv;            // [steps][win_ninst]: summed weights delivered to every instance
  unsigned long long *win_mask; // [win_ninst] window mode of the interleaved kernel: bit s = an event
                                // reaches the instance at step s of the window (deliveries are
                                // sparse: pp_window_kernel reads win_deliv only where a bit is set)
  int64_t win_stride, win_ninst;
  int32_t *win_done;            // [n_tgroup]: steps of the window completed for the group
  uint32_t *win_ticket;         // next (step, group) work item
  int64_t win_mark_cap;         // length of the two rings below
  int64_t *win_mark_step;       // ring: first step of the recent windows
  int64_t *win_mark_nsp;        //            and the length of the spike list at their start
  // probes recorded by the interleaved kernel itself in window mode (null otherwise): per group
  // the probed nodes (element of the voltage arena) and their column of the trace
  const int32_t *wp_first;      // [n_tgroup + 1]
  const int64_t *wp_pos;
  const int32_t *wp_col;
  double *trace;                // [trace_cap][n_probe]
  int64_t trace_row0, trace_cap;  // row of the first step of this launch
  int32_t n_probe, pad3;
  int64_t *step_ctr;            // [0] step, [1] trace row that a replayed CUDA graph starts from
  const struct CellClass *ccls; // cell-window mode (cn_cell.cuh): shared-memory layout per class
  const struct CellSeg *cseg;   //   and elimination plan
  const uint16_t *cseg_child, *cdist;
  const int32_t *cseg_lvl, *cplan_noff;
  uint32_t *cwin_smctr;         // [256] per-SM arrival counter (which warp of a CTA solves)
  double q10, dt, celsius;
  double fxw_scale, fxw_inv;    // fixed-point scale of the per-step event-weight sums (window modes)
  DTable tab[CN_MAX_TABLES];
};

// ------------------------------------------------------------------------------------------
// mechanism arithmetic
// ------------------------------------------------------------------------------------------

// Reciprocal to ~1 ulp without the special-case handling of an IEEE division: MUFU.RCP64H seed
// plus two Newton steps.  Every argument here is a positive, finite, O(1)..O(1e3) quantity
// (pivots of a diagonally dominant row-normalised matrix, sums of rate constants).
__device__ __forceinline__ double rcp_fast(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);
}

// The same with ONE correction step of third order (r (1 + e + e^2), e = 1 - x r): three dependent
// fp64 operations behind the MUFU instead of four, relative error ~ e^3 (< 1e-17 from the ~2e-6
// seed).  Used where the reciprocal sits on the dependent chain of an elimination.
__device__ __forceinline__ double rcp_chain(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);
  const double t = fma(e, e, e);
  return fma(r, t, r);
}

// Sums that several threads add to in no fixed order -- conductance / current of the point
// processes of a node, weights of the events that reach a synapse in one step -- are accumulated
// as 64-bit FIXED-POINT integers (resolution 2^-44 = 5.7e-14 of the row-normalised unit, range
// +-2^19): integer addition is associative, so the sum does not depend on the order in which the
// atomics land and a run is bit-reproducible (SURVEY.md 7 "accumulation of point-process
// currents"; PAPER.md L196 contention).  The slot is a double-sized word holding the integer; an
// addend beyond +-2^18 raises the overflow flag (cn_sync: CN_ERR_OVERFLOW).
#define CN_FX 17592186044416.0            // 2^44
#define CN_FX_INV 5.684341886080802e-14   // 2^-44
__device__ __forceinline__ void fx_add(double *slot, double val, int32_t *overflow) {
  if (!(fabs(val) < 262144.0)) *overflow = 2;
  const long long q = __double2ll_rn(val * CN_FX);
  if (q != 0)  // (an addend that rounds to 0 -- a current towards a reversal potential of 0 mV, a
               // synapse that has decayed below the resolution -- costs no atomic)
    atomicAdd(reinterpret_cast<unsigned long long *>(slot), (unsigned long long)q);
}
__device__ __forceinline__ double fx_get(double raw) {
  return (double)__double_as_longlong(raw) * CN_FX_INV;
}
__device__ __forceinline__ bool fx_nonzero(double raw) { return __double_as_longlong(raw) != 0; }
// The same for the event weights that reach a synapse in one step (window modes), with a scale the
// host derives from the model: the largest sum of |weights| that can meet on one synapse fits 62
// bits, so the sum cannot overflow and keeps every bit a double could hold for such weights.
__device__ __forceinline__ void fxw_add(double *slot, double w, double scale) {
  atomicAdd(reinterpret_cast<unsigned long long *>(slot), (unsigned long long)__double2ll_rn(w * scale));
}
__device__ __forceinline__ double fxw_get(double raw, double inv) {
  return (double)__double_as_longlong(raw) * inv;
}

// exp(x) for |x| < 700 to ~1 ulp without the special-case handling of the library routine:
// x = n ln2 + r with |r| <= ln2/2 (two-part ln2), Taylor polynomial of degree 13 (truncation
// 4e-18), scaling by 2^n through the exponent field.  Every argument here is a bounded rate
// exponent (|x| < 50 for |v| < 500 mV).
__device__ __forceinline__ double exp_lean(double x) {
  const double t = fma(x, 1.4426950408889634, 6755399441055744.0);  // round to nearest integer
  const double nf = t - 6755399441055744.0;
  double r = fma(nf, -6.93147180369123816490e-01, x);
  r = fma(nf, -1.90821492927058770002e-10, r);
  double p = 1.6059043836821613e-10;            // 1/13!
  p = fma(p, r, 2.08767569878681e-09);          // 1/12!
  p = fma(p, r, 2.505210838544172e-08);         // 1/11!
  p = fma(p, r, 2.755731922398589e-07);         // 1/10!
  p = fma(p, r, 2.7557319223985893e-06);        // 1/9!
  p = fma(p, r, 2.48015873015873e-05);          // 1/8!
  p = fma(p, r, 1.984126984126984e-04);         // 1/7!
  p = fma(p, r, 1.3888888888888889e-03);        // 1/6!
  p = fma(p, r, 8.333333333333333e-03);         // 1/5!
  p = fma(p, r, 4.1666666666666664e-02);        // 1/4!
  p = fma(p, r, 1.6666666666666666e-01);        // 1/3!
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);
  const int n = __double2loint(t);
  return p * __hiloint2double((n + 1023) << 20, 0);
}

// N independent exponentials in lockstep: the same operations per value as exp_lean (bit-identical
// results), written side by side so that the N Horner chains fill each other's DFMA latency
// (one chain alone issues one DFMA per ~8 cycles; the compiler keeps separately inlined
// exp_lean calls one after the other).
template <int N>
__device__ __forceinline__ void exp_lean_n(const double (&x)[N], double (&y)[N]) {
  double t[N], r[N], p[N];
#pragma unroll
  for (int i = 0; i < N; ++i) t[i] = fma(x[i], 1.4426950408889634, 6755399441055744.0);
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const double nf = t[i] - 6755399441055744.0;
    r[i] = fma(nf, -6.93147180369123816490e-01, x[i]);
    r[i] = fma(nf, -1.90821492927058770002e-10, r[i]);
  }
  constexpr double c[13] = {2.08767569878681e-09,   2.505210838544172e-08,  2.755731922398589e-07,
                            2.7557319223985893e-06, 2.48015873015873e-05,   1.984126984126984e-04,
                            1.3888888888888889e-03, 8.333333333333333e-03,  4.1666666666666664e-02,
                            1.6666666666666666e-01, 0.5,                    1.0,
                            1.0};
#pragma unroll
  for (int i = 0; i < N; ++i) p[i] = 1.6059043836821613e-10;  // 1/13!
#pragma unroll
  for (int k = 0; k < 13; ++k) {
#pragma unroll
    for (int i = 0; i < N; ++i) p[i] = fma(p[i], r[i], c[k]);
  }
#pragma unroll
  for (int i = 0; i < N; ++i)
    y[i] = p[i] * __hiloint2double((__double2loint(t[i]) + 1023) << 20, 0);
}

__device__ __forceinline__ double cnexp(double y, double yinf, double tau, double dt) {
  return y + (1.0 - exp_lean(-dt * rcp_fast(tau))) * (yinf - y);
}

// cnexp towards 0 with the factor c = 1 - exp(-dt/tau) precomputed by the host (per instance for
// ExpSyn / Exp2Syn, per table for AMPA+NMDA): the same expression as cnexp(y, 0, tau, dt)
__device__ __forceinline__ double decay(double y, double c) { return y + c * (0.0 - y); }

// HH gates advanced over dt with cnexp at the new v: y += (1 - exp(-dt*q10*(a+b))) * (a/(a+b) - y).
// The textbook rate functions + cnexp; divisions by constants are multiplications by their
// reciprocals, 1/tau is never formed, and the three exponentials in v/10 share one evaluation
// (exp(-(v+40)/10) = exp(-(v+35)/10) e^-0.5, exp(-(v+55)/10) = exp(-(v+35)/10) e^-2): differences
// of a few ulp in the rates.
// LOCKSTEP: the four exponentials of the rates and the three of the updates are evaluated side by
// side (exp_lean_n: same operations, same bits, 3-4 Horner chains in flight) -- config 2 13.96 ->
// 13.40 us per dt on the on-chip kernel; the interleaved kernel keeps the one-after-the-other form
// (at its 128-register limit the lockstep form costs more than it saves: 112.9 -> 115.7 us).
template <bool LOCKSTEP>
__device__ __forceinline__ void hh_advance(double v, double q10dt, double &m, double &h,
                                           double &n) {
  if constexpr (!LOCKSTEP) {
    const double x65 = v + 65.0;
    const double e10 = exp_lean(-(v + 35.0) * 0.1);
    double al, be, s, u;
    // m: alpha = 0.1 vtrap(-(v+40), 10) with vtrap(x, y) = x / (exp(x/y) - 1); removable
    // singularity: y (1 - x/(2y)) for |x/y| < 1e-6
    u = -(v + 40.0) * 0.1;
    al = fabs(u) < 1e-6 ? 1.0 - 0.5 * u : u * rcp_fast(e10 * 0.60653065971263342 - 1.0);
    be = 4.0 * exp_lean(x65 * (-1.0 / 18.0));
    s = al + be;
    m += (1.0 - exp_lean(-q10dt * s)) * (al * rcp_fast(s) - m);
    // h
    al = 0.07 * exp_lean(x65 * -0.05);
    be = rcp_fast(e10 + 1.0);
    s = al + be;
    h += (1.0 - exp_lean(-q10dt * s)) * (al * rcp_fast(s) - h);
    // n: alpha = 0.01 vtrap(-(v+55), 10)
    u = -(v + 55.0) * 0.1;
    al = fabs(u) < 1e-6 ? 0.1 * (1.0 - 0.5 * u) : 0.1 * u * rcp_fast(e10 * 0.1353352832366127 - 1.0);
    be = 0.125 * exp_lean(x65 * -0.0125);
    s = al + be;
    n += (1.0 - exp_lean(-q10dt * s)) * (al * rcp_fast(s) - n);
  } else {
  const double x65 = v + 65.0;
  // the four exponentials of the rates, then the three of the updates, each set in lockstep
  const double xr[4] = {-(v + 35.0) * 0.1, x65 * (-1.0 / 18.0), x65 * -0.05, x65 * -0.0125};
  double er[4];
  exp_lean_n<4>(xr, er);
  const double e10 = er[0];
  // m: alpha = 0.1 vtrap(-(v+40), 10) with vtrap(x, y) = x / (exp(x/y) - 1); removable
  // singularity: y (1 - x/(2y)) for |x/y| < 1e-6
  double u = -(v + 40.0) * 0.1;
  const double al_m = fabs(u) < 1e-6 ? 1.0 - 0.5 * u : u * rcp_fast(e10 * 0.60653065971263342 - 1.0);
  const double s_m = al_m + 4.0 * er[1];
  // h
  const double al_h = 0.07 * er[2];
  const double s_h = al_h + rcp_fast(e10 + 1.0);
  // n: alpha = 0.01 vtrap(-(v+55), 10)
  u = -(v + 55.0) * 0.1;
  const double al_n =
      fabs(u) < 1e-6 ? 0.1 * (1.0 - 0.5 * u) : 0.1 * u * rcp_fast(e10 * 0.1353352832366127 - 1.0);
  const double s_n = al_n + 0.125 * er[3];
  const double xu[3] = {-q10dt * s_m, -q10dt * s_h, -q10dt * s_n};
  double eu[3];
  exp_lean_n<3>(xu, eu);
  m += (1.0 - eu[0]) * (al_m * rcp_fast(s_m) - m);
  h += (1.0 - eu[1]) * (al_h * rcp_fast(s_h) - h);
  n += (1.0 - eu[2]) * (al_n * rcp_fast(s_n) - n);
  }
}

__device__ __forceinline__ void hhform_gate(double v, const double *g6, double &xinf,
                                            double &xtau) {
  // (k may be negative: rcp_fast handles either sign; every argument is finite and non-zero)
  const double u = (v - g6[4]) * rcp_fast(g6[5]);
  xinf = rcp_fast(1.0 + exp_lean((g6[0] - v) * rcp_fast(g6[1])));
  const double eu = exp_lean(u);
  xtau = g6[2] + g6[3] * rcp_fast(eu + rcp_fast(eu));
}

__device__ __forceinline__ double ipow(double x, int p) {
  double r = 1.0;
  for (int j = 0; j < p; ++j) r *= x;
  return r;
}

__device__ __forceinline__ double mgblock(double v, double mg) {
  return rcp_fast(1.0 + exp_lean(-0.062 * v) * (mg * (1.0 / 3.57)));
}

// ------------------------------------------------------------------------------------------
// nrn_cur: conductance G (row-normalised) and G*E into the shared-memory system
// ------------------------------------------------------------------------------------------

// Where a group's node (shared-memory slot = node*G + cell) lives in the schedule-ordered arrays.
struct GroupView {
  int64_t ab;             // first slot of the group
  const int32_t *noff;    // class table: node -> round*32 + p*G
  int G, lgG;
  bool direct;            // per-node arrays are indexed by slot itself (cn_cell.cuh: arrays in
                          // shared memory, by local node)
  __device__ __forceinline__ int64_t gpos(int slot) const {
    return direct ? (int64_t)slot : ab + noff[slot >> lgG] + (slot & (G - 1));
  }
};

// Distributed table, lockstep over the group's cells: instance j = k*G + c sits on node
// nodes[k] of cell c.  At most one instance per node and table, so plain read-modify-write.
// par / st: the table's parameter and state arrays (T.param / T.state in HBM, or their copies in
// shared memory); the `stride` threads lane, lane + stride, ... share the instances.
template <class NodeT>
__device__ __forceinline__ void cur_distributed(const DTable &T, double *const *par,
                                                double *const *st, int64_t ib, int cnt,
                                                const GroupView &gv, const NodeT *nodes,
                                                double *D, double *R, double *I,
                                                const double *v_g, int lane, int stride = 32) {
  const int G = gv.G, lgG = gv.lgG;
  const int tot = cnt << lgG;
  switch (T.type) {
    case T_HH: {
      const double ena = T.glob[0], ek = T.glob[1];
      for (int j = lane; j < tot; j += stride) {
        const int64_t q = ib + j;
        const int slot = ((int)nodes[j >> lgG] << lgG) + (j & (G - 1));
        const double m = st[0][q], h = st[1][q], n = st[2][q];
        const double invc = par[4][q];
        const double gna = par[0][q] * m * m * m * h;
        const double n2 = n * n;
        const double gk = par[1][q] * n2 * n2;
        const double gl = par[2][q];
        D[slot] += (gna + gk + gl) * invc;
        R[slot] += (gna * ena + gk * ek + gl * par[3][q]) * invc;
      }
      break;
    }
    case T_HHFORM: {
      const int p = (int)T.glob[0], qq = (int)T.glob[1];
      const double E = T.glob[2];
      const bool to_ica = T.glob[3] != 0.0;
      // four instances per lane and pass with every load issued before the first use (clamped
      // indices, no branches around the loads): when parameters and states stream from HBM the
      // loop is bound by the latency of these loads (config 5)
      for (int j0 = lane; j0 < tot; j0 += 4 * stride) {
        double gb[4], sm[4], sh[4], ic[4];
        int sl[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int j = min(j0 + u * stride, tot - 1);
          const int64_t q = ib + j;
          gb[u] = par[0][q];
          sm[u] = st[0][q];
          sh[u] = st[1][q];
          ic[u] = par[1][q];
          sl[u] = ((int)nodes[j >> lgG] << lgG) + (j & (G - 1));
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          if (j0 + u * stride < tot) {
            const int slot = sl[u];
            const double g = gb[u] * ipow(sm[u], p) * ipow(sh[u], qq);
            D[slot] += g * ic[u];
            R[slot] += g * E * ic[u];
            if (to_ica) I[slot] += g * (v_g[gv.gpos(slot)] - E);  // ica uses v_old (still in HBM)
          }
        }
      }
      break;
    }
    case T_SK: {
      const double E = T.glob[0];
      for (int j = lane; j < tot; j += stride) {
        const int64_t q = ib + j;
        const int slot = ((int)nodes[j >> lgG] << lgG) + (j & (G - 1));
        const double g = par[0][q] * st[0][q];
        const double invc = par[1][q];
        D[slot] += g * invc;
        R[slot] += g * E * invc;
      }
      break;
    }
    default: break;  // PAS is folded into dstat/rstat; CADYN carries no current
  }
}

// ------------------------------------------------------------------------------------------
// nrn_state with the new v (in R)
// ------------------------------------------------------------------------------------------

template <class NodeT>
__device__ __forceinline__ void state_distributed(const DTable &T, double *const *par,
                                                  double *const *st, int64_t ib, int cnt,
                                                  const GroupView &gv, const NodeT *nodes,
                                                  const double *R, double *cai_g,
                                                  const double *I, int lane, double dt,
                                                  double q10, int stride = 32) {
  (void)par;
  const int G = gv.G, lgG = gv.lgG;
  const int tot = cnt << lgG;
  switch (T.type) {
    case T_HH:
      for (int j = lane; j < tot; j += stride) {
        const int64_t q = ib + j;
        const int slot = ((int)nodes[j >> lgG] << lgG) + (j & (G - 1));
        double sm = st[0][q], sh = st[1][q], sn = st[2][q];
        hh_advance<true>(R[slot], q10 * dt, sm, sh, sn);
        st[0][q] = sm;
        st[1][q] = sh;
        st[2][q] = sn;
      }
      break;
    case T_HHFORM: {
      const int p = (int)T.glob[0], qq = (int)T.glob[1];
      for (int j0 = lane; j0 < tot; j0 += 4 * stride) {  // (four instances per pass: loads first)
        double sm[4], sh[4], vv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int j = min(j0 + u * stride, tot - 1);
          const int64_t q = ib + j;
          sm[u] = st[0][q];
          sh[u] = st[1][q];
          vv[u] = R[((int)nodes[j >> lgG] << lgG) + (j & (G - 1))];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int j = j0 + u * stride;
          if (j < tot) {
            const int64_t q = ib + j;
            double xinf, xtau;
            if (p > 0) {
              hhform_gate(vv[u], T.glob + 4, xinf, xtau);
              st[0][q] = cnexp(sm[u], xinf, xtau, dt);
            }
            if (qq > 0) {
              hhform_gate(vv[u], T.glob + 10, xinf, xtau);
              st[1][q] = cnexp(sh[u], xinf, xtau, dt);
            }
          }
        }
      }
      break;
    }
    case T_SK:
      for (int j = lane; j < tot; j += stride) {
        const int64_t q = ib + j;
        const int slot = ((int)nodes[j >> lgG] << lgG) + (j & (G - 1));
        double cai = cai_g[gv.gpos(slot)];
        if (cai < 1e-9) cai = 1e-9;
        const double zinf = 1.0 / (1.0 + pow(T.glob[1] / cai, T.glob[2]));
        st[0][q] = cnexp(st[0][q], zinf, T.glob[3], dt);
      }
      break;
    case T_CADYN: {
      // derivimplicit on a linear ODE: one Newton step of backward Euler is exact (L278)
      const double kappa = 1e4 * T.glob[0] / (2.0 * 96485.33212 * T.glob[1]);
      const double taud = T.glob[2], cmin = T.glob[3];
      for (int j = lane; j < tot; j += stride) {
        const int slot = ((int)nodes[j >> lgG] << lgG) + (j & (G - 1));
        const int64_t gp = gv.gpos(slot);
        const double y0 = cai_g[gp];
        cai_g[gp] = (y0 + dt * (-kappa * I[slot] + cmin / taud)) / (1.0 + dt / taud);
      }
      break;
    }
    default: break;
  }
}

// ------------------------------------------------------------------------------------------
// the step kernel: one warp per group
// ------------------------------------------------------------------------------------------

#define CN_PF 4  // rounds of prefetch distance for the schedule-ordered streams

template <int WPB>
// (registers: the prefetched streams must stay in registers -- a spill store waits for its load
// and the prefetch distance is gone -- so the bound asks for 12 warps per SM, not 16)
__global__ void __launch_bounds__(WPB * 32, WPB >= 8 ? 1 : 12 / WPB)
    step_kernel(const __grid_constant__ DModel M,
                                                        int64_t k) {
  extern __shared__ double smem[];
  if (k < 0) k = M.step_ctr[0] - k - 1;  // replayed graph: the device counter + offset
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = blockIdx.x * WPB + warp;
  if (g >= M.n_group) return;
  const GroupInfo gi = M.grp[g];
  const ClassInfo ci = M.cls[gi.cls];
  const int n = ci.n, G = ci.G, lgG = ci.lgG;
  const int nG = n << lgG;
  double *D = smem + (size_t)warp * M.warp_smem_doubles;
  double *R = D + nG;
  double *I = R + nG;  // only valid when ci.needs_ica
  const int64_t ab = gi.ab_base;
  const double dt = M.dt;
  const int c = lane & (G - 1), p = lane >> lgG;
  const int P = 32 >> lgG;
  const int rounds = ci.rounds;
  GroupView gv;
  gv.ab = ab;
  gv.noff = M.node_off + ci.nodeoff_off;
  gv.G = G;
  gv.lgG = lgG;
  gv.direct = false;

  // schedule-ordered streams of this lane: slot (round r, lane) = ab + r*32 + lane
  const uint32_t *__restrict__ sched = M.sched + ci.sched_off + p;
  const double *__restrict__ as = M.a_s + ab + lane;
  const double *__restrict__ bs = M.b_s + ab + lane;
  const double *__restrict__ dss = M.dstat + ab + lane;
  const double *__restrict__ rss = M.rstat + ab + lane;
  double *__restrict__ vs = M.v + ab + lane;
  double *__restrict__ pps = M.ppdr + 2 * ab + lane;  // point processes: pp_coop_kernel put the
  const bool has_pp = M.ppdr != nullptr;              // conductance / current of this dt here
  // (a node that carries point processes is marked by a NEGATIVE static diagonal, which is > 0).
  // Their conductance / current rows are requested together with the node's other streams and
  // looked at only when the round is worked on: nothing here may depend on a load just issued,
  // or the prefetch distance is lost (one L2 round trip per round).
  auto take_pp = [&](int r, double &d, double &rr, double pd, double pr) {
    if (!has_pp || d > 0.0) return;
    d = -d;
    if (fx_nonzero(pd) || fx_nonzero(pr)) {
      d += fx_get(pd);
      rr += fx_get(pr);
      pps[(size_t)r * 64] = 0.0;
      pps[(size_t)r * 64 + 32] = 0.0;
    }
  };

  // issue the first CN_PF rounds of loads and the root's terms before anything else
  uint32_t e_[CN_PF];
  double a_[CN_PF], b_[CN_PF], d_[CN_PF], r_[CN_PF], v_[CN_PF], pd_[CN_PF], pr_[CN_PF];
#pragma unroll
  for (int u = 0; u < CN_PF; ++u) {
    e_[u] = CN_IDLE;
    a_[u] = b_[u] = d_[u] = r_[u] = v_[u] = pd_[u] = pr_[u] = 0.0;
    if (u < rounds) {
      e_[u] = sched[u * P];
      a_[u] = as[(size_t)u * 32];
      b_[u] = bs[(size_t)u * 32];
      d_[u] = dss[(size_t)u * 32];
      r_[u] = rss[(size_t)u * 32];
      v_[u] = vs[(size_t)u * 32];
      if (has_pp) {
        pd_[u] = pps[(size_t)u * 64];
        pr_[u] = pps[(size_t)u * 64 + 32];
      }
    }
  }
  double d_root = 1.0, r_root = 0.0, pd_root = 0.0, pr_root = 0.0;
  if (p == 0) {
    d_root = dss[(size_t)rounds * 32];
    r_root = vs[(size_t)rounds * 32] + rss[(size_t)rounds * 32];
    if (has_pp) {
      pd_root = pps[(size_t)rounds * 64];
      pr_root = pps[(size_t)rounds * 64 + 32];
    }
  }

  // ---- zero the system -------------------------------------------------------------------
  for (int j = lane; j < nG; j += 32) {
    D[j] = 0.0;
    R[j] = 0.0;
  }
  if (ci.needs_ica)
    for (int j = lane; j < nG; j += 32) I[j] = 0.0;
  __syncwarp();

  // ---- nrn_cur -------------------------------------------------------------------------
  for (int t = 0; t < M.n_table; ++t) {
    const DTable &T = M.tab[t];
    if (!T.is_point) {  // (point processes: pp_coop_kernel, one thread per instance)
      const int cnt = T.cls_cnt[gi.cls];
      if (cnt > 0) {
        cur_distributed(T, T.param, T.state, T.grp_instbase[g], cnt, gv, M.dist_nodes + T.cls_nodeoff[gi.cls], D,
                        R, I, M.v, lane);
        __syncwarp();
      }
    }
  }

  // ---- Hines triangularisation: rounds of P independent nodes per cell -------------------
  for (int r0 = 0; r0 < rounds; r0 += CN_PF) {
#pragma unroll
    for (int u = 0; u < CN_PF; ++u) {
      const int r = r0 + u;
      if (r < rounds) {
        const uint32_t e = e_[u];
        if ((e & 0xFFFFu) != CN_IDLE) {
          const int si = ((e & 0xFFFFu) << lgG) + c, sp = ((e >> 16) << lgG) + c;
          double ds = d_[u], rs = v_[u] + r_[u];
          take_pp(r, ds, rs, pd_[u], pr_[u]);
          const double di = D[si] + ds, ri = R[si] + rs;
          const double rinv = rcp_fast(di);  // (pivots of a diagonally dominant matrix: > 0, O(1))
          const double f = a_[u] * rinv;
          D[sp] -= f * b_[u];
          R[sp] -= f * ri;
          D[si] = b_[u] * rinv;   // back-substitution multiplier
          R[si] = ri * rinv;
        }
        __syncwarp();
        const int rn = r + CN_PF;  // refill this ring slot
        e_[u] = CN_IDLE;
        if (rn < rounds) {  // (idle slots hold benign padding: loaded like any other)
          e_[u] = sched[rn * P];
          a_[u] = as[(size_t)rn * 32];
          b_[u] = bs[(size_t)rn * 32];
          d_[u] = dss[(size_t)rn * 32];
          r_[u] = rss[(size_t)rn * 32];
          v_[u] = vs[(size_t)rn * 32];
          if (has_pp) {
            pd_[u] = pps[(size_t)rn * 64];
            pr_[u] = pps[(size_t)rn * 64 + 32];
          }
        }
      }
    }
  }
  // root: local node 0, stored in the extra round
  if (p == 0) {
    take_pp(rounds, d_root, r_root, pd_root, pr_root);
    const double u0 = (R[c] + r_root) * rcp_fast(D[c] + d_root);
    R[c] = u0;
    vs[(size_t)rounds * 32] = u0;
  }
  __syncwarp();
  // ---- back-substitution, rounds in reverse; v_new is stored in schedule order ---------------
  {
    uint32_t en = rounds > 0 ? sched[(rounds - 1) * P] : CN_IDLE;
    for (int r = rounds - 1; r >= 0; --r) {
      const uint32_t e = en;
      if (r > 0) en = sched[(r - 1) * P];
      if ((e & 0xFFFFu) != CN_IDLE) {
        const int si = ((e & 0xFFFFu) << lgG) + c, sp = ((e >> 16) << lgG) + c;
        const double u = R[si] - D[si] * R[sp];
        R[si] = u;
        vs[(size_t)r * 32] = u;
      }
      __syncwarp();
    }
  }

  // ---- nrn_state with the new v --------------------------------------------------------------
  for (int t = 0; t < M.n_table; ++t) {
    const DTable &T = M.tab[t];
    if (T.n_state == 0 && T.type != T_CADYN) continue;
    if (!T.is_point) {
      const int cnt = T.cls_cnt[gi.cls];
      if (cnt > 0) {
        state_distributed(T, T.param, T.state, T.grp_instbase[g], cnt, gv, M.dist_nodes + T.cls_nodeoff[gi.cls],
                          R, M.cai, I, lane, dt, M.q10);
        __syncwarp();
      }
    }
  }

  // ---- threshold detection on the roots (warp ballot, one atomic per warp) --------------------
  {
    bool fire = false;
    int pc = 0;
    if (p == 0 && c < gi.ncell) {
      pc = gi.cell_base + c;
      const bool above = R[c] > M.thr[pc];
      fire = above && !M.flag[pc];
      M.flag[pc] = (unsigned char)above;
    }
    const unsigned ball = __ballot_sync(0xffffffffu, fire);
    if (ball) {
      unsigned long long base = 0;
      const int leader = __ffs(ball) - 1;
      if (lane == leader) base = atomicAdd(M.n_sp, (unsigned long long)__popc(ball));
      base = __shfl_sync(0xffffffffu, base, leader);
      if (fire) {
        const unsigned long long pos = base + __popc(ball & ((1u << lane) - 1u));
        if ((int64_t)pos < M.sp_cap) {
          M.sp_gid[pos] = M.gid_of_pcell[pc];
          M.sp_step[pos] = k + 1;
        } else {
          *M.overflow = 1;
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// event delivery for step k (L64): every spike (gid, s) with a NetCon of delay k - s
// ------------------------------------------------------------------------------------------

__device__ __forceinline__ void receive(const DModel &M, int64_t nc) {
  const DTable &T = M.tab[M.nc_tab[nc]];
  const int64_t q = M.nc_inst[nc];
  const double w = M.nc_w[nc];
  switch (T.type) {
    case T_EXPSYN: atomicAdd(&T.state[0][q], w); break;
    case T_EXP2SYN: {
      const double wf = w * T.param[4][q];  // param[4] = peak-normalisation factor
      atomicAdd(&T.state[0][q], wf);
      atomicAdd(&T.state[1][q], wf);
      break;
    }
    case T_AMPANMDA: {
      const double wa = w * T.glob[7], wn = w * T.glob[8];  // factors appended by the host
      atomicAdd(&T.state[0][q], wa);
      atomicAdd(&T.state[1][q], wa);
      atomicAdd(&T.state[2][q], wn);
      atomicAdd(&T.state[3][q], wn);
      break;
    }
    default: break;
  }
}

__device__ __forceinline__ void deliver_source(const DModel &M, int32_t gid, int32_t d,
                                               int lane) {
  int64_t lo = M.src_first[gid], hi = M.src_first[gid + 1];
  if (lo >= hi) return;
  // lower / upper bound of delay d in the delay-sorted NetCon list of this source
  int64_t a = lo, b = hi;
  while (a < b) {
    const int64_t mid = (a + b) >> 1;
    if (M.nc_d[mid] < d) a = mid + 1; else b = mid;
  }
  const int64_t first = a;
  b = hi;
  while (a < b) {
    const int64_t mid = (a + b) >> 1;
    if (M.nc_d[mid] <= d) a = mid + 1; else b = mid;
  }
  for (int64_t nc = first + lane; nc < a; nc += 32) receive(M, nc);
}

__global__ void __launch_bounds__(128) deliver_kernel(const __grid_constant__ DModel M,
                                                      int64_t k) {
  if (k < 0) k = M.step_ctr[0] - k - 1;  // replayed graph: the device counter + offset
  const int lane = threadIdx.x & 31;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarp = ((int64_t)gridDim.x * blockDim.x) >> 5;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    unsigned long long ns = *M.n_sp;
    if ((int64_t)ns > M.sp_cap) ns = (unsigned long long)M.sp_cap;
    M.sp_end[k % M.wr] = (int64_t)ns;  // all spikes with step <= k are recorded by now
  }
  const int64_t s_lo = k - M.maxd, s_hi = k - M.mind;  // spike steps that may deliver now
  if (s_hi < 0) return;
  const int64_t i_lo = (s_lo - 1 >= 0) ? M.sp_end[(s_lo - 1) % M.wr] : 0;
  const int64_t i_hi = M.sp_end[s_hi % M.wr];
  for (int64_t i = i_lo + warp; i < i_hi; i += nwarp)
    deliver_source(M, M.sp_gid[i], (int32_t)(k - M.sp_step[i]), lane);
  if (M.n_stim > 0) {
    int64_t a = 0, b = M.n_stim;
    while (a < b) {
      const int64_t mid = (a + b) >> 1;
      if (M.stim_step[mid] < s_lo) a = mid + 1; else b = mid;
    }
    for (int64_t i = a + warp; i < M.n_stim && M.stim_step[i] <= s_hi; i += nwarp)
      deliver_source(M, M.stim_gid[i], (int32_t)(k - M.stim_step[i]), lane);
  }
}

// ------------------------------------------------------------------------------------------
// window mode: everything the events and point processes contribute to the next `nsteps` steps
// (nsteps <= smallest delay, so every event delivered in the window stems from a spike recorded
// before it).  deliver_window_kernel sums the weights per (step, instance); pp_window_kernel then
// advances every point process through the window and leaves its conductance / current of every
// step in win_rows, where the interleaved kernel picks them up.  Same arithmetic per step as
// deliver_kernel + pp_step_kernel (types whose current depends on v cannot run in this mode).
// ------------------------------------------------------------------------------------------

__global__ void __launch_bounds__(128) deliver_window_kernel(const __grid_constant__ DModel M,
                                                             int64_t k0, int nsteps, int64_t widx) {
  const int lane = threadIdx.x & 31;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarp = ((int64_t)gridDim.x * blockDim.x) >> 5;
  unsigned long long ns = *M.n_sp;
  if ((int64_t)ns > M.sp_cap) ns = (unsigned long long)M.sp_cap;
  // spikes that can matter carry steps >= k0 - maxd: they were recorded in the windows that end
  // at or after that step (the spike list is ordered by window, not by step)
  int64_t i_lo = (int64_t)ns;
  int64_t end_step = k0;  // first step after window j
  // (the ring of window marks holds maxd + 64 windows: enough even if every window is one step)
  for (int64_t j = widx - 1; j >= 0 && j > widx - M.win_mark_cap + 1; --j) {
    if (end_step < k0 - M.maxd) break;
    i_lo = M.win_mark_nsp[j % M.win_mark_cap];
    end_step = M.win_mark_step[j % M.win_mark_cap];
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    M.win_mark_step[widx % M.win_mark_cap] = k0;
    M.win_mark_nsp[widx % M.win_mark_cap] = (int64_t)ns;
  }
  auto deliver = [&](int32_t gid, int64_t step) {
    const int64_t lo = M.src_first[gid], hi = M.src_first[gid + 1];
    // delays d with k0 <= step + d < k0 + nsteps, in the delay-sorted list of this source
    const int64_t d_lo = k0 - step, d_hi = k0 + nsteps - 1 - step;
    int64_t a = lo, b = hi;
    while (a < b) {
      const int64_t mid = (a + b) >> 1;
      if (M.nc_d[mid] < d_lo) a = mid + 1; else b = mid;
    }
    for (int64_t nc = a + lane; nc < hi; nc += 32) {
      const int64_t d = M.nc_d[nc];
      if (d > d_hi) break;
      const DTable &T = M.tab[M.nc_tab[nc]];
      fxw_add(&M.win_deliv[(step + d - k0) * M.win_ninst + T.pp_goff + M.nc_inst[nc]], M.nc_w[nc],
              M.fxw_scale);
      if (M.win_mask) atomicOr(&M.win_mask[T.pp_goff + M.nc_inst[nc]], 1ull << (step + d - k0));
    }
  };
  for (int64_t i = i_lo + warp; i < (int64_t)ns; i += nwarp) deliver(M.sp_gid[i], M.sp_step[i]);
  for (int64_t i = warp; i < M.n_stim; i += nwarp) {
    const int64_t st = M.stim_step[i];
    if (st + M.maxd >= k0 && st + M.mind < k0 + nsteps) deliver(M.stim_gid[i], st);
  }
}

__global__ void __launch_bounds__(256) pp_window_kernel(const __grid_constant__ DModel M,
                                                        int64_t k0, int nsteps) {
  const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t nth = (int64_t)gridDim.x * blockDim.x;
  const double dt = M.dt;
  for (int t = 0; t < M.n_table; ++t) {
    const DTable &T = M.tab[t];
    if (!T.is_point) continue;
    const uint32_t *__restrict__ ws = T.pp_wslot;
    for (int64_t q = tid; q < T.pp_tape_end; q += nth) {
      double *rows = M.win_rows + ws[q];
      double *dl = M.win_deliv + T.pp_goff + q;
      unsigned long long mask = 0;  // steps of the window at which an event reaches this instance
      if (T.type != T_ICLAMP) {
        mask = M.win_mask[T.pp_goff + q];
        if (mask) M.win_mask[T.pp_goff + q] = 0;
      }
      switch (T.type) {
        case T_EXPSYN: {
          double g = T.state[0][q];
          const double c0 = T.param[0][q], e = T.param[1][q], sc = T.param[2][q];
          for (int s = 0; s < nsteps; ++s, rows += M.win_stride, dl += M.win_ninst) {
            if (mask >> s & 1ull) {
              g += fxw_get(*dl, M.fxw_inv);
              *dl = 0.0;
            }
            if (g != 0.0) {
              const double gs = g * sc;
              fx_add(rows, gs, M.overflow);
              fx_add(rows + 32, gs * e, M.overflow);
              g = decay(g, c0);
            }
          }
          T.state[0][q] = g;
          break;
        }
        case T_EXP2SYN: {
          double A = T.state[0][q], B = T.state[1][q];
          const double c0 = T.param[0][q], c1 = T.param[1][q], e = T.param[2][q], sc = T.param[3][q],
                       f = T.param[4][q];
          for (int s = 0; s < nsteps; ++s, rows += M.win_stride, dl += M.win_ninst) {
            if (mask >> s & 1ull) {
              const double wf = fxw_get(*dl, M.fxw_inv) * f;
              A += wf;
              B += wf;
              *dl = 0.0;
            }
            if (A != 0.0 || B != 0.0) {
              const double gs = (B - A) * sc;
              if (gs != 0.0) {
                fx_add(rows, gs, M.overflow);
                fx_add(rows + 32, gs * e, M.overflow);
              }
              A = decay(A, c0);
              B = decay(B, c1);
            }
          }
          T.state[0][q] = A;
          T.state[1][q] = B;
          break;
        }
        case T_ICLAMP: {
          const double del = T.param[0][q], dur = T.param[1][q];
          for (int s = 0; s < nsteps; ++s, rows += M.win_stride) {
            const double t_mid = ((double)(k0 + s) + 0.5) * dt;
            if (t_mid >= del && t_mid < del + dur)
              fx_add(rows + 32, T.param[2][q] * T.param[3][q], M.overflow);
          }
          break;
        }
        default: break;
      }
    }
  }
}

__global__ void probe_kernel(const double *__restrict__ v, const int64_t *__restrict__ pos,
                             int n_probe, double *__restrict__ trace, int64_t row,
                             const int64_t *__restrict__ ctr, int64_t cap) {
  if (row < 0) row = ctr[1] - row - 1;  // replayed graph: the device counter + offset
  if (row >= cap) return;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j < n_probe) trace[row * n_probe + j] = v[pos[j]];
}

__global__ void set_ctr_kernel(int64_t *ctr, int64_t k, int64_t row) {
  ctr[0] = k;
  ctr[1] = row;
}

__global__ void gather_kernel(const double *__restrict__ src, const int64_t *__restrict__ pos,
                              int64_t n, double *__restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = src[pos[i]];
}

__global__ void scatter_kernel(double *__restrict__ dst, const int64_t *__restrict__ pos,
                               int64_t n, const double *__restrict__ src) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[pos[i]] = src[i];
}

}  // namespace cn
