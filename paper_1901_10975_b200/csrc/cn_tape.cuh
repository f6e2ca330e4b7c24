// cn_tape.cuh -- the interleaved step kernel: one warp integrates 32 cells of one shape class for
// one dt, ONE LANE PER CELL ("one cell per thread", Fig. 5D), re-designed for B200:
//
//   * Every per-node quantity of the 32 cells is a ROW of 32 doubles (256 B).  All rows of a group
//     are laid out in the order the elimination visits them -- a TAPE: per node a, b, static
//     diagonal, static rhs, v, then the parameter and state rows of the mechanisms on that node.
//     The kernel never computes an address from the tree: it reads the tape front to back.
//   * The tape is staged through a shared-memory ring by 1-D TMA bulk copies
//     (cp.async.bulk.shared.global + mbarrier complete_tx), S chunks of CH rows in flight per warp,
//     issued by one lane; HBM latency is hidden by the ring, not by occupancy.
//   * Nodes are visited in depth-first post-order (children before parents, L196), so a node's
//     contribution to its parent stays in REGISTERS when the parent is next (chains), and goes
//     through a small shared-memory stack at branch points (depth <= height in branch points).
//     No per-node shared-memory system: the shared memory per warp is ring + stack + program.
//   * Triangularisation (L66) writes the back-substitution multiplier and reduced rhs of every
//     node to a SCRATCH tape in reverse order; back-substitution streams it back through the same
//     ring (it is re-read within microseconds: L2-resident), computes v_new, runs nrn_state (L67)
//     on the mechanisms of the node and detects threshold crossings at the root (L68).
//   * Control is uniform across the warp: the per-class PROGRAM (one uint4 per node) says where
//     the node's rows are, how it hands its contribution to the parent, and which mechanisms sit
//     on it.  Lanes never diverge.
// Point processes of these cells are evaluated by pp_tape_kernel (one thread per instance) which
// adds conductance and current into two dynamic tape rows of the node (L60, L65).
#pragma once
#include "cn_device.cuh"

namespace cn {

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes,
                                         uint32_t bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
      ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(bar), "r"(parity)
      : "memory");
}

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

// x / (exp(x/y) - 1) for y = 10 (both HH uses), removable singularity as in vtrap()
__device__ __forceinline__ double vtrap10(double x) {
  const double u = x * 0.1;
  if (fabs(u) < 1e-6) return 10.0 * (1.0 - 0.5 * u);
  return x * rcp_fast(exp(u) - 1.0);
}

// HH gates advanced over dt with cnexp at the new v: y += (1 - exp(-dt*q10*(a+b))) * (a/(a+b) - y).
// Same formulas as hh_rates() + cnexp(); divisions by constants are multiplications by their
// reciprocals and 1/tau is never formed (differences of a few ulp).
__device__ __forceinline__ void hh_advance(double v, double q10dt, double &m, double &h,
                                           double &n) {
  double al, be, s;
  al = 0.1 * vtrap10(-(v + 40.0));
  be = 4.0 * exp(-(v + 65.0) * (1.0 / 18.0));
  s = al + be;
  m += (1.0 - exp(-q10dt * s)) * (al * rcp_fast(s) - m);
  al = 0.07 * exp(-(v + 65.0) * 0.05);
  be = rcp_fast(exp(-(v + 35.0) * 0.1) + 1.0);
  s = al + be;
  h += (1.0 - exp(-q10dt * s)) * (al * rcp_fast(s) - h);
  al = 0.01 * vtrap10(-(v + 55.0));
  be = 0.125 * exp(-(v + 65.0) * 0.0125);
  s = al + be;
  n += (1.0 - exp(-q10dt * s)) * (al * rcp_fast(s) - n);
}

__device__ __forceinline__ void bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// One CTA = one group of 32 cells, W warps.  Warp w runs leaf task w (a set of whole subtrees);
// warp 0 then runs the top task (the part of the tree above the cut, root included), after which
// every warp back-substitutes its leaf task.  S stages of CH rows per warp; S * CH is a power of 2.
//
// Program entry (uint4, one per node in task order; built by the host, uniform per class):
//   x = byte offset in the ring of the node's first tape row (low 16 bits) and of its first
//       scratch row (high 16 bits), relative to the task's segments
//   y = element offset of the node's scratch record on the group's scratch tape
//   z = flags (8 bits) | chunks to wait for, forward (4) | chunks freed, forward (4)
//       | chunks to wait for, backward (4) | chunks freed, backward (4) | tape rows (8)
//   w = mask of the distributed mechanism tables with an instance on this node (20 bits)
//       | exchange slot: own slot of a cut subtree root, first import slot of a top node (8 bits)
//       | number of import slots (4 bits)
template <int S, int CH>
__global__ void __launch_bounds__(128, 4) tape_step_kernel(const __grid_constant__ DModel M,
                                                        int64_t k) {
  extern __shared__ __align__(128) unsigned char sm_raw[];
  constexpr uint32_t RB = S * CH * 256u;  // ring bytes per warp
  static_assert((RB & (RB - 1)) == 0 && RB <= 65536u, "ring must be a power of two <= 64 KB");
  static_assert((S & (S - 1)) == 0, "stages must be a power of two");
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int W = M.tape_W;
  const int nthreads = W * 32;
  const uint32_t lane8 = (uint32_t)lane * 8u;
  const TapeGroup tg = M.tgrp[blockIdx.x];
  const TapeClass tc = M.tcls[tg.cls];
  // shared memory: rings | program | stacks | exchange slots | mbarriers
  const unsigned char *ringc = sm_raw + (size_t)warp * RB;
  uint4 *prog = reinterpret_cast<uint4 *>(sm_raw + (size_t)W * RB);
  double *stk = reinterpret_cast<double *>(prog + M.tape_prog_cap) +
                (size_t)warp * M.tape_stack_cap * 64;
  double *xs = reinterpret_cast<double *>(prog + M.tape_prog_cap) +
               (size_t)W * M.tape_stack_cap * 64;
  uint64_t *mbar = reinterpret_cast<uint64_t *>(xs + (size_t)M.tape_xs_cap * 64) +
                   (size_t)warp * (S + 1);
  const uint32_t ring_s = smem_u32(ringc), bar_s = smem_u32(mbar);
  double *__restrict__ tape = M.tape + tg.tape_base;
  double *__restrict__ scr = M.scratch + tg.scratch_base;
  double *__restrict__ tape_l = tape + lane;
  double *__restrict__ scr_l = scr + lane;
  const double dt = M.dt;
  const double q10dt = M.q10 * dt;
  const TapeTask *tasks = M.ttask + (size_t)tg.cls * (W + 1);

  // the host pads the tapes so that no record wraps around the ring: row i of a record is at a
  // fixed distance from its first row
#define CN_RD(base, i) (*reinterpret_cast<const double *>((base) + (uint32_t)(i) * 256u))

  // chunk c of a row stream goes to stage c % S
  auto issue = [&](const double *base, int c, int total_rows) {
    const int rows = min(CH, total_rows - c * CH);
    const uint32_t bytes = (uint32_t)rows * 256u;
    const int s = c & (S - 1);
    mbar_expect_tx(bar_s + 8 * s, bytes);
    bulk_g2s(ring_s + (uint32_t)s * (CH * 256), base + (size_t)c * (CH * 32), bytes,
             bar_s + 8 * s);
  };

  uint32_t phase = 0;  // bit s: parity the next wait on stage s looks for
  uint32_t ws = 0;     // stage of the next chunk to wait for
  int ci = S;          // next chunk to issue

  const TapeTask leaf = tasks[warp];
  if (lane == 0) {
    for (int s = 0; s <= S; ++s) mbar_init(bar_s + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    // this warp's slice of the program (warp 0: also the top task's, which follows the leaves')
    const int q0 = leaf.p0, q1 = leaf.p1;
    uint32_t bytes = 0;
    if (warp == 0) {
      bytes = (uint32_t)(leaf.p1 - leaf.p0 + tasks[W].p1 - tasks[W].p0) * 16u;
      mbar_expect_tx(bar_s + 8 * S, bytes);
      if (leaf.p1 > leaf.p0)
        bulk_g2s(smem_u32(prog + leaf.p0), M.prog + tc.prog_off + leaf.p0,
                 (uint32_t)(leaf.p1 - leaf.p0) * 16u, bar_s + 8 * S);
      bulk_g2s(smem_u32(prog + tasks[W].p0), M.prog + tc.prog_off + tasks[W].p0,
               (uint32_t)(tasks[W].p1 - tasks[W].p0) * 16u, bar_s + 8 * S);
    } else {
      bytes = (uint32_t)(q1 - q0) * 16u;
      mbar_expect_tx(bar_s + 8 * S, bytes);
      if (bytes) bulk_g2s(smem_u32(prog + q0), M.prog + tc.prog_off + q0, bytes, bar_s + 8 * S);
    }
    const int nchunk0 = ((int)leaf.nrows + CH - 1) / CH;
    for (int c = 0; c < S && c < nchunk0; ++c)
      issue(tape + (size_t)leaf.row0 * 32, c, (int)leaf.nrows);
  }
  __syncwarp();
  mbar_wait(bar_s + 8 * S, 0);

  int sp = 0;
  // ==========================================================================================
  // forward: nrn_cur + tree terms + triangularisation, children before parents.
  // phase 0: the warp's leaf task; phase 1 (warp 0 only, after all leaves): the top task
  // ==========================================================================================
  const int n_fwd = warp == 0 ? 2 : 1;
  for (int ph = 0; ph < n_fwd; ++ph) {
    const TapeTask tk = ph == 0 ? leaf : tasks[W];
    const double *tseg = tape + (size_t)tk.row0 * 32;
    const int nchunk = ((int)tk.nrows + CH - 1) / CH;
    if (ph == 1) {
      bar_sync(1, nthreads);  // every leaf task has exported its subtree roots
      ws = 0;
      ci = S;
      if (lane == 0)
        for (int c = 0; c < S && c < nchunk; ++c) issue(tseg, c, (int)tk.nrows);
    }
    uint32_t grow = tk.row0 * 32u;  // element offset of the current record on the group's tape
    double accD = 0.0, accR = 0.0;
    for (int j = tk.p0; j < tk.p1; ++j) {
      const uint4 e = prog[j];
      const uint32_t fl = e.z;
      for (uint32_t nw = (fl >> 8) & 15u; nw; --nw) {
        mbar_wait(bar_s + 8 * ws, (phase >> ws) & 1u);
        phase ^= 1u << ws;
        ws = (ws + 1) & (S - 1);
      }
      const unsigned char *rb = ringc + ((e.x & 0xFFFFu) + lane8);
      double *__restrict__ srec = scr_l + e.y;
      const double a = CN_RD(rb, 0), b = CN_RD(rb, 1);
      const double v_old = CN_RD(rb, 4);
      double D = CN_RD(rb, 2), R = v_old + CN_RD(rb, 3);
      double mult, rp;
      if ((fl & (0xFFu & ~PG_FWD_IN)) == PG_FWD && e.w == 0u) {
        // FAST PATH (most nodes): interior or tip of an unbranched stretch, no mechanism rows;
        // the contribution to the parent stays in registers
        if (fl & PG_FWD_IN) {
          D += accD;
          R += accR;
        }
        const double rinv = rcp_fast(D);
        const double f = a * rinv;
        rp = R * rinv;
        mult = b * rinv;
        accD = -(f * b);
        accR = -(f * R);
      } else {
      double *__restrict__ trec = tape_l + grow;
      uint32_t cur = 5, scur = 2;
      if (fl & PG_FWD_IN) {
        D += accD;
        R += accR;
      }
      if (fl & PG_POP) {
        --sp;
        D += stk[sp * 64 + lane];
        R += stk[sp * 64 + 32 + lane];
      }
      for (uint32_t ni = e.w >> 28, s0 = (e.w >> 20) & 255u; ni; --ni, ++s0) {  // cut subtrees
        D += xs[s0 * 64 + lane];
        R += xs[s0 * 64 + 32 + lane];
      }
      if (fl & PG_HAS_PP) {  // conductance / current of the point processes (pp_tape_kernel)
        const double pd = CN_RD(rb, 5), pr = CN_RD(rb, 6);
        D += pd;
        R += pr;
        if (pd != 0.0 || pr != 0.0) {
          trec[5 * 32] = 0.0;
          trec[6 * 32] = 0.0;
        }
        cur = 7;
      }
      double ica = 0.0;
      if (fl & PG_NEED_ICA) ++scur;
      if (fl & PG_HAS_CAI) {
        srec[scur * 32] = CN_RD(rb, cur);
        ++cur;
        ++scur;
      }
      for (uint32_t mk = e.w & 0xFFFFFu; mk; mk &= mk - 1) {
        const DTable &T = M.tab[__ffs(mk) - 1];
        const unsigned char *mr = rb + cur * 256u;
        switch (T.type) {
          case T_HH: {
            const double m = CN_RD(mr, 5), h = CN_RD(mr, 6), nn = CN_RD(mr, 7);
            const double invc = CN_RD(mr, 4);
            const double gna = CN_RD(mr, 0) * m * m * m * h;
            const double n2 = nn * nn;
            const double gk = CN_RD(mr, 1) * n2 * n2;
            const double gl = CN_RD(mr, 2);
            D += (gna + gk + gl) * invc;
            R += (gna * T.glob[0] + gk * T.glob[1] + gl * CN_RD(mr, 3)) * invc;
            srec[scur * 32] = m;
            srec[(scur + 1) * 32] = h;
            srec[(scur + 2) * 32] = nn;
            cur += 8;
            scur += 3;
            break;
          }
          case T_HHFORM: {
            const double ms = CN_RD(mr, 2), hs = CN_RD(mr, 3);
            const double g = CN_RD(mr, 0) * ipow(ms, (int)T.glob[0]) * ipow(hs, (int)T.glob[1]);
            const double invc = CN_RD(mr, 1);
            D += g * invc;
            R += g * T.glob[2] * invc;
            if (T.glob[3] != 0.0) ica += g * (v_old - T.glob[2]);
            srec[scur * 32] = ms;
            srec[(scur + 1) * 32] = hs;
            cur += 4;
            scur += 2;
            break;
          }
          case T_SK: {
            const double z = CN_RD(mr, 2);
            const double g = CN_RD(mr, 0) * z;
            const double invc = CN_RD(mr, 1);
            D += g * invc;
            R += g * T.glob[0] * invc;
            srec[scur * 32] = z;
            cur += 3;
            scur += 1;
            break;
          }
          default: break;  // PAS is folded into the static rows; CADYN carries no current
        }
      }
      if (fl & PG_NEED_ICA) srec[2 * 32] = ica;
      const double rinv = rcp_fast(D);
      rp = R * rinv;
      mult = 0.0;
      if (!(fl & PG_ROOT)) {
        const double f = a * rinv;
        const double cD = -(f * b), cR = -(f * R);
        mult = b * rinv;  // back-substitution multiplier
        const uint32_t kind = fl & PG_KIND;
        if (kind == PG_FWD) {
          accD = cD;
          accR = cR;
        } else if (kind == PG_PUSH) {
          stk[sp * 64 + lane] = cD;
          stk[sp * 64 + 32 + lane] = cR;
          ++sp;
        } else if (kind == PG_ADD) {
          stk[(sp - 1) * 64 + lane] += cD;
          stk[(sp - 1) * 64 + 32 + lane] += cR;
        } else {  // root of a cut subtree: export to the top task
          const uint32_t s0 = (e.w >> 20) & 255u;
          xs[s0 * 64 + lane] = cD;
          xs[s0 * 64 + 32 + lane] = cR;
        }
      }
      }
      srec[0] = mult;
      srec[32] = rp;
      grow += (fl >> 24) * 32u;
      // stages whose rows are all consumed are refilled S chunks ahead
      uint32_t nf = (fl >> 12) & 15u;
      if (nf) {
        __syncwarp();
        if (lane == 0)
          for (; nf; --nf, ++ci)
            if (ci < nchunk) issue(tseg, ci, (int)tk.nrows);
        ci = __shfl_sync(0xffffffffu, ci, 0);
      }
    }
    if (ph == 0 && warp != 0) bar_arrive(1, nthreads);
  }

  // ==========================================================================================
  // backward: back-substitution (L66), nrn_state with the new v (L67), threshold at the root
  // (L68).  phase 0 (warp 0 only): the top task; phase 1 (after it): the warp's leaf task
  // ==========================================================================================
  asm volatile("fence.proxy.async;" ::: "memory");  // scratch written above, read by bulk copies
  __syncwarp();
  for (int ph = warp == 0 ? 0 : 1; ph < 2; ++ph) {
    const TapeTask tk = ph == 0 ? tasks[W] : leaf;
    const double *sseg = scr + (size_t)tk.srow0 * 32;
    const int nsch = ((int)tk.nsrows + CH - 1) / CH;
    if (lane == 0)
      for (int c = 0; c < S && c < nsch; ++c) issue(sseg, c, (int)tk.nsrows);
    ws = 0;
    ci = S;
    if (ph == 1) {  // the top task has written v of every cut subtree's parent
      if (warp == 0) bar_arrive(2, nthreads);
      else bar_sync(2, nthreads);
    }
    uint32_t grow = (tk.row0 + tk.nrows) * 32u;
    double v_prev = 0.0;
    sp = 0;
    for (int j = tk.p1 - 1; j >= tk.p0; --j) {
      const uint4 e = prog[j];
      const uint32_t fl = e.z;
      grow -= (fl >> 24) * 32u;
      for (uint32_t nw = (fl >> 16) & 15u; nw; --nw) {
        mbar_wait(bar_s + 8 * ws, (phase >> ws) & 1u);
        phase ^= 1u << ws;
        ws = (ws + 1) & (S - 1);
      }
      const unsigned char *sb = ringc + ((e.x >> 16) + lane8);
      double *__restrict__ trec = tape_l + grow;
      if ((fl & (0xFFu & ~PG_FWD_IN)) == PG_FWD && e.w == 0u) {
        // FAST PATH: the parent is the node just solved
        v_prev = fma(-CN_RD(sb, 0), v_prev, CN_RD(sb, 1));
        trec[4 * 32] = v_prev;
      } else {
      const uint32_t kind = fl & PG_KIND;
      double vp = v_prev;
      if (kind == PG_ADD) vp = stk[(sp - 1) * 32 + lane];
      if (kind == PG_PUSH) vp = stk[(--sp) * 32 + lane];
      if (kind == 0 && !(fl & PG_ROOT)) vp = xs[((e.w >> 20) & 255u) * 64 + lane];
      const double v = fma(-CN_RD(sb, 0), vp, CN_RD(sb, 1));  // the root's multiplier is 0
      if (fl & PG_POP) stk[(sp++) * 32 + lane] = v;
      for (uint32_t ni = e.w >> 28, s0 = (e.w >> 20) & 255u; ni; --ni, ++s0)
        xs[s0 * 64 + lane] = v;  // v of the parent of cut subtrees
      v_prev = v;
      trec[4 * 32] = v;
      uint32_t cur = 5 + ((fl & PG_HAS_PP) ? 2u : 0u), scur = 2;
      double ica = 0.0, cai = 0.0;
      uint32_t cai_row = 0;
      if (fl & PG_NEED_ICA) ica = CN_RD(sb, scur++);
      if (fl & PG_HAS_CAI) {
        cai = CN_RD(sb, scur++);
        cai_row = cur++;
      }
      for (uint32_t mk = e.w & 0xFFFFFu; mk; mk &= mk - 1) {
        const DTable &T = M.tab[__ffs(mk) - 1];
        const unsigned char *ms = sb + scur * 256u;
        switch (T.type) {
          case T_HH: {
            double m = CN_RD(ms, 0), h = CN_RD(ms, 1), nn = CN_RD(ms, 2);
            hh_advance(v, q10dt, m, h, nn);
            trec[(cur + 5) * 32] = m;
            trec[(cur + 6) * 32] = h;
            trec[(cur + 7) * 32] = nn;
            cur += 8;
            scur += 3;
            break;
          }
          case T_HHFORM: {
            double xinf, xtau;
            if ((int)T.glob[0] > 0) {
              hhform_gate(v, T.glob + 4, xinf, xtau);
              trec[(cur + 2) * 32] = cnexp(CN_RD(ms, 0), xinf, xtau, dt);
            }
            if ((int)T.glob[1] > 0) {
              hhform_gate(v, T.glob + 10, xinf, xtau);
              trec[(cur + 3) * 32] = cnexp(CN_RD(ms, 1), xinf, xtau, dt);
            }
            cur += 4;
            scur += 2;
            break;
          }
          case T_SK: {
            const double ca = cai < 1e-9 ? 1e-9 : cai;
            const double zinf = 1.0 / (1.0 + pow(T.glob[1] / ca, T.glob[2]));
            trec[(cur + 2) * 32] = cnexp(CN_RD(ms, 0), zinf, T.glob[3], dt);
            cur += 3;
            scur += 1;
            break;
          }
          case T_CADYN: {
            // derivimplicit on a linear ODE: one Newton step of backward Euler is exact (L278)
            const double kappa = 1e4 * T.glob[0] / (2.0 * 96485.33212 * T.glob[1]);
            cai = (cai + dt * (-kappa * ica + T.glob[3] / T.glob[2])) / (1.0 + dt / T.glob[2]);
            trec[cai_row * 32] = cai;
            break;
          }
          default: break;
        }
      }
      if (fl & PG_ROOT) {  // warp-ballot threshold detection, one atomic per warp
        bool fire = false;
        const int pc = tg.cell_base + lane;
        if (lane < tg.ncell) {
          const bool above = v > M.thr[pc];
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
      uint32_t nf = (fl >> 20) & 15u;
      if (nf) {
        __syncwarp();
        if (lane == 0)
          for (; nf; --nf, ++ci)
            if (ci < nsch) issue(sseg, ci, (int)tk.nsrows);
        ci = __shfl_sync(0xffffffffu, ci, 0);
      }
    }
  }
#undef CN_RD
}

// ------------------------------------------------------------------------------------------------
// point processes on tape cells: current + conductance into the node's dynamic rows, then the
// state decay (independent of v for these types, so cur and state fuse exactly; L65, L67)
// ------------------------------------------------------------------------------------------------

__global__ void __launch_bounds__(256) pp_tape_kernel(const __grid_constant__ DModel M,
                                                      int64_t k) {
  const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t nth = (int64_t)gridDim.x * blockDim.x;
  const double dt = M.dt;
  const double t_mid = ((double)k + 0.5) * dt;
  double *__restrict__ tape = M.tape;
  for (int t = 0; t < M.n_table; ++t) {
    const DTable &T = M.tab[t];
    if (!T.is_point) continue;
    const uint32_t *__restrict__ tgt = reinterpret_cast<const uint32_t *>(T.pp_slot);
    switch (T.type) {
      case T_EXPSYN:
        for (int64_t q = T.pp_tape_begin + tid; q < T.pp_tape_end; q += nth) {
          const double g = T.state[0][q];
          if (g != 0.0) {
            const double gs = g * T.param[2][q];
            atomicAdd(&tape[tgt[q]], gs);
            atomicAdd(&tape[tgt[q] + 32], gs * T.param[1][q]);
            T.state[0][q] = cnexp(g, 0.0, T.param[0][q], dt);
          }
        }
        break;
      case T_EXP2SYN:
        for (int64_t q = T.pp_tape_begin + tid; q < T.pp_tape_end; q += nth) {
          const double A = T.state[0][q], B = T.state[1][q];
          if (A != 0.0 || B != 0.0) {
            const double gs = (B - A) * T.param[3][q];
            if (gs != 0.0) {
              atomicAdd(&tape[tgt[q]], gs);
              atomicAdd(&tape[tgt[q] + 32], gs * T.param[2][q]);
            }
            T.state[0][q] = cnexp(A, 0.0, T.param[0][q], dt);
            T.state[1][q] = cnexp(B, 0.0, T.param[1][q], dt);
          }
        }
        break;
      case T_ICLAMP:
        for (int64_t q = T.pp_tape_begin + tid; q < T.pp_tape_end; q += nth) {
          const double del = T.param[0][q];
          if (t_mid >= del && t_mid < del + T.param[1][q])
            atomicAdd(&tape[tgt[q] + 32], T.param[2][q] * T.param[3][q]);
        }
        break;
      case T_AMPANMDA:
        for (int64_t q = T.pp_tape_begin + tid; q < T.pp_tape_end; q += nth) {
          const double a0 = T.state[0][q], a1 = T.state[1][q], a2 = T.state[2][q],
                       a3 = T.state[3][q];
          if (a0 != 0.0 || a1 != 0.0 || a2 != 0.0 || a3 != 0.0) {
            const double v = tape[tgt[q] - 32];  // the v row precedes the two dynamic rows
            const double gs =
                ((a1 - a0) + T.glob[4] * (a3 - a2) * mgblock(v, T.glob[5])) * T.param[0][q];
            atomicAdd(&tape[tgt[q]], gs);
            atomicAdd(&tape[tgt[q] + 32], gs * T.glob[6]);
            T.state[0][q] = cnexp(a0, 0.0, T.glob[0], dt);
            T.state[1][q] = cnexp(a1, 0.0, T.glob[1], dt);
            T.state[2][q] = cnexp(a2, 0.0, T.glob[2], dt);
            T.state[3][q] = cnexp(a3, 0.0, T.glob[3], dt);
          }
        }
        break;
      default: break;
    }
  }
}

// state s of mixed-layout instances: loc >= 0 -> table array, loc < 0 -> tape element -(loc+1)
__global__ void gather_state_kernel(const double *__restrict__ tape,
                                    const double *__restrict__ st,
                                    const int64_t *__restrict__ loc, int64_t n, int s,
                                    double *__restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int64_t l = loc[i];
  out[i] = l >= 0 ? st[l] : tape[-(l + 1) + (int64_t)s * 32];
}

}  // namespace cn
