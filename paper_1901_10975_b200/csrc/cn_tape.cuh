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

// S stages of CH rows; S * CH must be a power of two.
template <int S, int CH>
__global__ void __launch_bounds__(32) tape_step_kernel(const __grid_constant__ DModel M,
                                                       int64_t k) {
  extern __shared__ __align__(128) unsigned char sm_raw[];
  constexpr int RING_ROWS = S * CH;
  static_assert((RING_ROWS & (RING_ROWS - 1)) == 0, "ring rows must be a power of two");
  const int lane = threadIdx.x;
  const TapeGroup tg = M.tgrp[blockIdx.x];
  const TapeClass tc = M.tcls[tg.cls];
  double *ring = reinterpret_cast<double *>(sm_raw);
  uint4 *prog = reinterpret_cast<uint4 *>(ring + RING_ROWS * 32);
  double *stk = reinterpret_cast<double *>(prog + M.tape_prog_cap);
  uint64_t *mbar = reinterpret_cast<uint64_t *>(stk + M.tape_stack_cap * 64);
  const uint32_t ring_s = smem_u32(ring), bar_s = smem_u32(mbar);
  double *__restrict__ tape = M.tape + tg.tape_base;
  double *__restrict__ scr = M.scratch + tg.scratch_base;
  const int n = tc.n;
  const int nchunk = (tc.n_rows + CH - 1) / CH;
  const int nsch = (tc.n_srows + CH - 1) / CH;
  const double dt = M.dt;

#define CN_ROW(r) ring[((((uint32_t)(r)) & (RING_ROWS - 1)) << 5) + lane]

  // chunk c of a row stream goes to stage c % S
  auto issue = [&](const double *base, int c, int total_rows) {
    const int rows = min(CH, total_rows - c * CH);
    const uint32_t bytes = (uint32_t)rows * 256u;
    const int s = c % S;
    mbar_expect_tx(bar_s + 8 * s, bytes);
    bulk_g2s(ring_s + (uint32_t)s * (CH * 256), base + (size_t)c * (CH * 32), bytes,
             bar_s + 8 * s);
  };

  if (lane == 0) {
    for (int s = 0; s <= S; ++s) mbar_init(bar_s + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_expect_tx(bar_s + 8 * S, (uint32_t)n * 16u);
    bulk_g2s(smem_u32(prog), M.prog + tc.prog_off, (uint32_t)n * 16u, bar_s + 8 * S);
    for (int c = 0; c < S && c < nchunk; ++c) issue(tape, c, tc.n_rows);
  }
  __syncwarp();
  mbar_wait(bar_s + 8 * S, 0);

  // ------------------------------------------------------------------------------------------
  // forward: nrn_cur + tree terms + triangularisation, children before parents
  // ------------------------------------------------------------------------------------------
  int c_wait = -1, c_free = 0, sp = 0;
  double accD = 0.0, accR = 0.0, v_root = 0.0;
  for (int j = 0; j < n; ++j) {
    const uint4 e = prog[j];
    const uint32_t row = e.x, sr = e.y, fl = e.z, len = (e.z >> 8) & 0xFFu;
    const int c_last = (int)((row + len - 1) / CH);
    while (c_wait < c_last) {
      ++c_wait;
      mbar_wait(bar_s + 8 * (c_wait % S), (uint32_t)(c_wait / S) & 1u);
    }
    const double a = CN_ROW(row), b = CN_ROW(row + 1);
    const double v_old = CN_ROW(row + 4);
    double D = CN_ROW(row + 2), R = v_old + CN_ROW(row + 3);
    uint32_t cur = row + 5, scur = sr + 2;
    if (fl & PG_FWD_IN) {
      D += accD;
      R += accR;
    }
    if (fl & PG_POP) {
      --sp;
      D += stk[sp * 64 + lane];
      R += stk[sp * 64 + 32 + lane];
    }
    if (fl & PG_HAS_PP) {  // conductance / current of the point processes (pp_tape_kernel)
      const double pd = CN_ROW(cur), pr = CN_ROW(cur + 1);
      D += pd;
      R += pr;
      if (pd != 0.0 || pr != 0.0) {
        tape[(size_t)cur * 32 + lane] = 0.0;
        tape[(size_t)(cur + 1) * 32 + lane] = 0.0;
      }
      cur += 2;
    }
    double ica = 0.0;
    if (fl & PG_NEED_ICA) ++scur;
    if (fl & PG_HAS_CAI) {
      scr[(size_t)scur * 32 + lane] = CN_ROW(cur);
      ++cur;
      ++scur;
    }
    for (uint32_t mk = e.w; mk; mk &= mk - 1) {
      const DTable &T = M.tab[__ffs(mk) - 1];
      switch (T.type) {
        case T_HH: {
          const double m = CN_ROW(cur + 5), h = CN_ROW(cur + 6), nn = CN_ROW(cur + 7);
          const double invc = CN_ROW(cur + 4);
          const double gna = CN_ROW(cur) * m * m * m * h;
          const double n2 = nn * nn;
          const double gk = CN_ROW(cur + 1) * n2 * n2;
          const double gl = CN_ROW(cur + 2);
          D += (gna + gk + gl) * invc;
          R += (gna * T.glob[0] + gk * T.glob[1] + gl * CN_ROW(cur + 3)) * invc;
          scr[(size_t)scur * 32 + lane] = m;
          scr[(size_t)(scur + 1) * 32 + lane] = h;
          scr[(size_t)(scur + 2) * 32 + lane] = nn;
          cur += 8;
          scur += 3;
          break;
        }
        case T_HHFORM: {
          const double ms = CN_ROW(cur + 2), hs = CN_ROW(cur + 3);
          const double g = CN_ROW(cur) * ipow(ms, (int)T.glob[0]) * ipow(hs, (int)T.glob[1]);
          const double invc = CN_ROW(cur + 1);
          D += g * invc;
          R += g * T.glob[2] * invc;
          if (T.glob[3] != 0.0) ica += g * (v_old - T.glob[2]);
          scr[(size_t)scur * 32 + lane] = ms;
          scr[(size_t)(scur + 1) * 32 + lane] = hs;
          cur += 4;
          scur += 2;
          break;
        }
        case T_SK: {
          const double z = CN_ROW(cur + 2);
          const double g = CN_ROW(cur) * z;
          const double invc = CN_ROW(cur + 1);
          D += g * invc;
          R += g * T.glob[0] * invc;
          scr[(size_t)scur * 32 + lane] = z;
          cur += 3;
          scur += 1;
          break;
        }
        default: break;  // PAS is folded into the static rows; CADYN carries no current
      }
    }
    if (fl & PG_NEED_ICA) scr[(size_t)(sr + 2) * 32 + lane] = ica;
    double mult = 0.0, rp;
    if (fl & PG_ROOT) {
      rp = R / D;
      v_root = rp;
    } else {
      const double rinv = 1.0 / D;
      const double f = a * rinv;
      const double cD = -(f * b), cR = -(f * R);
      mult = b * rinv;  // back-substitution multiplier
      rp = R * rinv;
      const uint32_t kind = fl & PG_KIND;
      if (kind == PG_FWD) {
        accD = cD;
        accR = cR;
      } else if (kind == PG_PUSH) {
        stk[sp * 64 + lane] = cD;
        stk[sp * 64 + 32 + lane] = cR;
        ++sp;
      } else {
        stk[(sp - 1) * 64 + lane] += cD;
        stk[(sp - 1) * 64 + 32 + lane] += cR;
      }
    }
    scr[(size_t)sr * 32 + lane] = mult;
    scr[(size_t)(sr + 1) * 32 + lane] = rp;
    // stages whose rows are all consumed are refilled S chunks ahead
    const int c_next = (int)((row + len) / CH);
    if (c_free < c_next) {
      __syncwarp();
      if (lane == 0)
        for (int c = c_free; c < c_next; ++c)
          if (c + S < nchunk) issue(tape, c + S, tc.n_rows);
      c_free = c_next;
    }
  }

  // ------------------------------------------------------------------------------------------
  // backward: back-substitution (L66), nrn_state with the new v (L67), threshold at the root (L68)
  // ------------------------------------------------------------------------------------------
  asm volatile("fence.proxy.async;" ::: "memory");  // scratch written above, read by bulk copies
  __syncwarp();
  if (lane == 0)
    for (int c = 0; c < S && c < nsch; ++c) issue(scr, c, tc.n_srows);
  int b_wait = -1, b_free = 0;
  double v_prev = 0.0;
  sp = 0;
  for (int j = n - 1; j >= 0; --j) {
    const uint4 e = prog[j];
    const uint32_t row = e.x, sr = e.y, fl = e.z, slen = (e.z >> 16) & 0xFFu;
    const int c_last = (int)((sr + slen - 1) / CH);
    while (b_wait < c_last) {
      ++b_wait;
      const int s = b_wait % S;
      const int used = (nchunk > s ? (nchunk - s + S - 1) / S : 0) + b_wait / S;
      mbar_wait(bar_s + 8 * s, (uint32_t)used & 1u);
    }
    const uint32_t kind = fl & PG_KIND;
    double vp = v_prev;
    if (kind == PG_ADD) vp = stk[(sp - 1) * 32 + lane];
    if (kind == PG_PUSH) vp = stk[(--sp) * 32 + lane];
    double v = CN_ROW(sr + 1);
    if (!(fl & PG_ROOT)) v -= CN_ROW(sr) * vp;
    if (fl & PG_POP) stk[(sp++) * 32 + lane] = v;
    v_prev = v;
    tape[(size_t)(row + 4) * 32 + lane] = v;
    uint32_t cur = row + 5 + ((fl & PG_HAS_PP) ? 2u : 0u), scur = sr + 2;
    double ica = 0.0, cai = 0.0;
    uint32_t cai_row = 0;
    if (fl & PG_NEED_ICA) ica = CN_ROW(scur++);
    if (fl & PG_HAS_CAI) {
      cai = CN_ROW(scur++);
      cai_row = cur++;
    }
    for (uint32_t mk = e.w; mk; mk &= mk - 1) {
      const DTable &T = M.tab[__ffs(mk) - 1];
      switch (T.type) {
        case T_HH: {
          double minf, mtau, hinf, htau, ninf, ntau;
          hh_rates(v, M.q10, minf, mtau, hinf, htau, ninf, ntau);
          tape[(size_t)(cur + 5) * 32 + lane] = cnexp(CN_ROW(scur), minf, mtau, dt);
          tape[(size_t)(cur + 6) * 32 + lane] = cnexp(CN_ROW(scur + 1), hinf, htau, dt);
          tape[(size_t)(cur + 7) * 32 + lane] = cnexp(CN_ROW(scur + 2), ninf, ntau, dt);
          cur += 8;
          scur += 3;
          break;
        }
        case T_HHFORM: {
          double xinf, xtau;
          if ((int)T.glob[0] > 0) {
            hhform_gate(v, T.glob + 4, xinf, xtau);
            tape[(size_t)(cur + 2) * 32 + lane] = cnexp(CN_ROW(scur), xinf, xtau, dt);
          }
          if ((int)T.glob[1] > 0) {
            hhform_gate(v, T.glob + 10, xinf, xtau);
            tape[(size_t)(cur + 3) * 32 + lane] = cnexp(CN_ROW(scur + 1), xinf, xtau, dt);
          }
          cur += 4;
          scur += 2;
          break;
        }
        case T_SK: {
          const double ca = cai < 1e-9 ? 1e-9 : cai;
          const double zinf = 1.0 / (1.0 + pow(T.glob[1] / ca, T.glob[2]));
          tape[(size_t)(cur + 2) * 32 + lane] = cnexp(CN_ROW(scur), zinf, T.glob[3], dt);
          cur += 3;
          scur += 1;
          break;
        }
        case T_CADYN: {
          // derivimplicit on a linear ODE: one Newton step of backward Euler is exact (L278)
          const double kappa = 1e4 * T.glob[0] / (2.0 * 96485.33212 * T.glob[1]);
          cai = (cai + dt * (-kappa * ica + T.glob[3] / T.glob[2])) / (1.0 + dt / T.glob[2]);
          tape[(size_t)cai_row * 32 + lane] = cai;
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
    const int c_next = (int)((sr + slen) / CH);
    if (b_free < c_next) {
      __syncwarp();
      if (lane == 0)
        for (int c = b_free; c < c_next; ++c)
          if (c + S < nsch) issue(scr, c + S, tc.n_srows);
      b_free = c_next;
    }
  }
  (void)v_root;
#undef CN_ROW
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
