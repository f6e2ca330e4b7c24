// cn_cell.cuh -- the on-chip window kernel ("every minimum spike
// delay interval"): ONE CTA KEEPS ONE CELL ON CHIP FOR A WHOLE MIN-DELAY WINDOW.
//
// No event can arrive sooner than the smallest NetCon delay after the spike that causes it, so
// for `nsteps` <= min-delay steps a cell depends on nothing but itself and on events whose spikes
// were recorded before the window (summed per (step, synapse) by deliver_window_kernel).  The CTA
// loads the cell once -- tree coefficients, voltages, parameters and states of every distributed
// mechanism, cai, and the cell's elimination plan -- into shared memory, runs the whole hot path
// nsteps times there:
//     point processes (events of the step, conductances; L64, L65) -> nrn_cur of the distributed
//     mechanisms (L65) -> Hines solve (L66) -> voltage update -> nrn_state (L67) -> threshold (L68)
// and writes voltages and states back once.  Between the load and the store nothing but the few
// synapse states of the cell, the delivered weights and the spike list touches L2 / HBM: the step
// is bound by the fp64 pipe and by the dependent chain of the elimination, not by memory.
//
// Elimination: the tree is cut into unbranched CHAINS (cn_finalize.hpp build_cell_plan); one
// thread eliminates a whole chain with the contribution to the parent travelling in registers
// (and the parent's v on the way back); the chains of one level of the tree of chains run side by
// side on the lanes of one warp, one barrier per level; where chains meet, the parent's chain
// sums its children's contributions in a fixed order (no atomics: runs are bit-reproducible).
// Every per-node array in shared memory is in PLAN ORDER -- the nodes of a chain side by side --
// so the chain loops address shared memory by a running index: no index loads on the chain.
//
// Used for models whose cells all sit on the warp-cooperative layout with one cell per warp and
// fit the device at once (configs 1 and 2 by default; option onchip=1 forces it for any model
// whose largest cell fits the shared memory of a CTA).  Gap junctions need the peer's voltage of
// every step and exclude this mode.
#pragma once
#include "cn_device.cuh"

namespace cn {

#ifdef CN_TRACE
__device__ long long g_cell_trace[16];
#define CN_CT(i) do { if (tid == 0 && blockIdx.x == 0) { const long long t_ = clock64(); g_cell_trace[i] += t_ - tprev; tprev = t_; } } while (0)
#else
#define CN_CT(i)
#endif

// the point processes of one cell for one step: events delivered at this step, conductance and
// current into the node's fixed-point accumulators PD / PR (several instances may sit on one node:
// shared-memory integer atomics, the sum does not depend on their order), state decay
template <int NT>
__device__ __forceinline__ void cell_point_processes(const DModel &M, const long long *ppq, int s,
                                                     int64_t k, double *PD, double *PR,
                                                     const double *V, int tid) {
  const double t_mid = ((double)k + 0.5) * M.dt;
  for (int t = 0; t < M.n_table; ++t) {
    const DTable &T = M.tab[t];
    if (!T.is_point) continue;
    const int64_t q0 = ppq[2 * t], q1 = ppq[2 * t + 1];
    double *dl0 = M.win_deliv ? M.win_deliv + (size_t)s * M.win_ninst + T.pp_goff : nullptr;
    for (int64_t q = q0 + tid; q < q1; q += NT) {
      const int nd = T.pp_local[q];
      double w = 0.0;
      if (dl0 && T.type != T_ICLAMP) {
        const double raw = dl0[q];
        if (fx_nonzero(raw)) {
          w = fxw_get(raw, M.fxw_inv);
          dl0[q] = 0.0;
        }
      }
      switch (T.type) {
        case T_EXPSYN: {
          double gg = T.state[0][q];
          if (w != 0.0) gg += w;
          if (gg != 0.0) {
            const double gs = gg * T.param[2][q];
            fx_add(&PD[nd], gs, M.overflow);
            fx_add(&PR[nd], gs * T.param[1][q], M.overflow);
            T.state[0][q] = decay(gg, T.param[0][q]);
          }
          break;
        }
        case T_EXP2SYN: {
          double a = T.state[0][q], b = T.state[1][q];
          if (w != 0.0) {
            const double wf = w * T.param[4][q];
            a += wf;
            b += wf;
          }
          if (a != 0.0 || b != 0.0) {
            const double gs = (b - a) * T.param[3][q];
            if (gs != 0.0) {
              fx_add(&PD[nd], gs, M.overflow);
              fx_add(&PR[nd], gs * T.param[2][q], M.overflow);
            }
            T.state[0][q] = decay(a, T.param[0][q]);
            T.state[1][q] = decay(b, T.param[1][q]);
          }
          break;
        }
        case T_ICLAMP: {
          const double del = T.param[0][q];
          if (t_mid >= del && t_mid < del + T.param[1][q])
            fx_add(&PR[nd], T.param[2][q] * T.param[3][q], M.overflow);
          break;
        }
        case T_AMPANMDA: {
          double a0 = T.state[0][q], a1 = T.state[1][q], a2 = T.state[2][q], a3 = T.state[3][q];
          if (w != 0.0) {
            const double wa = w * T.glob[7], wn = w * T.glob[8];
            a0 += wa;
            a1 += wa;
            a2 += wn;
            a3 += wn;
          }
          if (a0 != 0.0 || a1 != 0.0 || a2 != 0.0 || a3 != 0.0) {
            const double gs =
                ((a1 - a0) + T.glob[4] * (a3 - a2) * mgblock(V[nd], T.glob[5])) * T.param[0][q];
            fx_add(&PD[nd], gs, M.overflow);
            fx_add(&PR[nd], gs * T.glob[6], M.overflow);
            T.state[0][q] = decay(a0, T.glob[9]);
            T.state[1][q] = decay(a1, T.glob[10]);
            T.state[2][q] = decay(a2, T.glob[11]);
            T.state[3][q] = decay(a3, T.glob[12]);
          }
          break;
        }
        default: break;
      }
    }
  }
}

// Hines solve of one cell in shared memory (L66).  D / R come in as the assembled diagonal / right
// side and leave as back-substitution multipliers / the new voltages.  `st`: this thread's index
// among the SW solving threads (>= SW: not solving).
template <int NT>
__device__ __forceinline__ void cell_solve(const CellClass &cc, const CellSeg *segs,
                                           const int32_t *lvl, const uint16_t *child,
                                           const double *A, const double *B, double *D, double *R,
                                           double *CD, double *CR, int n, int st, int SW, int tid) {
  for (int L = 0; L < cc.n_lev; ++L) {
    const int s1 = lvl[L + 1];
    if (st < SW)
      for (int sg = lvl[L] + st; sg < s1; sg += SW) {
        const CellSeg S = segs[sg];
        const uint16_t *chn = child + S.child_off;
        double accD = 0.0, accR = 0.0;
        for (int c = 0; c < (int)S.nchild; ++c) {
          accD += CD[chn[c]];
          accR += CR[chn[c]];
        }
        // operands of the next node are fetched while the current one is on the dependent chain:
        // pivot -> reciprocal -> contribution (one DADD, MUFU + 3 DFMA, one DMUL)
        const int x0 = S.first, len = S.len;
        double d0 = D[x0], r0 = R[x0], a0 = A[x0], b0 = B[x0];
        for (int j = 0; j < len; ++j) {
          const int x = x0 + j, xn = j + 1 < len ? x + 1 : x;
          const double d1 = D[xn], r1 = R[xn], a1 = A[xn], b1 = B[xn];
          const double di = d0 + accD, ri = r0 + accR;
          const double ab = a0 * b0, ar = a0 * ri;
          const double rinv = rcp_chain(di);
          accD = -(ab * rinv);
          accR = -(ar * rinv);
          D[x] = b0 * rinv;  // back-substitution multiplier
          R[x] = ri * rinv;
          d0 = d1; r0 = r1; a0 = a1; b0 = b1;
        }
        CD[x0 + len - 1] = accD;
        CR[x0 + len - 1] = accR;
      }
    __syncthreads();
  }
  if (tid == 0) {  // the root is the last node of the plan
    const uint16_t *chn = child + cc.root_child_off;
    double accD = 0.0, accR = 0.0;
    for (int c = 0; c < cc.root_nchild; ++c) {
      accD += CD[chn[c]];
      accR += CR[chn[c]];
    }
    R[n - 1] = (R[n - 1] + accR) * rcp_fast(D[n - 1] + accD);
  }
  __syncthreads();
  for (int L = cc.n_lev - 1; L >= 0; --L) {
    const int s1 = lvl[L + 1];
    if (st < SW)
      for (int sg = lvl[L] + st; sg < s1; sg += SW) {
        const CellSeg S = segs[sg];
        double vp = R[S.par];
        const int x0 = S.first, len = S.len;
        int x = x0 + len - 1;
        double m0 = D[x], r0 = R[x];
        for (int j = len - 1; j >= 0; --j, --x) {
          const int xn = j > 0 ? x - 1 : x;
          const double m1 = D[xn], r1 = R[xn];
          vp = fma(-m0, vp, r0);
          R[x] = vp;
          m0 = m1; r0 = r1;
        }
      }
    __syncthreads();
  }
}

// NT threads per CTA: 64 for small cells (more CTAs per SM), up to 256 for large ones
template <int NT>
__global__ void __launch_bounds__(NT)
    cell_window_kernel(const __grid_constant__ DModel M, int64_t k0, int nsteps, int64_t trace_row0) {
  extern __shared__ double csm[];
  const int tid = threadIdx.x;
  const double dt = M.dt;
  // which warp of this CTA runs the elimination: CTAs that arrive on the same SM take turns, so
  // that their solving warps sit on different quarters (schedulers, fp64 pipes) of the SM
  __shared__ int swarp_s;
  __shared__ int cnt_s[CN_MAX_TABLES];          // instances per table of this cell
  __shared__ long long ppq_s[2 * CN_MAX_TABLES];  // point-process instance range per table
  if (tid == 0) {
    uint32_t smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    swarp_s = (int)(atomicAdd(M.cwin_smctr + (smid & 255u), 1u) % (uint32_t)(NT / 32));
  }
  __syncthreads();
  // the solving threads: the 32 lanes of warp `swarp` first, then those of the next warp
  const int st = (tid - swarp_s * 32 + NT) % NT;
  const int SW = NT < 64 ? NT : 64;
  for (int g = blockIdx.x; g < M.n_group; g += gridDim.x) {
    const GroupInfo gi = M.grp[g];
    const ClassInfo ci = M.cls[gi.cls];
    const CellClass &cc = M.ccls[gi.cls];
    const int n = ci.n;
    const int64_t ab = gi.ab_base;
    // shared memory, per node in plan order: A B DS RS V D R CD CR [I] [CAI]; then the
    // mechanism block; then the plan: chains, levels, child positions, node positions per table
    double *A = csm, *B = A + n, *DS = B + n, *RS = DS + n, *V = RS + n, *D = V + n, *R = D + n;
    double *CD = R + n, *CR = CD + n;  // contribution of the last node of a chain to its parent
    double *nx = CR + n;
    double *I = nullptr, *CAI = nullptr;
    if (ci.needs_ica) { I = nx; nx += n; }
    if (M.cai) { CAI = nx; nx += n; }
    double *MB = nx;
    CellSeg *segs = reinterpret_cast<CellSeg *>(MB + cc.mech_doubles);
    int32_t *lvl = reinterpret_cast<int32_t *>(segs + cc.n_seg);
    uint16_t *child = reinterpret_cast<uint16_t *>(lvl + cc.n_lev + 1);
    uint16_t *dist = child + cc.n_child;
    __syncthreads();  // (the previous cell's stores are done with shared memory)
    // ---- load the cell ---------------------------------------------------------------------------
    {
      const int32_t *__restrict__ pno = M.cplan_noff + cc.noff_off;
      for (int i = tid; i < n; i += NT) {
        const int64_t q = ab + pno[i];
        A[i] = M.a_s[q];
        B[i] = M.b_s[q];
        DS[i] = fabs(M.dstat[q]);  // (a negative static diagonal marks nodes with point processes)
        RS[i] = M.rstat[q];
        V[i] = M.v[q];
        if (CAI) CAI[i] = M.cai[q];
      }
      for (int i = tid; i < cc.n_seg; i += NT) segs[i] = M.cseg[cc.seg_off + i];
      for (int i = tid; i <= cc.n_lev; i += NT) lvl[i] = M.cseg_lvl[cc.lvl_off + i];
      for (int i = tid; i < cc.n_child; i += NT) child[i] = M.cseg_child[cc.child_off + i];
      for (int i = tid; i < cc.n_dist; i += NT) dist[i] = M.cdist[cc.dist_base + i];
      for (int t = tid; t < M.n_table; t += NT) {
        const DTable &T = M.tab[t];
        cnt_s[t] = T.is_point || T.type == T_PAS ? 0 : T.cls_cnt[gi.cls];
        ppq_s[2 * t] = T.is_point ? T.pp_first[g] : 0;
        ppq_s[2 * t + 1] = T.is_point ? T.pp_first[g + 1] : 0;
      }
    }
    __syncthreads();
    for (int t = 0; t < M.n_table; ++t) {
      const DTable &T = M.tab[t];
      const int cnt = cnt_s[t];
      if (cnt == 0 || T.type == T_CADYN) continue;
      const int64_t ib = T.grp_instbase[g];
      double *dst = MB + cc.mech_off[t];
      for (int j = 0; j < T.n_param; ++j, dst += cnt)
        for (int i = tid; i < cnt; i += NT) dst[i] = T.param[j][ib + i];
      for (int j = 0; j < T.n_state; ++j, dst += cnt)
        for (int i = tid; i < cnt; i += NT) dst[i] = T.state[j][ib + i];
    }
    const int pc = gi.cell_base;
    bool flag = false;
    double thr = 0.0;
    if (tid == 0) {
      flag = M.flag[pc] != 0;
      thr = M.thr[pc];
    }
    bool any_pp = false;
    for (int t = 0; t < M.n_table; ++t) any_pp = any_pp || ppq_s[2 * t + 1] > ppq_s[2 * t];
    GroupView gv;
    gv.ab = 0;
    gv.noff = nullptr;
    gv.G = 1;
    gv.lgG = 0;
    gv.direct = true;
    __syncthreads();
#ifdef CN_TRACE
    long long tprev = clock64();
#endif
    for (int s = 0; s < nsteps; ++s) {
      const int64_t k = k0 + s;
      // ---- the system starts from the static terms: D = static diagonal, R = v + static rhs -------
      for (int i = tid; i < n; i += NT) {
        D[i] = DS[i];
        R[i] = V[i] + RS[i];
        CD[i] = 0.0;  // (the chains' contribution rows double as the point processes' accumulators)
        CR[i] = 0.0;
        if (I) I[i] = 0.0;
      }
      __syncthreads();
      CN_CT(0);
      if (any_pp) {
        cell_point_processes<NT>(M, ppq_s, s, k, CD, CR, V, tid);
        __syncthreads();
        for (int i = tid; i < n; i += NT) {
          D[i] += fx_get(CD[i]);
          R[i] += fx_get(CR[i]);
        }
        __syncthreads();
      }
      CN_CT(1);
      // ---- nrn_cur of the distributed mechanisms (one instance per node and table) ----------------
      for (int t = 0; t < M.n_table; ++t) {
        const DTable &T = M.tab[t];
        const int cnt = cnt_s[t];
        if (cnt == 0 || T.type == T_CADYN) continue;
        double *par[CN_MAX_PARAM], *sta[CN_MAX_STATE];
        double *p = MB + cc.mech_off[t];
#pragma unroll
        for (int j = 0; j < CN_MAX_PARAM; ++j) par[j] = p + (j < T.n_param ? j : 0) * cnt;
#pragma unroll
        for (int j = 0; j < CN_MAX_STATE; ++j) sta[j] = p + (T.n_param + (j < T.n_state ? j : 0)) * cnt;
        cur_distributed(T, par, sta, 0, cnt, gv, dist + cc.dist_off[t], D, R, I, V, tid, NT);
        __syncthreads();
      }
      CN_CT(2);
      cell_solve<NT>(cc, segs, lvl, child, A, B, D, R, CD, CR, n, st, SW, tid);
      CN_CT(3);
      // ---- voltage update, threshold at the root (L66, L68), probes -------------------------------
      for (int i = tid; i < n; i += NT) V[i] = R[i];
      if (tid == 0) {
        const bool above = R[n - 1] > thr;
        if (above && !flag) {
          const unsigned long long pos = atomicAdd(M.n_sp, 1ull);
          if ((int64_t)pos < M.sp_cap) {
            M.sp_gid[pos] = M.gid_of_pcell[pc];
            M.sp_step[pos] = k + 1;
          } else {
            *M.overflow = 1;
          }
        }
        flag = above;
      }
      if (M.wp_first) {
        const int64_t row = trace_row0 + s;
        if (row < M.trace_cap)
          for (int p = M.wp_first[g] + tid; p < M.wp_first[g + 1]; p += NT)
            M.trace[row * M.n_probe + M.wp_col[p]] = R[M.wp_pos[p]];
      }
      CN_CT(4);
      // ---- nrn_state with the new v (L67), tables in description order -----------------------------
      for (int t = 0; t < M.n_table; ++t) {
        const DTable &T = M.tab[t];
        const int cnt = cnt_s[t];
        if (cnt == 0 || (T.n_state == 0 && T.type != T_CADYN)) continue;
        double *par[CN_MAX_PARAM], *sta[CN_MAX_STATE];
        double *p = MB + cc.mech_off[t];
#pragma unroll
        for (int j = 0; j < CN_MAX_PARAM; ++j) par[j] = p + (j < T.n_param ? j : 0) * cnt;
#pragma unroll
        for (int j = 0; j < CN_MAX_STATE; ++j) sta[j] = p + (T.n_param + (j < T.n_state ? j : 0)) * cnt;
        state_distributed(T, par, sta, 0, cnt, gv, dist + cc.dist_off[t], R, CAI, I, tid, dt, M.q10, NT);
        __syncthreads();  // (SK reads the cai that the cai dynamics of an earlier table wrote)
      }
      __syncthreads();
      CN_CT(5);
    }

    // ---- store the cell -----------------------------------------------------------------------------
    {
      const int32_t *__restrict__ pno = M.cplan_noff + cc.noff_off;
      for (int i = tid; i < n; i += NT) {
        const int64_t q = ab + pno[i];
        M.v[q] = V[i];
        if (CAI) M.cai[q] = CAI[i];
      }
    }
    for (int t = 0; t < M.n_table; ++t) {
      const DTable &T = M.tab[t];
      const int cnt = cnt_s[t];
      if (cnt == 0 || T.n_state == 0) continue;
      const int64_t ib = T.grp_instbase[g];
      const double *src = MB + cc.mech_off[t] + (size_t)T.n_param * cnt;
      for (int j = 0; j < T.n_state; ++j, src += cnt)
        for (int i = tid; i < cnt; i += NT) T.state[j][ib + i] = src[i];
    }
    if (tid == 0) M.flag[pc] = (unsigned char)flag;
  }
}

}  // namespace cn
