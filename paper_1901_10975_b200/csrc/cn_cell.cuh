// cn_cell.cuh -- the on-chip window kernel ("every minimum spike
// delay interval"): ONE CTA KEEPS ONE CELL ON CHIP FOR A WHOLE MIN-DELAY WINDOW.
//
// No event can arrive sooner than the smallest NetCon delay after the spike that causes it, so
// for `nsteps` <= min-delay steps a cell depends on nothing but itself and on events whose spikes
// were recorded before the window (summed per (step, synapse) by deliver_window_kernel).  The CTA
// loads the cell once -- tree coefficients, voltages, parameters and states of every distributed
// mechanism, cai -- into shared memory, runs the whole hot path nsteps times there:
//     point processes (events of the step, conductances; L64, L65) -> nrn_cur of the distributed
//     mechanisms (L65) -> Hines solve (L66) -> voltage update -> nrn_state (L67) -> threshold (L68)
// and writes voltages and states back once.  Between the load and the store nothing but the few
// synapse states of the cell, the delivered weights and the spike list touches L2 / HBM: the step
// is bound by the fp64 pipe and by the dependent chain of the elimination, not by memory.
// All warps share the mechanism work (one thread per instance) and the elimination (one thread per
// unbranched chain of the tree, the chains of one level side by side).
// Used for models whose cells all sit on the warp-cooperative layout with one cell per warp and
// fit the device at once (configs 1 and 2; option onchip=1 forces it for any model whose largest
// cell fits the shared memory of a CTA).  Gap junctions need the peer's voltage of every step and
// exclude this mode.
#pragma once
#include "cn_device.cuh"

namespace cn {

// NT threads per CTA: 64 for small cells (more CTAs per SM), up to 256 for large ones
template <int NT>
__global__ void __launch_bounds__(NT)
    cell_window_kernel(const __grid_constant__ DModel M, int64_t k0, int nsteps, int64_t trace_row0) {
  extern __shared__ double csm[];
  const int tid = threadIdx.x;
  const double dt = M.dt;
  for (int g = blockIdx.x; g < M.n_group; g += gridDim.x) {
    const GroupInfo gi = M.grp[g];
    const ClassInfo ci = M.cls[gi.cls];
    const CellClass &cc = M.ccls[gi.cls];
    const int n = ci.n;
    const int64_t ab = gi.ab_base;
    const int32_t *__restrict__ noff = M.node_off + ci.nodeoff_off;
    // shared memory: A B DS RS V D R CD CR [I] [CAI] by local node, then the mechanism block
    double *A = csm, *B = A + n, *DS = B + n, *RS = DS + n, *V = RS + n, *D = V + n, *R = D + n;
    double *CD = R + n, *CR = CD + n;  // contribution of the last node of a chain to its parent
    double *nx = CR + n;
    double *I = nullptr, *CAI = nullptr;
    if (ci.needs_ica) { I = nx; nx += n; }
    if (M.cai) { CAI = nx; nx += n; }
    double *MB = nx;
    __syncthreads();  // (the previous cell's stores are done with shared memory)
    // ---- load the cell ---------------------------------------------------------------------------
    for (int i = tid; i < n; i += NT) {
      const int64_t q = ab + noff[i];
      A[i] = M.a_s[q];
      B[i] = M.b_s[q];
      DS[i] = fabs(M.dstat[q]);  // (a negative static diagonal marks nodes with point processes)
      RS[i] = M.rstat[q];
      V[i] = M.v[q];
      if (CAI) CAI[i] = M.cai[q];
    }
    for (int t = 0; t < M.n_table; ++t) {
      const DTable &T = M.tab[t];
      if (T.is_point || T.type == T_PAS) continue;
      const int cnt = T.cls_cnt[gi.cls];
      if (cnt == 0) continue;
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
    GroupView gv;
    gv.ab = 0;
    gv.noff = nullptr;
    gv.G = 1;
    gv.lgG = 0;
    gv.direct = true;
    __syncthreads();

    for (int s = 0; s < nsteps; ++s) {
      const int64_t k = k0 + s;
      // ---- zero the system --------------------------------------------------------------------
      for (int i = tid; i < n; i += NT) {
        D[i] = 0.0;
        R[i] = 0.0;
        if (I) I[i] = 0.0;
      }
      __syncthreads();
      // ---- point processes of the cell: events of this step, conductance / current, decay --------
      // (several instances may sit on one node: shared-memory atomics)
      {
        const double t_mid = ((double)k + 0.5) * dt;
        for (int t = 0; t < M.n_table; ++t) {
          const DTable &T = M.tab[t];
          if (!T.is_point) continue;
          const int64_t q0 = T.pp_first[g], q1 = T.pp_first[g + 1];
          double *dl0 = M.win_deliv ? M.win_deliv + (size_t)s * M.win_ninst + T.pp_goff : nullptr;
          for (int64_t q = q0 + tid; q < q1; q += NT) {
            const int nd = T.pp_local[q];
            double w = 0.0;
            if (dl0 && T.type != T_ICLAMP) {
              w = dl0[q];
              if (w != 0.0) dl0[q] = 0.0;
            }
            switch (T.type) {
              case T_EXPSYN: {
                double gg = T.state[0][q];
                if (w != 0.0) gg += w;
                if (gg != 0.0) {
                  const double gs = gg * T.param[2][q];
                  atomicAdd(&D[nd], gs);
                  atomicAdd(&R[nd], gs * T.param[1][q]);
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
                    atomicAdd(&D[nd], gs);
                    atomicAdd(&R[nd], gs * T.param[2][q]);
                  }
                  T.state[0][q] = decay(a, T.param[0][q]);
                  T.state[1][q] = decay(b, T.param[1][q]);
                }
                break;
              }
              case T_ICLAMP: {
                const double del = T.param[0][q];
                if (t_mid >= del && t_mid < del + T.param[1][q])
                  atomicAdd(&R[nd], T.param[2][q] * T.param[3][q]);
                break;
              }
              case T_AMPANMDA: {
                double a0 = T.state[0][q], a1 = T.state[1][q], a2 = T.state[2][q],
                       a3 = T.state[3][q];
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
                  atomicAdd(&D[nd], gs);
                  atomicAdd(&R[nd], gs * T.glob[6]);
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
      __syncthreads();
      // ---- nrn_cur of the distributed mechanisms (one instance per node and table) ----------------
      for (int t = 0; t < M.n_table; ++t) {
        const DTable &T = M.tab[t];
        if (T.is_point || T.type == T_PAS || T.type == T_CADYN) continue;
        const int cnt = T.cls_cnt[gi.cls];
        if (cnt == 0) continue;
        double *par[CN_MAX_PARAM], *st[CN_MAX_STATE];
        double *p = MB + cc.mech_off[t];
#pragma unroll
        for (int j = 0; j < CN_MAX_PARAM; ++j) par[j] = p + (j < T.n_param ? j : 0) * cnt;
#pragma unroll
        for (int j = 0; j < CN_MAX_STATE; ++j) st[j] = p + (T.n_param + (j < T.n_state ? j : 0)) * cnt;
        cur_distributed(T, par, st, 0, cnt, gv, M.dist_nodes + T.cls_nodeoff[gi.cls], D, R, I, V,
                        tid, NT);
        __syncthreads();
      }
      // ---- Hines solve (L66): one thread per unbranched chain, one barrier per level of the tree
      // of chains (cn_finalize.hpp build_cell_segments).  Along a chain the contribution to the
      // parent, and on the way back the parent's v, travel in registers; where chains meet, the
      // parent's chain sums the contributions of its children in a fixed order. ----------------------
      {
        const CellSeg *__restrict__ segs = M.cseg + cc.seg_off;
        const int32_t *__restrict__ lvl = M.cseg_lvl + cc.lvl_off;
        for (int L = 0; L < cc.n_lev; ++L) {
          const int s1 = lvl[L + 1];
          for (int sg = lvl[L] + tid; sg < s1; sg += NT) {
            const CellSeg S = segs[sg];
            const uint16_t *__restrict__ nd = M.cseg_nodes + S.node_off;
            const uint16_t *__restrict__ chn = M.cseg_child + S.child_off;
            double accD = 0.0, accR = 0.0;
            for (int c = 0; c < (int)S.nchild; ++c) {
              accD += CD[chn[c]];
              accR += CR[chn[c]];
            }
            int x = nd[0];
            for (int j = 0; j < (int)S.len; ++j) {
              const int xn = j + 1 < (int)S.len ? nd[j + 1] : x;
              const double di = (D[x] + DS[x]) + accD, ri = (R[x] + (V[x] + RS[x])) + accR;
              const double a = A[x], b = B[x];
              const double rinv = rcp_chain(di);
              const double f = a * rinv;
              D[x] = b * rinv;  // back-substitution multiplier
              R[x] = ri * rinv;
              accD = -(f * b);
              accR = -(f * ri);
              if (j + 1 == (int)S.len) {
                CD[x] = accD;
                CR[x] = accR;
              }
              x = xn;
            }
          }
          __syncthreads();
        }
        if (tid == 0) {
          const uint16_t *__restrict__ chn = M.cseg_child + cc.root_child_off;
          double accD = 0.0, accR = 0.0;
          for (int c = 0; c < cc.root_nchild; ++c) {
            accD += CD[chn[c]];
            accR += CR[chn[c]];
          }
          R[0] = ((R[0] + (V[0] + RS[0])) + accR) * rcp_fast((D[0] + DS[0]) + accD);
        }
        __syncthreads();
        for (int L = cc.n_lev - 1; L >= 0; --L) {
          const int s1 = lvl[L + 1];
          for (int sg = lvl[L] + tid; sg < s1; sg += NT) {
            const CellSeg S = segs[sg];
            const uint16_t *__restrict__ nd = M.cseg_nodes + S.node_off;
            double vp = R[S.par];
            for (int j = (int)S.len - 1; j >= 0; --j) {
              const int x = nd[j];
              vp = fma(-D[x], vp, R[x]);
              R[x] = vp;
            }
          }
          __syncthreads();
        }
      }
      // ---- voltage update, threshold at the root (L66, L68), probes -------------------------------
      for (int i = tid; i < n; i += NT) V[i] = R[i];
      if (tid == 0) {
        const bool above = R[0] > thr;
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
      // ---- nrn_state with the new v (L67), tables in description order -----------------------------
      for (int t = 0; t < M.n_table; ++t) {
        const DTable &T = M.tab[t];
        if (T.is_point || (T.n_state == 0 && T.type != T_CADYN)) continue;
        const int cnt = T.cls_cnt[gi.cls];
        if (cnt == 0) continue;
        double *par[CN_MAX_PARAM], *st[CN_MAX_STATE];
        double *p = MB + cc.mech_off[t];
#pragma unroll
        for (int j = 0; j < CN_MAX_PARAM; ++j) par[j] = p + (j < T.n_param ? j : 0) * cnt;
#pragma unroll
        for (int j = 0; j < CN_MAX_STATE; ++j) st[j] = p + (T.n_param + (j < T.n_state ? j : 0)) * cnt;
        state_distributed(T, par, st, 0, cnt, gv, M.dist_nodes + T.cls_nodeoff[gi.cls], R, CAI, I,
                          tid, dt, M.q10, NT);
        __syncthreads();  // (SK reads the cai that the cai dynamics of an earlier table wrote)
      }
      __syncthreads();
    }

    // ---- store the cell -----------------------------------------------------------------------------
    for (int i = tid; i < n; i += NT) {
      const int64_t q = ab + noff[i];
      M.v[q] = V[i];
      if (CAI) M.cai[q] = CAI[i];
    }
    for (int t = 0; t < M.n_table; ++t) {
      const DTable &T = M.tab[t];
      if (T.is_point || T.n_state == 0) continue;
      const int cnt = T.cls_cnt[gi.cls];
      if (cnt == 0) continue;
      const int64_t ib = T.grp_instbase[g];
      const double *src = MB + cc.mech_off[t] + (size_t)T.n_param * cnt;
      for (int j = 0; j < T.n_state; ++j, src += cnt)
        for (int i = tid; i < cnt; i += NT) T.state[j][ib + i] = src[i];
    }
    if (tid == 0) M.flag[pc] = (unsigned char)flag;
  }
}

}  // namespace cn
