// cn_tape.cuh -- the interleaved step kernel: 32 cells of one shape class are integrated for one
// dt with ONE LANE PER CELL ("one cell per thread", Fig. 5D), re-designed for B200:
//
//   * Every per-node quantity of the 32 cells is a ROW of 32 doubles (256 B).  All rows of a group
//     are laid out in the order they are consumed -- a TAPE: per node a, b, static diagonal,
//     static rhs, v (+ two dynamic rows for point processes); per node with distributed
//     mechanisms a second record with a copy of v and the parameter / state rows.  The kernel
//     never computes an address from the tree: it reads the tape front to back.
//   * One CTA (W = 8 warps) owns one group at a time and takes groups until none is left
//     (persistent).  The linear system of the group stays ON CHIP for the whole step:
//     triangularisation (L66) leaves (multiplier, reduced rhs) of every node there,
//     back-substitution reads them back.  Rows that only their own warp touches live in TENSOR
//     MEMORY (tcgen05.st / tcgen05.ld, a per-lane scratchpad), rows where several warps meet in
//     shared memory; that leaves room for two CTAs per SM.  Nothing but the tape is read from HBM
//     and nothing but v and the states is written.
//   * The tree is compiled by the host into W record lists (a static schedule of the elimination
//     over W warps, children before parents, L196).  A chain hands its contribution to the parent
//     in REGISTERS; at a branch point the contributions meet in the parent's system row.  Warps
//     synchronise only through mbarriers in shared memory (WAIT records / signal flags).
//   * Each warp streams its own segment of the tape through a shared-memory ring with 1-D TMA bulk
//     copies (cp.async.bulk.shared.global + mbarrier complete_tx), S chunks of CH rows in flight,
//     issued by one lane; the ring of a warp that has finished its part of a group already loads
//     the next group while the back-substitution runs.
//   * nrn_state (L67) of step k is evaluated at the start of step k+1, in the mechanism record,
//     just before nrn_cur (L65) needs the states: same arithmetic on the same values (the new v
//     and the old states), but the states are read and written once per step and the
//     back-substitution carries no mechanism work.  cn_get_state runs the pending update first.
//   * One launch integrates a WINDOW of up to min-delay steps (L62): (step, group) work items are
//     handed out by a ticket counter, a group's next step may run on another SM once the previous
//     one is published (release / acquire through L2).  Events and point processes of the window
//     are prepared by deliver_window_kernel / pp_window_kernel (cn_device.cuh), probed voltages
//     are recorded at the end of every (step, group) item; with cells on the other kernel or
//     point processes that depend on v: one launch per dt, pp_step_kernel in front.
//   * Control is uniform across a warp; lanes never diverge.
// Host side: cn_tape_program.hpp compiles the per-class programs; DESIGN.md 5.1 has the rationale
// and profiles/r01_README.md the measurements behind every choice.
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
__device__ __forceinline__ uint4 lds_u4(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
               : "r"(addr));
  return v;
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
// Signals between the warps of a CTA: every record that another warp waits for arrives on an
// mbarrier of its own after its shared-memory writes (release; all lanes write, __syncwarp, one
// lane arrives); the waiting warp sleeps in mbarrier.try_wait (acquire) instead of spinning on a
// flag, which would take issue slots from the warps that work.  (Plain volatile flags are NOT
// enough either: measured, the rows can then be read before they are written.)
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// kernel modes: TM_ADVANCE: the states on the tape still wait for nrn_state of the previous step;
// TM_FLUSH: apply that update and nothing else; TM_WINDOW: one launch integrates `nsteps` steps,
// work items (step, group) are handed out by a ticket counter (see the kernel)
enum { TM_ADVANCE = 1, TM_FLUSH = 2, TM_WINDOW = 4 };

// One mechanism record: nrn_state of the previous step (if `mode & TM_ADVANCE`: the states on the
// tape are still those the previous nrn_cur used) followed by nrn_cur of this step with the
// advanced states.  rb = the record in the ring (this lane's column), trec = the same record on
// the tape.  Row order: v copy, [cai], [ica of the previous step], then per table its parameter
// and state rows.  Returns the row-normalised conductance / current sums in gD, gR.
__device__ __forceinline__ void mech_record(const DModel &M, const unsigned char *rb,
                                            double *__restrict__ trec, uint32_t fl,
                                            uint32_t mask, int mode, double dt, double q10dt,
                                            double &gD, double &gR) {
#define CN_RD(base, i) (*reinterpret_cast<const double *>((base) + (uint32_t)(i) * 256u))
  const bool adv = mode & TM_ADVANCE;
  const double v = CN_RD(rb, 0);
  uint32_t cur = 1, cai_row = 0, ica_row = 0;
  double cai = 0.0, ica_prev = 0.0, ica = 0.0;
  if (fl & RM_HAS_CAI) {
    cai = CN_RD(rb, cur);
    cai_row = cur++;
  }
  if (fl & RM_NEED_ICA) {
    ica_prev = CN_RD(rb, cur);
    ica_row = cur++;
  }
  gD = 0.0;
  gR = 0.0;
  for (uint32_t mk = mask; mk; mk &= mk - 1) {
    const DTable &T = M.tab[__ffs(mk) - 1];
    const unsigned char *mr = rb + cur * 256u;
    switch (T.type) {
      case T_HH: {
        double m = CN_RD(mr, 5), h = CN_RD(mr, 6), nn = CN_RD(mr, 7);
        if (adv) {
          hh_advance<false>(v, q10dt, m, h, nn);
          trec[(cur + 5) * 32] = m;
          trec[(cur + 6) * 32] = h;
          trec[(cur + 7) * 32] = nn;
        }
        const double invc = CN_RD(mr, 4);
        const double gna = CN_RD(mr, 0) * m * m * m * h;
        const double n2 = nn * nn;
        const double gk = CN_RD(mr, 1) * n2 * n2;
        const double gl = CN_RD(mr, 2);
        gD += (gna + gk + gl) * invc;
        gR += (gna * T.glob[0] + gk * T.glob[1] + gl * CN_RD(mr, 3)) * invc;
        cur += 8;
        break;
      }
      case T_HHFORM: {
        double ms = CN_RD(mr, 2), hs = CN_RD(mr, 3);
        if (adv) {
          double xinf, xtau;
          if ((int)T.glob[0] > 0) {
            hhform_gate(v, T.glob + 4, xinf, xtau);
            ms = cnexp(ms, xinf, xtau, dt);
            trec[(cur + 2) * 32] = ms;
          }
          if ((int)T.glob[1] > 0) {
            hhform_gate(v, T.glob + 10, xinf, xtau);
            hs = cnexp(hs, xinf, xtau, dt);
            trec[(cur + 3) * 32] = hs;
          }
        }
        const double g = CN_RD(mr, 0) * ipow(ms, (int)T.glob[0]) * ipow(hs, (int)T.glob[1]);
        const double invc = CN_RD(mr, 1);
        gD += g * invc;
        gR += g * T.glob[2] * invc;
        if (T.glob[3] != 0.0) ica += g * (v - T.glob[2]);
        cur += 4;
        break;
      }
      case T_SK: {
        double z = CN_RD(mr, 2);
        if (adv) {
          const double ca = cai < 1e-9 ? 1e-9 : cai;
          const double zinf = 1.0 / (1.0 + pow(T.glob[1] / ca, T.glob[2]));
          z = cnexp(z, zinf, T.glob[3], dt);
          trec[(cur + 2) * 32] = z;
        }
        const double g = CN_RD(mr, 0) * z;
        const double invc = CN_RD(mr, 1);
        gD += g * invc;
        gR += g * T.glob[0] * invc;
        cur += 3;
        break;
      }
      case T_CADYN: {
        // derivimplicit on a linear ODE: one Newton step of backward Euler is exact (L278)
        if (adv) {
          const double kappa = 1e4 * T.glob[0] / (2.0 * 96485.33212 * T.glob[1]);
          cai = (cai + dt * (-kappa * ica_prev + T.glob[3] / T.glob[2])) / (1.0 + dt / T.glob[2]);
          trec[cai_row * 32] = cai;
        }
        break;
      }
      default: break;  // PAS is folded into the static rows
    }
  }
  if ((fl & RM_NEED_ICA) && !(mode & TM_FLUSH)) trec[ica_row * 32] = ica;
#undef CN_RD
}

// One CTA = W warps = one group of 32 cells at a time (persistent over groups).  See the header
// of this file and the record layout in cn_device.cuh.
// Shared memory: W rings of S stages x CH rows | system: tape_sys_cap x (32 + 32) doubles | one
// or two program buffers of tape_prog_cap records | W*S + 2 + tape_bar_cap mbarriers | TMEM base.
// Tensor memory as a per-lane scratchpad (Blackwell: 512 columns x 128 lanes x 32 bit per SM; a
// warp addresses the 32 lanes of its quarter, thread i <-> lane i): (multiplier, reduced rhs) of a
// plain chain node = 4 columns.  SASS: STTM / LDTM.
__device__ __forceinline__ void tm_store2(uint32_t taddr, double a, double b) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr),
               "r"(__double2loint(a)), "r"(__double2hiint(a)), "r"(__double2loint(b)),
               "r"(__double2hiint(b))
               : "memory");
}
__device__ __forceinline__ void tm_load2(uint32_t taddr, double &a, double &b) {
  uint32_t r0, r1, r2, r3;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
               : "r"(taddr)
               : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
  a = __hiloint2double((int)r1, (int)r0);
  b = __hiloint2double((int)r3, (int)r2);
}
constexpr int CN_TMEM_COLS = 256;  // per CTA: two CTAs share the 512 columns of an SM

#ifdef CN_TRACE
__device__ long long g_trace[148 * 16 * 8 * 8];
#define CN_TR(i) if (lane == 0 && it < 8 && blockIdx.x < 148) g_trace[((blockIdx.x * 16 + warp) * 8 + it) * 8 + (i)] = clock64()
// per record of the backward (B) / forward (F) sweep of item 3 of the first 8 CTAs: clock, record word
__device__ long long g_trace2[2 * 8 * 16 * 128 * 2];
#define CN_TR2(dir, j0, j, ey) if (lane == 0 && it == 3 && blockIdx.x < 8 && (j) - (j0) < 128) { \
    long long *q_ = g_trace2 + ((((dir) * 8 + blockIdx.x) * 16 + warp) * 128 + ((j) - (j0))) * 2; \
    q_[0] = clock64(); q_[1] = (long long)(ey); }
#else
#define CN_TR(i)
#define CN_TR2(dir, j0, j, ey)
#endif
template <int MAXT>
__global__ void __launch_bounds__(MAXT, 512 / MAXT) tape_step_kernel(const __grid_constant__ DModel M,
                                                          int64_t k, int mode, int nsteps) {
  extern __shared__ __align__(128) unsigned char sm_raw[];
  if (k < 0) k = M.step_ctr[0] - k - 1;  // replayed graph: the device counter + offset
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int W = M.tape_W, S = M.tape_S, CH = M.tape_CH;
  const uint32_t RB = (uint32_t)(S * CH) * 256u;  // ring bytes per warp
  const uint32_t lane8 = (uint32_t)lane * 8u;
  const unsigned char *ringc = sm_raw + (size_t)warp * RB + lane8;  // this lane's column
  double *sys_l = reinterpret_cast<double *>(sm_raw + (size_t)W * RB) + lane;
  uint4 *progbuf = reinterpret_cast<uint4 *>(sm_raw + (size_t)W * RB +
                                             (size_t)M.tape_sys_cap * 512);
  const int PB = M.tape_pbuf;  // program buffers: 2 (the next program loads during the group) or 1
  uint64_t *mbar_all = reinterpret_cast<uint64_t *>(progbuf + (size_t)PB * M.tape_prog_cap);
  const uint32_t ring_s = smem_u32(sm_raw + (size_t)warp * RB);
  const uint32_t bar_s = smem_u32(mbar_all + (size_t)warp * S);  // S ring barriers of this warp
  const uint32_t pbar_s = smem_u32(mbar_all + (size_t)W * S);    // 2 program barriers
  const int NB = M.tape_bar_cap;  // signal mbarriers: one per signalling record of a program
  const uint32_t sbar_s = smem_u32(mbar_all + (size_t)W * S + 2);
  const double dt = M.dt;
  const double q10dt = M.q10 * dt;
  const bool flush = mode & TM_FLUSH;
  const int ngrp = M.n_tgroup;

#define CN_RD(base, i) (*reinterpret_cast<const double *>((base) + (uint32_t)(i) * 256u))

  if (threadIdx.x == 0) {
    for (int s = 0; s < W * S + 2 + NB; ++s) mbar_init(smem_u32(mbar_all + s), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (blockIdx.x >= ngrp) return;
  uint32_t *tm_base_s = reinterpret_cast<uint32_t *>(mbar_all + (size_t)W * S + 2 + NB);
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                     smem_u32(tm_base_s)),
                 "n"(CN_TMEM_COLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  // this warp's lanes of tensor memory (quarter warp % 4); its slots start at TapeTask::tm_base
  const uint32_t tm_warp = *tm_base_s + (((uint32_t)(warp & 3) * 32u) << 16);

  // ring: chunk c of a segment (whole records, at most CH rows) goes to stage c % S; the program's
  // CHUNK records say when a stage is free again and what to request into it
  uint32_t phase = 0;  // bit s: parity the next wait on stage s looks for
  const double *seg = nullptr;
  auto issue = [&](uint32_t stage, uint32_t row, uint32_t rows) {  // one lane
    const uint32_t bytes = rows * 256u;
    mbar_expect_tx(bar_s + 8 * stage, bytes);
    bulk_g2s(ring_s + stage * (uint32_t)(CH * 256), seg + (size_t)row * 32, bytes,
             bar_s + 8 * stage);
  };
  // rows [r0, r1) of the segment towards L2, so that the bulk copy that follows PF rows later
  // finds them there (the ring holds two chunks per warp: its refills are latency-bound)
  uint32_t seg_rows = 0;
  const uint32_t PF = (uint32_t)M.tape_pf;
  auto prefetch = [&](uint32_t r0, uint32_t r1) {  // one lane
    r1 = min(r1, seg_rows);
    if (r0 < r1)
      asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(seg + (size_t)r0 * 32),
                   "r"((r1 - r0) * 256u)
                   : "memory");
  };
  auto start_segment = [&](const TapeGroup &g, const TapeTask &t) {
    seg = M.tape + g.tape_base + (size_t)t.row0 * 32;
    seg_rows = t.nrows;
    if (lane == 0) {
      uint32_t row = 0;
      for (int c = 0; c < S && c < t.nchunk; ++c) {
        const uint32_t rows = (t.head >> (8 * c)) & 255u;
        issue((uint32_t)c, row, rows);
        row += rows;
      }
      if (PF) prefetch(row, row + PF);
    }
  };
  auto load_program = [&](const TapeClass &c, int buf) {  // one thread
    const uint32_t bytes = (uint32_t)c.prog_len * 16u;
    mbar_expect_tx(pbar_s + 8 * buf, bytes);
    bulk_g2s(smem_u32(progbuf + (size_t)buf * M.tape_prog_cap), M.prog + c.prog_off, bytes,
             pbar_s + 8 * buf);
  };

  // Work items.  Per-step mode: item = group, CTA b takes b, b + gridDim.x, ...  Window mode: item
  // i = step * ngrp + group, handed out by a global ticket counter (any CTA, any order of
  // arrival); item (s, g) may start once (s - 1, g) is complete (win_done[g] >= s), which its
  // owner -- usually another SM -- publishes with release semantics after all its global writes.
  const bool window = mode & TM_WINDOW;
  const uint32_t ctl_t = 32u * (uint32_t)((W > 4 && W <= 8) ? 4 : W - 1);
  const uint32_t n_items = (uint32_t)ngrp * (uint32_t)(window ? nsteps : 1);
  // three shared slots for the tickets drawn by thread 0: the ticket drawn at the start of
  // iteration `it` goes to slot (it + 2) % 3 and is read after the barrier at the end of that
  // iteration; the slot is written again three iterations (three barriers) later, so no warp can
  // still be reading it (two slots were not enough: thread 0 overwrote slot 0 at it = 0 while a
  // delayed warp could still be reading its first ticket from it)
  uint32_t *item_s = tm_base_s + 1;
  auto item_ready = [&](uint32_t item) -> bool {  // one lane
    const uint32_t s = item / (uint32_t)ngrp;
    if (!window || s == 0) return true;
    int32_t d;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];"
                 : "=r"(d)
                 : "l"(M.win_done + item % (uint32_t)ngrp)
                 : "memory");
    return d >= (int32_t)s;
  };
  auto wait_item = [&](uint32_t item, bool block) -> bool {  // whole warp; true when ready
    bool ok;
    do {
      ok = lane == 0 ? item_ready(item) : true;
      ok = __shfl_sync(0xffffffffu, ok, 0);
    } while (!ok && block);
    if (ok && window) asm volatile("fence.proxy.async;" ::: "memory");  // bulk copies read what
    return ok;                                                        // another SM just wrote
  };
  uint32_t cur, nxt;
  if (window) {
    if (threadIdx.x == 0) {
      item_s[0] = atomicAdd(M.win_ticket, 1u);
      item_s[1] = atomicAdd(M.win_ticket, 1u);
    }
    __syncthreads();
    cur = item_s[0];
    nxt = item_s[1];
  } else {
    cur = blockIdx.x;
    nxt = cur + gridDim.x;
  }
  if (cur < n_items) {
  TapeGroup tg = M.tgrp[cur % (uint32_t)ngrp];
  TapeClass tc = M.tcls[tg.cls];
  TapeTask tk = M.ttask[(size_t)tg.cls * W + warp];
  if (threadIdx.x == 0) load_program(tc, 0);
  wait_item(cur, true);
  start_segment(tg, tk);

  for (uint32_t it = 0; cur < n_items; ++it) {
    const uint32_t sphase = it & 1u;  // every signal mbarrier completes once per group
    const int g = (int)(cur % (uint32_t)ngrp);
    const int step_in = (int)(cur / (uint32_t)ngrp);  // step of the window
    const int64_t kk = k + step_in;
    const int smode = (mode & ~TM_ADVANCE) | ((mode & TM_ADVANCE) || step_in > 0 ? TM_ADVANCE : 0);
    const bool has_next = nxt < n_items;
    bool next_started = false;
    TapeGroup tgn = tg;
    TapeClass tcn = tc;
    TapeTask tkn = tk;
    if (has_next) {
      tgn = M.tgrp[nxt % (uint32_t)ngrp];
      tcn = M.tcls[tgn.cls];
      tkn = M.ttask[(size_t)tgn.cls * W + warp];
    }
    // Per-item control duties (ticket, program request, publishing the item) belong to the first
    // lane of the CONTROL WARP: the warp with the shortest list of the group (ctl_warp: the host
    // pairs the longest list, warp 0, with the shortest, warp 4, for 5..8 warps).  The
    // fence + release at the end of an item cost that lane ~2.4 us (measured); warp 0 would
    // start its -- longest -- forward sweep that much late.  The ticket of the item after the
    // next is drawn now and stored after the forward sweep, so that nobody waits for the
    // atomic's return.
    uint32_t ticket_r = 0;
    if (window && threadIdx.x == ctl_t) ticket_r = atomicAdd(M.win_ticket, 1u);
    CN_TR(0);
    const uint32_t pb = PB == 2 ? (it & 1u) : 0u;
    mbar_wait(pbar_s + 8 * pb, (PB == 2 ? it >> 1 : it) & 1u);
    CN_TR(1);
    const uint4 *prog = progbuf + (size_t)pb * M.tape_prog_cap;
    double *__restrict__ tape_l = M.tape + tg.tape_base + lane;
    const int p0 = tk.p0, p1 = tk.p1;

    // ========================================================================================
    // forward: mechanism records (nrn_state of the previous step, nrn_cur), then tree terms and
    // triangularisation, children before parents
    // ========================================================================================
    double accD = 0.0, accR = 0.0;
    // window mode: conductance / current rows of the warp's next point-process node, requested one
    // such node ahead (they sit in an L2-resident buffer, not on the tape)
    const double *wrow = M.win_rows + (size_t)step_in * M.win_stride + tg.pp_base +
                         (size_t)tk.pp0 * 64u + lane;
    double ppd = 0.0, ppr = 0.0;
    if (window && !flush) {
      ppd = __ldcg(wrow);
      ppr = __ldcg(wrow + 32);
    }
    // (a running 32-bit shared address: the compiler otherwise rebuilds &prog[j] from constants
    // in front of every record's load, on the warp's only instruction stream)
    uint32_t pa = smem_u32(prog + p0);
    for (int j = p0; j < p1; ++j, pa += 16) {
      const uint4 e = lds_u4(pa);
      const uint32_t ty = e.y & RT_MASK;
      CN_TR2(1, p0, j, (uint64_t)e.y | (uint64_t)e.x << 32);
      if (ty == RT_RUN) {
        // a run of plain chain nodes: each hands its contribution to the next in registers
        if (flush) continue;
        const unsigned char *rb = ringc + (e.x & 0xFFFFu);
        if (!(e.x & (1u << 24))) {
          accD = 0.0;
          accR = 0.0;
        }
        if (e.z & (1u << 20)) {  // (multiplier, reduced rhs) to the warp's tensor-memory slots
          uint32_t ta = tm_warp + ((uint32_t)tk.tm_base + (e.z & 1023u)) * 4u;
          // (the operands of the next node are fetched while the current one is on the dependent
          // chain: pivot -> reciprocal -> contribution = one DADD, MUFU + 3 DFMA, one DMUL)
          double a = CN_RD(rb, 0), b = CN_RD(rb, 1), d = CN_RD(rb, 2), vr = CN_RD(rb, 4) + CN_RD(rb, 3);
#pragma unroll 1
          for (int q = (int)((e.x >> 16) & 255u); q; --q) {
            const unsigned char *rn = rb + (q > 1 ? 5 * 256 : 0);
            const double a1 = CN_RD(rn, 0), b1 = CN_RD(rn, 1), d1 = CN_RD(rn, 2),
                         vr1 = CN_RD(rn, 4) + CN_RD(rn, 3);
            const double D = d + accD, R = vr + accR;
            const double ab = a * b, aR = a * R;
            const double rinv = rcp_chain(D);
            tm_store2(ta, b * rinv, R * rinv);
            accD = -(ab * rinv);
            accR = -(aR * rinv);
            rb = rn;
            a = a1; b = b1; d = d1; vr = vr1;
            ta += 4;
          }
        } else {
        double *srow = sys_l + (e.z & 1023u) * 64u;
        double a = CN_RD(rb, 0), b = CN_RD(rb, 1), d = CN_RD(rb, 2), vr = CN_RD(rb, 4) + CN_RD(rb, 3);
#pragma unroll 1
        for (int q = (int)((e.x >> 16) & 255u); q; --q) {
          const unsigned char *rn = rb + (q > 1 ? 5 * 256 : 0);
          const double a1 = CN_RD(rn, 0), b1 = CN_RD(rn, 1), d1 = CN_RD(rn, 2),
                       vr1 = CN_RD(rn, 4) + CN_RD(rn, 3);
          const double D = d + accD, R = vr + accR;
          const double ab = a * b, aR = a * R;
          const double rinv = rcp_chain(D);
          srow[0] = b * rinv;
          srow[32] = R * rinv;
          accD = -(ab * rinv);
          accR = -(aR * rinv);
          rb = rn;
          a = a1; b = b1; d = d1; vr = vr1;
          srow += 64;
        }
        }
        if (e.y & (1u << 26)) {  // the run ends with the top of its chain: contribution to the parent's row
          double *prow = sys_l + ((e.y >> 16) & 1023u) * 64u;
          if (e.y & (1u << 27)) {
            prow[0] += accD;
            prow[32] += accR;
          } else {
            prow[0] = accD;
            prow[32] = accR;
          }
          if (e.w & (1u << 24)) {
            __syncwarp();
            if (lane == 0) mbar_arrive(sbar_s + 8 * ((e.w >> 16) & 255u));
          }
        }
        continue;
      }
      if (ty == RT_CHUNK) {
        // the previous chunk is consumed: refill its stage, then wait for the next chunk
        const uint32_t rows = (e.x >> 16) & 255u;
        if (rows) {
          __syncwarp();
          if (lane == 0) {
            issue(e.z & 0xFFFFu, e.x & 0xFFFFu, rows);
            if (PF) prefetch((e.x & 0xFFFFu) + PF, (e.x & 0xFFFFu) + rows + PF);
          }
        }
        const uint32_t s = e.z >> 16;
        mbar_wait(bar_s + 8 * s, (phase >> s) & 1u);
        phase ^= 1u << s;
        continue;
      }
      if (ty == RT_WAIT) {
        if (!flush) mbar_wait(sbar_s + 8 * e.z, sphase);
        continue;
      }
      const uint32_t fl = e.y & 0xFFFFu;
      const unsigned char *rb = ringc + (e.x & 0xFFFFu);
      double *srow = sys_l + (e.z & 1023u) * 64u;
      if (ty == RT_ELIM) {
        if (flush) continue;
        if (e.x & (1u << 24)) mbar_wait(sbar_s + 8 * ((e.x >> 16) & 255u), sphase);  // (its own wait)
        const double a = CN_RD(rb, 0), b = CN_RD(rb, 1);
        double D = CN_RD(rb, 2), R = CN_RD(rb, 4) + CN_RD(rb, 3);
        if (fl & RF_FWD_IN) {
          D += accD;
          R += accR;
        }
        if (fl & RF_HAS_ACC) {
          D += srow[0];
          R += srow[32];
        }
        if (fl & RF_HAS_PP) {  // conductance / current of the point processes
          if (window) {  // (pp_window_kernel: this step's block of win_rows, prefetched)
            D += fx_get(ppd);
            R += fx_get(ppr);
            if (fx_nonzero(ppd) || fx_nonzero(ppr)) {  // consumed: the row is zero for the next window
              __stcg(const_cast<double *>(wrow), 0.0);  // (no memset of the whole buffer per window)
              __stcg(const_cast<double *>(wrow) + 32, 0.0);
            }
            wrow += 64;
            ppd = __ldcg(wrow);
            ppr = __ldcg(wrow + 32);
          } else {  // (pp_step_kernel: the two dynamic rows of the record, cleared after use)
            const double pd = CN_RD(rb, 5), pr = CN_RD(rb, 6);  // (fixed-point sums)
            D += fx_get(pd);
            R += fx_get(pr);
            if (fx_nonzero(pd) || fx_nonzero(pr)) {
              double *trec = tape_l + (e.w & 0xFFFFu) * 32u;
              trec[5 * 32] = 0.0;
              trec[6 * 32] = 0.0;
            }
          }
        }
        const double ab = a * b, aR = a * R;
        const double rinv = rcp_chain(D);
        const uint32_t kind = fl & RK_KIND;
        double mult = 0.0;
        if (kind != RK_ROOT) {
          const double cD = -(ab * rinv), cR = -(aR * rinv);
          mult = b * rinv;  // back-substitution multiplier
          if (kind == RK_FWD) {
            accD = cD;
            accR = cR;
          } else {
            double *prow = sys_l + ((e.z >> 10) & 1023u) * 64u;
            if (kind == RK_STORE) {
              prow[0] = cD;
              prow[32] = cR;
            } else {
              prow[0] += cD;
              prow[32] += cR;
            }
          }
        }
        if (fl & RF_TMEM) {
          tm_store2(tm_warp + ((uint32_t)tk.tm_base + (e.z & 1023u)) * 4u, mult, R * rinv);
        } else {
          srow[0] = mult;
          srow[32] = R * rinv;
        }
      } else {  // RT_MECH
        double gD, gR;
        mech_record(M, rb, tape_l + (e.y >> 16) * 32u, fl, e.w, smode, dt, q10dt, gD, gR);
        if (!flush) {
          srow[0] = gD;
          srow[32] = gR;
        }
      }
      if ((fl & RF_SIG_F) && !flush) {
        __syncwarp();
        if (lane == 0) mbar_arrive(sbar_s + 8 * (ty == RT_MECH ? e.z >> 16 : e.y >> 16));
      }
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    CN_TR(2);
    if (threadIdx.x == ctl_t) {
      if (PB == 2 && has_next) load_program(tcn, (it + 1) & 1);
      if (window) item_s[(it + 2) % 3] = ticket_r;  // read after the barrier at the end of this iteration
    }
    // this warp's ring is idle until the next group: start loading it now
    __syncwarp();
    if (has_next && wait_item(nxt, false)) {
      start_segment(tgn, tkn);
      next_started = true;
    }

    // ========================================================================================
    // backward: back-substitution (L66), v to the tape, threshold at the root (L68)
    // ========================================================================================
    if (!flush) {
      double v_prev = 0.0;
      uint32_t pab = smem_u32(prog + tk.b0);
      for (int j = tk.b0; j < tk.b1; ++j, pab += 16) {
        const uint4 e = lds_u4(pab);
        const uint32_t ty = e.y & RT_MASK;
        CN_TR2(0, tk.b0, j, (uint64_t)e.y | (uint64_t)e.x << 32);
        if (ty == RT_RUN) {
          // the parent of the run's last node: the node just solved, or a row that keeps its v
          // (a parent on another warp: the run waits for it itself)
          if (e.y & (1u << 24)) mbar_wait(sbar_s + 8 * ((e.y >> 16) & 255u), sphase);
          const int q = (int)((e.x >> 16) & 255u);
          if (e.x & (1u << 25)) v_prev = sys_l[((e.z >> 21) & 1023u) * 64u + 32];
          double *trow = tape_l + ((e.w & 0xFFFFu) + 5u * (uint32_t)q + 4u) * 32u;
          if (e.z & (1u << 20)) {
            uint32_t ta = tm_warp + ((uint32_t)tk.tm_base + (e.z & 1023u) + (uint32_t)q) * 4u;
#pragma unroll 1
            for (int i = q; i; --i) {
              ta -= 4;
              trow -= 5 * 32;
              double mult, rp;
              tm_load2(ta, mult, rp);
              v_prev = fma(-mult, v_prev, rp);
              *trow = v_prev;
            }
            continue;
          }
          const double *srow = sys_l + ((e.z & 1023u) + (uint32_t)q) * 64u;
#pragma unroll 2
          for (int i = q; i; --i) {
            srow -= 64;
            trow -= 5 * 32;
            v_prev = fma(-srow[0], v_prev, srow[32]);
            *trow = v_prev;
          }
          continue;
        }
        if (ty == RT_WAIT) {
          mbar_wait(sbar_s + 8 * e.z, sphase);
          CN_TR(3);
          continue;
        }
        const uint32_t fl = e.y & 0xFFFFu;
        if (fl & RF_WAIT_B) {
          mbar_wait(sbar_s + 8 * (e.y >> 16), sphase);
          CN_TR(3);
        }
        double *srow = sys_l + (e.z & 1023u) * 64u;
        double vp = v_prev;
        if (fl & RF_BW_ROW) vp = sys_l[((e.z >> 10) & 1023u) * 64u + 32];
        double mult, rp;
        if (fl & RF_TMEM) {
          tm_load2(tm_warp + ((uint32_t)tk.tm_base + (e.z & 1023u)) * 4u, mult, rp);
        } else {
          mult = srow[0];
          rp = srow[32];
        }
        const double v = fma(-mult, vp, rp);  // the root's multiplier is 0
        if (fl & RF_HAS_ACC) srow[32] = v;  // children that did not hand over in registers read it
        v_prev = v;
        tape_l[(e.w & 0xFFFFu) * 32u + 4 * 32] = v;
        if (fl & RF_MECHV) tape_l[(e.w >> 16) * 32u] = v;
        if (fl & RF_SIG_B) {
          __syncwarp();
          if (lane == 0) mbar_arrive(sbar_s + 8 * (e.x & 0xFFFFu));
        }
        if ((fl & RK_KIND) == RK_ROOT) {  // warp-ballot threshold detection, one atomic per warp
          bool fire = false;
          const int pc = tg.cell_base + lane;
          if (lane < tg.ncell) {
            const bool above = v > M.thr[pc];
            fire = above && !__ldcg(M.flag + pc);  // (another SM may have written it last step)
            __stcg(M.flag + pc, (unsigned char)above);
          }
          const unsigned ball = __ballot_sync(0xffffffffu, fire);
          if (ball) {
            unsigned long long sbase = 0;
            const int leader = __ffs(ball) - 1;
            if (lane == leader) sbase = atomicAdd(M.n_sp, (unsigned long long)__popc(ball));
            sbase = __shfl_sync(0xffffffffu, sbase, leader);
            if (fire) {
              const unsigned long long pos = sbase + __popc(ball & ((1u << lane) - 1u));
              if ((int64_t)pos < M.sp_cap) {
                M.sp_gid[pos] = M.gid_of_pcell[pc];
                M.sp_step[pos] = kk + 1;
              } else {
                *M.overflow = 1;
              }
            }
          }
        }
      }
    }
    CN_TR(4);
    __syncthreads();  // the system rows of this group are dead from here on
    if (M.wp_first && !flush) {  // window mode: the probed voltages of this (step, group)
      const int64_t row = M.trace_row0 + step_in;
      if (row < M.trace_cap)
        for (int p = M.wp_first[g] + (int)threadIdx.x; p < M.wp_first[g + 1]; p += (int)blockDim.x)
          M.trace[row * M.n_probe + M.wp_col[p]] =
              *reinterpret_cast<const volatile double *>(M.v + M.wp_pos[p]);  // (never from L1)
    }
    // one program buffer: the next group's program is requested first, so that its latency runs
    // beside the fence and the release below
    if (PB == 1 && has_next && threadIdx.x == ctl_t) load_program(tcn, 0);
    // the signal mbarriers this program did not use complete their phase too
    for (int b = (flush ? 0 : tc.n_bar) + (int)threadIdx.x; b < NB; b += (int)blockDim.x)
      mbar_arrive(sbar_s + 8 * b);
    if (window) {
      if (threadIdx.x == ctl_t) {  // every global write of the CTA for (step, group) is visible first
        __threadfence();
        asm volatile("fence.proxy.async;" ::: "memory");
        asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(M.win_done + g), "r"(step_in + 1)
                     : "memory");
      }
    }
    if (has_next && !next_started) {  // the next item was not ready when the forward sweep ended
      wait_item(nxt, true);
      start_segment(tgn, tkn);
    }
    CN_TR(5);
    cur = nxt;
    nxt = window ? item_s[(it + 2) % 3] : nxt + gridDim.x;
    tg = tgn;
    tc = tcn;
    tk = tkn;
  }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*tm_base_s),
                 "n"(CN_TMEM_COLS)
                 : "memory");
#undef CN_RD
}

// ------------------------------------------------------------------------------------------------
// point processes, one thread per instance: current + conductance into the node's dynamic rows,
// then the state decay (independent of v for these types, so cur and state fuse exactly; L65, L67)
// ------------------------------------------------------------------------------------------------

template <bool COOP>
__global__ void __launch_bounds__(256) pp_step_kernel(const __grid_constant__ DModel M,
                                                      int64_t k) {
  if (k < 0) k = M.step_ctr[0] - k - 1;  // replayed graph: the device counter + offset
  const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t nth = (int64_t)gridDim.x * blockDim.x;
  const double dt = M.dt;
  const double t_mid = ((double)k + 0.5) * dt;
  // targets: the node's conductance row on its group's tape (current row: + 32), or, for the
  // warp-cooperative groups (COOP, instances [0, pp_tape_begin)), its row pair in M.ppdr
  double *__restrict__ tape = COOP ? M.ppdr : M.tape;
  for (int t = 0; t < M.n_table; ++t) {
    const DTable &T = M.tab[t];
    if (!T.is_point) continue;
    const uint32_t *__restrict__ tgt = reinterpret_cast<const uint32_t *>(T.pp_slot);
    switch (T.type) {
      case T_EXPSYN:
        for (int64_t q = (COOP ? 0 : T.pp_tape_begin) + tid; q < (COOP ? T.pp_tape_begin : T.pp_tape_end); q += nth) {
          const double g = T.state[0][q];
          if (g != 0.0) {
            const double gs = g * T.param[2][q];
            fx_add(&tape[tgt[q]], gs, M.overflow);
            fx_add(&tape[tgt[q] + 32], gs * T.param[1][q], M.overflow);
            T.state[0][q] = decay(g, T.param[0][q]);
          }
        }
        break;
      case T_EXP2SYN:
        for (int64_t q = (COOP ? 0 : T.pp_tape_begin) + tid; q < (COOP ? T.pp_tape_begin : T.pp_tape_end); q += nth) {
          const double A = T.state[0][q], B = T.state[1][q];
          if (A != 0.0 || B != 0.0) {
            const double gs = (B - A) * T.param[3][q];
            if (gs != 0.0) {
              fx_add(&tape[tgt[q]], gs, M.overflow);
              fx_add(&tape[tgt[q] + 32], gs * T.param[2][q], M.overflow);
            }
            T.state[0][q] = decay(A, T.param[0][q]);
            T.state[1][q] = decay(B, T.param[1][q]);
          }
        }
        break;
      case T_ICLAMP:
        for (int64_t q = (COOP ? 0 : T.pp_tape_begin) + tid; q < (COOP ? T.pp_tape_begin : T.pp_tape_end); q += nth) {
          const double del = T.param[0][q];
          if (t_mid >= del && t_mid < del + T.param[1][q])
            fx_add(&tape[tgt[q] + 32], T.param[2][q] * T.param[3][q], M.overflow);
        }
        break;
      case T_AMPANMDA:
        for (int64_t q = (COOP ? 0 : T.pp_tape_begin) + tid; q < (COOP ? T.pp_tape_begin : T.pp_tape_end); q += nth) {
          const double a0 = T.state[0][q], a1 = T.state[1][q], a2 = T.state[2][q],
                       a3 = T.state[3][q];
          if (a0 != 0.0 || a1 != 0.0 || a2 != 0.0 || a3 != 0.0) {
            // v of the node: on the tape the v row precedes the two dynamic rows
            const double v = COOP ? M.v[(size_t)(tgt[q] >> 6) * 32 + (tgt[q] & 31u)] : tape[tgt[q] - 32];
            const double gs =
                ((a1 - a0) + T.glob[4] * (a3 - a2) * mgblock(v, T.glob[5])) * T.param[0][q];
            fx_add(&tape[tgt[q]], gs, M.overflow);
            fx_add(&tape[tgt[q] + 32], gs * T.glob[6], M.overflow);
            T.state[0][q] = decay(a0, T.glob[9]);
            T.state[1][q] = decay(a1, T.glob[10]);
            T.state[2][q] = decay(a2, T.glob[11]);
            T.state[3][q] = decay(a3, T.glob[12]);
          }
        }
        break;
      case T_GAP:  // L228: the peer's voltage as the previous step left it (this kernel runs
                   // before any voltage of step k is written)
        for (int64_t q = (COOP ? 0 : T.pp_tape_begin) + tid; q < (COOP ? T.pp_tape_begin : T.pp_tape_end); q += nth) {
          const double gs = T.param[0][q];
          fx_add(&tape[tgt[q]], gs, M.overflow);
          fx_add(&tape[tgt[q] + 32], gs * M.v[(int64_t)T.param[1][q]], M.overflow);
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

// the inverse (checkpoint load): loc already includes the state's row offset
__global__ void scatter_state_kernel(double *__restrict__ tape, double *__restrict__ st,
                                     const int64_t *__restrict__ loc, int64_t n,
                                     const double *__restrict__ src) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int64_t l = loc[i];
  if (l >= 0) st[l] = src[i]; else tape[-(l + 1)] = src[i];
}

}  // namespace cn
