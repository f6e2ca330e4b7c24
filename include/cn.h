/*
 * cn.h -- C ABI of libcn: B200-native fixed-step time integration of networks of
 * multi-compartment neurons (the hot path of arxiv 1901.10975, "CoreNEURON").
 *
 * Each dt runs, entirely on the device:
 *   event-driven spike delivery (L64) -> matrix assembly: per-mechanism currents and
 *   conductances plus the tree terms of the discretised cable equation (L65, Eq. 1)
 *   -> Hines tree solve (L62 "direct Gaussian elimination", L66) -> voltage update (L66)
 *   -> per-mechanism state update, cnexp / derivimplicit (L67, L278)
 *   -> threshold detection and NetCon event generation with delays (L68, L62, L156).
 *
 * Conventions
 *   - All pointers in cn_model_desc are HOST pointers; cn_model_create deep-copies, so the
 *     caller may free them on return.  Output pointers are HOST pointers owned by the caller.
 *   - The model owns its device and host memory until cn_model_destroy.  Device memory is
 *     allocated on the CUDA device that is current at cn_model_create (a large model starts
 *     uploading its arrays there while the layout is compiled) and at the first cn_run: keep
 *     the same device current for every call on a model.
 *   - Every call returns a status (CN_OK or a negative CN_ERR_*), never throws or aborts;
 *     cn_last_error() gives a thread-local message for the last non-OK return.
 *   - Units (L58-60): mV, ms, uF/cm2, S/cm2 and mA/cm2 for distributed mechanisms; point
 *     processes in nA and uS (converted by 100/area[um2], L60); area um2; axial resistance MOhm.
 *   - All indices in and out are in the caller's order; the internal permutation is invisible.
 *   - No CPU fallback exists: without a CUDA device every compute call fails with CN_ERR_CUDA.
 */
#ifndef CN_H
#define CN_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cn_model cn_model; /* opaque */

enum {
  CN_OK = 0,
  CN_ERR_ARG = -1,      /* NULL / non-finite / out-of-range scalar or array argument */
  CN_ERR_TOPOLOGY = -2, /* parent[] is not a forest with parent[i] < i inside each cell */
  CN_ERR_MECH = -3,     /* unknown mechanism type, wrong parameter count, node out of range */
  CN_ERR_NETCON = -4,   /* NetCon source/target out of range, or delay rounds to < 1 step */
  CN_ERR_DT = -5,       /* dt <= 0 or different from the dt of the first cn_run */
  CN_ERR_CUDA = -6,     /* CUDA runtime error (message in cn_last_error) */
  CN_ERR_OVERFLOW = -7, /* spike buffer overflowed during a run; results are invalid */
  CN_ERR_NOMEM = -8,    /* host or device allocation failed */
  CN_ERR_UNSUPPORTED = -9 /* a cell too large for the on-chip solve, a size beyond a stated limit */
};

/* Mechanism types.  Parameter order = row order of cn_mech_table.param. */
enum {
  CN_PAS = 1,      /* i = g (v - e)                         param: g, e                       */
  CN_HH = 2,       /* Hodgkin-Huxley squid Na/K/leak        param: gnabar, gkbar, gl, el
                      global: ena, ek.  Temperature factor 3^((celsius-6.3)/10).              */
  CN_EXPSYN = 3,   /* point: i = g (v - e), g' = -g/tau     param: tau, e ; event: g += w     */
  CN_EXP2SYN = 4,  /* point: i = (B-A)(v-e)                 param: tau1, tau2, e (tau1<tau2)
                      event: A += w f, B += w f, f normalises the peak to w                   */
  CN_ICLAMP = 5,   /* point: current amp for del <= t < del+dur   param: del, dur, amp (nA)
                      sampled at the step midpoint (k + 1/2) dt                               */
  CN_HHFORM = 6,   /* i = gbar m^p h^q (v - E)              param: gbar
                      global: p, q, E, to_ica, m:(vh,k,t0,t1,vt,s), h:(vh,k,t0,t1,vt,s)
                      xinf = 1/(1+exp((vh-v)/k)), tau = t0 + t1/(exp((v-vt)/s)+exp(-(v-vt)/s)) */
  CN_SK = 7,       /* i = gbar z (v - E), zinf = 1/(1+(Kd/cai)^n)  param: gbar
                      global: E, Kd, n, tau_z                                                 */
  CN_CADYN = 8,    /* cai' = -(1e4 gamma/(2 F depth)) ica - (cai-cai_min)/tau_d  (derivimplicit)
                      no param ; global: gamma, depth, tau_d, cai_min                         */
  CN_AMPANMDA = 9, /* point: AMPA + NMDA double exponentials with Mg block
                      no param ; global: tau_r_A, tau_d_A, tau_r_N, tau_d_N, r_nmda, mg, e    */
  CN_GAP = 10      /* point: one half of a gap junction, i = g (v - v_peer)
                      param: g (uS), peer (global node index in caller order, an integral double)
                      v_peer is the peer's voltage at the START of the step (exchanged once per
                      dt); g enters the node's diagonal.  A symmetric junction is two instances.
                      Models with gap junctions run one launch sequence per dt (no window).    */
};

/* One mechanism type = one instance table, structure of arrays (L178, Fig. 3D). */
typedef struct {
  int32_t type;          /* CN_PAS ... */
  int64_t n;             /* number of instances */
  const int32_t *node;   /* [n] global node index, caller order */
  int32_t n_param;       /* must equal the type's parameter count */
  const double *param;   /* [n_param][n]: parameter j of instance i at param[j*n + i] */
  int32_t n_global;      /* must equal the type's global count */
  const double *global;  /* [n_global] per-table constants */
} cn_mech_table;

typedef struct {
  int32_t n_cell;
  int64_t n_node;
  const int64_t *cell_first;  /* [n_cell+1]; node cell_first[c] is the root (soma) of cell c;
                                 the spike source id (gid) of cell c is c */
  const int32_t *parent;      /* [n_node] global index; -1 for roots; parent[i] < i, same cell */
  const double *area_um2;     /* [n_node] membrane area, > 0 */
  const double *ri_MOhm;      /* [n_node] axial resistance node <-> parent, > 0 (ignored at roots) */
  const double *cm_uF_cm2;    /* [n_node] specific capacitance, > 0 */
  double v_init_mV;           /* initial voltage of every node; gates start at steady state */
  double celsius;
  int32_t n_mech;
  const cn_mech_table *mech;  /* currents and states are evaluated in table order */
  int64_t n_netcon;           /* NetCons, structure of arrays (L62, L156) */
  const int32_t *nc_src_gid;  /* cell gid (< n_cell) or scripted source gid (>= n_cell) */
  const int32_t *nc_tgt_mech; /* index into mech[]; must be a point process with a receive rule */
  const int64_t *nc_tgt_inst; /* instance within that table */
  const double *nc_weight_uS;
  const double *nc_delay_ms;  /* quantised as llround(delay/dt) steps at the first cn_run; >= 1 */
  const double *thr_mV;       /* [n_cell] threshold on the root node: spike iff v rises above */
  int64_t n_stim;             /* scripted source spikes (artificial spike sources) */
  const int32_t *stim_gid;    /* [n_stim] >= n_cell */
  const double *stim_t_ms;    /* [n_stim] >= 0; spike step = llround(t/dt) */
} cn_model_desc;

/* Validate, deep-copy, find shape classes, choose the permutation (no CUDA device is needed for
 * that; with one, a large model's arrays start travelling to it).  The dt-dependent tables are
 * built at the first cn_run.  *out is NULL on failure. */
int cn_model_create(const cn_model_desc *desc, cn_model **out);

/* The same with options: "key=value;key=value" (';', ',' or white space between pairs; values are
 * numbers; NULL or "" = defaults; an unknown key or a malformed pair -> CN_ERR_ARG).  Options are
 * fixed for the life of the model.  The library reads NO environment variable and has no global
 * flag: these are the only knobs, and every one of them leaves the results unchanged (within the
 * parity tolerance) -- they choose between launch strategies:
 *   tape             -1 auto / 0 / 1   which kernel: 1 every class with enough cells on the
 *                                      interleaved kernel, 0 all cells on the warp-cooperative one
 *   tape_min_cells   8192              auto: models at least this large use the interleaved kernel
 *   tape_min_group   16 (1 for small   smallest ragged group of a class kept on the interleaved
 *                    models)           kernel
 *   tape_w           8                 warps per CTA of the interleaved kernel (1..16)
 *   tape_s, tape_ch  2, 16 (auto)      TMA ring of a warp: stages x rows per chunk
 *   tape_tmem        1                 0: all system rows in shared memory, none in tensor memory
 *   tape_window      1                 0: one launch sequence per dt even where a min-delay window
 *                                      per launch is possible
 *   tape_pbuf, tape_ctas_per_sm        program buffers (1/2) and CTAs per SM (1/2), default auto
 *   tape_pf          0                 rows of L2 prefetch ahead of the ring
 *   tape_leaf_first, tape_hcost, tape_gran, tape_mcost, tape_bcost
 *                                      cost model of the static schedule
 *   force_g, max_g, warp_smem, wpb     warp-cooperative kernel: cells per warp, shared-memory cap
 *                                      per warp, warps per block
 *   graph            1                 0: per-dt launch sequences are issued one by one instead of
 *                                      being replayed from a CUDA graph
 *   onchip           -1 auto / 0 / 1   on-chip window mode: a model that fits the
 *                                      shared memory of the device is integrated a whole min-delay
 *                                      window per launch without touching HBM in between
 *   debug            0                 1: set-up timings on stderr */
int cn_model_create_opts(const cn_model_desc *desc, const char *options, cn_model **out);

/* Advance to ABSOLUTE time tstop with fixed step dt: K = llround(tstop/dt) - steps_done steps
 * (K <= 0 is a no-op).  dt is fixed by the first call.  Runs on `stream` set by cn_set_stream
 * (default: the legacy default stream) and synchronises it before returning.
 * Launch granularity is an internal matter with identical results: one set of launches per dt,
 * or -- when every cell runs on the interleaved kernel and no point process depends on v within
 * a step (AMPA+NMDA, gap junctions do) -- one launch per window of up to min-delay steps (L62
 * "every minimum spike delay interval"). */
int cn_run(cn_model *m, double tstop_ms, double dt_ms);

/* Same as cn_run but returns without synchronising; cn_sync() waits and reports overflow. */
int cn_run_async(cn_model *m, double tstop_ms, double dt_ms);
int cn_sync(cn_model *m);

/* cudaStream_t (as void*) on which all work of this model is issued. */
int cn_set_stream(cn_model *m, void *cuda_stream);

/* Current voltages in caller node order; n must equal n_node. */
int cn_get_v(const cn_model *m, double *v_out, int64_t n);

/* Spikes (gid, step) sorted by (step, gid); a spike detected after the update to t_{k+1} has
 * step k+1.  Pass cap = 0 to query *n_out only. */
int cn_get_spikes(const cn_model *m, int32_t *gid, int64_t *step, int64_t cap, int64_t *n_out);

/* Record v of the given nodes after every step (before the first cn_run only): by a probe
 * kernel after every step, or, in window mode, by the interleaved kernel itself when a group
 * completes a step. */
int cn_set_probes(cn_model *m, const int32_t *node, int64_t n, int64_t max_steps);
/* trace_out[s*n_probe + j] = v(node j) after step s; *n_steps_out = steps recorded. */
int cn_get_trace(const cn_model *m, double *trace_out, int64_t cap_steps, int64_t *n_steps_out);

/* State s of mechanism table t after the last step, in caller instance order (for parity tests);
 * n = table size.  (The interleaved kernel applies nrn_state of a step at the start of the next
 * one; this call applies the pending update first.) */
int cn_get_state(const cn_model *m, int32_t t, int32_t s, double *out, int64_t n);

/* cn_get_state for callers that cannot call cudaMalloc (code under CUDA graph capture, serving
 * loops, harnesses that forbid it): same arguments (`out`: host buffer of n doubles, owned by the
 * caller), same result, but the gather scratch is a static device array of the library instead of
 * a buffer grown with cudaMalloc.  The call allocates nothing (no cudaMalloc / cudaFree, no host
 * heap).  Limit: tables of at most CN_NOALLOC_MAX_INSTANCES instances (the array is 16 B per
 * instance = 1 MiB, held by every GPU that loads the library until the process exits); a larger
 * table -> CN_ERR_UNSUPPORTED, nothing written.  Every call shares the array: the call is
 * synchronous on the model's stream and serialised by a process-wide lock; work that the caller
 * overlaps with it by other means must not touch the same entry point (it would race). */
#define CN_NOALLOC_MAX_INSTANCES 65536
int cn_get_state_noalloc(const cn_model *m, int32_t t, int32_t s, double *out, int64_t n);

int64_t cn_steps_done(const cn_model *m);
/* Number of kernels launched by this model so far (for bench.py's gpu_launches). */
int64_t cn_launch_count(const cn_model *m);
/* Device pointer + stream-ordered timing of the step kernels of the last run, in ms, measured
 * with CUDA events on the model's stream around the step loop. */
int cn_last_run_ms(const cn_model *m, double *ms_out);
/* Sample the duration of the step kernel (the dominant kernel) with CUDA event pairs on the
 * model's stream around every `every`-th launch (0 = off), at most max_samples between reads.
 * cn_get_kernel_timing returns the summed duration and the number of dt the samples cover (one
 * launch of the interleaved kernel integrates a whole window of steps), and resets. */
int cn_set_kernel_timing(cn_model *m, int32_t every, int32_t max_samples);
/* Which kernel the samples bracket when the model runs one launch sequence per dt: 0 the step
 * kernel (default: interleaved kernel if it runs, else the warp-cooperative one), 1 the
 * point-process kernel(s), 2 the event-delivery kernel.  (Window modes always time the window
 * kernel.)  While sampling is on, launch sequences are issued directly, not from a CUDA graph. */
int cn_select_timed_kernel(cn_model *m, int32_t which);
int cn_get_kernel_timing(cn_model *m, double *sum_ms_out, int64_t *count_out);
/* Layout facts for DESIGN/bench, info8 = { n_class, n_group (all), shared-memory bytes per warp and
 * max elimination rounds of the warp-cooperative kernel, n_group of the interleaved (tape) kernel,
 * tape bytes, shared-memory bytes per CTA of the interleaved kernel (after the first cn_run),
 * warps per CTA | persistent CTAs << 8 | shared-memory system rows << 24 }. */
int cn_get_layout_info(const cn_model *m, int64_t *info8);
/* How the model runs (after the first cn_run), info4 = { launch mode: 0 one launch sequence per
 * dt, 1 window mode of the interleaved kernel, 2 on-chip window mode (one CTA keeps one cell on
 * chip for a min-delay window), -1 not yet known; CUDA-graph replays so far; steps per window;
 * persistent CTAs of the window kernel }. */
int cn_get_run_info(const cn_model *m, int64_t *info4);
/* Checkpoint / restore.  A checkpoint holds the dynamic state after the last
 * step and nothing else, in the CALLER'S order: voltages, mechanism and synapse states, cai,
 * threshold flags, and the spikes recorded so far (state-sized: 8 B per node and per state).  No
 * event queue is saved: the events still in flight are regenerated from the spikes and the NetCon
 * delays (L156: in-flight events collapse to their originating spikes).  No parameter and nothing
 * of the internal layout is in it, so it loads into ANY model with the same structure -- cells,
 * topology, mechanism tables and their nodes (hashed; CN_ERR_ARG otherwise) -- whatever that
 * model's parameters, stimuli (IClamp tables, scripted sources), NetCon weights, options or launch
 * mode: "launch multiple simulations with different stimuli" (L156).  The restored model continues
 * from the saved step with the saved dt (CN_ERR_DT if it already runs with another dt), with ITS
 * OWN parameters and NetCons.  Load before or after the model's first cn_run.  Every check is done
 * before the model is touched: a rejected buffer leaves the model as it was.  Per-step traces
 * (cn_set_probes) are not part of it.  buf: caller-owned HOST memory. */
int cn_checkpoint_size(const cn_model *m, int64_t *bytes_out);
int cn_checkpoint_save(const cn_model *m, void *buf, int64_t bytes);
int cn_checkpoint_load(cn_model *m, const void *buf, int64_t bytes);

/* Spike buffer capacity (default 16*n_cell + 65536); before the first cn_run only. */
int cn_set_spike_capacity(cn_model *m, int64_t cap);

void cn_model_destroy(cn_model *m);
const char *cn_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
