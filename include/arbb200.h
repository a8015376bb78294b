/* arbb200.h - C ABI of libarbb200: B200-native (sm_100a) stepping of many multi-compartment cells.
 *
 * The library implements ONE thing: the data-parallel hot path of arXiv 1901.07454 ("Arbor"),
 * /root/reference/PAPER.md section II (lines 92-158) and IV-C (lines 216-220): per time step
 *   deliver spike events into synapses
 *   mechanism currents from V(t)              (eq 2a at 127-131)
 *   assemble the implicit-Euler cable matrix
 *   solve it with the Hines / extended Thomas algorithm over the parent index
 *   V <- V', integrate mechanism state with V'
 *   threshold detection -> spikes
 * and once per minimum-delay epoch turn spikes into events on the targets' queues
 * (PAPER.md:96, 198-202).  Every step runs in hand-written CUDA kernels on the device; there is no
 * CPU fallback.  All arithmetic is fp64, indices int32/int64, times fp64.
 *
 * Units (reading R2): V mV, t ms, area um^2, cm uF/cm^2, density conductance S/cm^2,
 * point conductance uS, current nA, axial resistance MOhm.
 *
 * Pointer conventions: every pointer in arb_desc and every output buffer is a HOST pointer owned by
 * the caller; arb_desc arrays are read only during arb_plan / arb_create and never retained.  The
 * only DEVICE pointer is `dev_workspace`: one caller-owned allocation (the library never calls
 * cudaMalloc) that must stay alive, and untouched by the caller, until arb_destroy.
 *
 * Errors: every call returns 0 (or a count) on success or a negative ARB_E_* code; nothing throws
 * or aborts across the ABI; arb_last_error gives text.  A model may be used by one host thread at a
 * time; the library keeps no process-wide mutable state (models on several devices may coexist; the
 * calling thread's current device must be the one the workspace lives on).
 */
#ifndef ARBB200_H
#define ARBB200_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
  ARB_OK = 0,
  ARB_E_NULL = -1,      /* a required pointer is NULL                                            */
  ARB_E_INVALID = -2,   /* description or argument out of range (see arb_plan)                   */
  ARB_E_WORKSPACE = -3, /* device workspace smaller than arb_plan asked for, or misaligned       */
  ARB_E_CUDA = -4,      /* a CUDA runtime call or kernel failed                                  */
  ARB_E_OVERFLOW = -5,  /* spike / event buffer capacity exceeded (see "Capacities" below)        */
  ARB_E_NOMEM = -6,     /* host allocation failed                                                */
  ARB_E_DIVERGED = -7   /* a detector voltage became NaN / Inf (the explicit membrane currents of
                           reading R1 are only conditionally stable); the model is unusable after */
};

/* arb_probe selectors */
enum { ARB_PROBE_M = 0, ARB_PROBE_H = 1, ARB_PROBE_N = 2, ARB_PROBE_SYN_G = 3, ARB_PROBE_TIME = 4,
       ARB_PROBE_NSTEPS = 5, ARB_PROBE_STATS = 6, ARB_PROBE_TIMING = 7 };

/* arb_set_option keys */
enum {
  ARB_OPT_FUSED_STEPS = 1,   /* max grid steps integrated per kernel launch with the cell block's
                                state kept on-chip: 1 = one launch per time step (state streams
                                through HBM every step); 0 (default) = a whole min-delay epoch
                                (cells are independent within Delta_T)           */
  ARB_OPT_EPOCH_STEPS = 2,   /* cap on the epoch length in steps (default: floor(min delay / dt)) */
  ARB_OPT_OVERLAP = 4,       /* 1 (default): the cable kernels of one grid step (cell groups, forests by launch
                                class, block units) run side by side on streams forked from the model's
                                stream; 0: one after the other on the model's stream               */
  ARB_OPT_L2_PREFETCH = 5,   /* cell-group kernel: 1 (default) = ask the TMA unit to pull the next group's
                                records into L2 while the current group is integrated; 0 = off      */
  ARB_OPT_HOT_FIRST = 7,     /* cell-group kernel, one launch per grid step: 1 (default) = groups with an event in
                                the coming step are integrated first (their event-split steps take longer and
                                would otherwise end up at the tail of the launch); 0 = index order          */
  ARB_OPT_GROUP_CTAS = 6,    /* cell-group kernel: cap on the CTAs of a launch (0 = as many as are resident) */
  ARB_OPT_LINEARISED = 8,    /* 1: the conductance-linearised variant of the implicit Euler step (PAPER.md:152-156
                                with every membrane current g_k (V' - E_k) taken at the new voltage: conductances
                                on the diagonal, sources g_k E_k on the right-hand side; the matrix is assembled
                                and eliminated every step; unconditionally stable).  0 (default): explicit membrane
                                currents, the equation as printed at PAPER.md:154 (reading R1), matrix
                                factorised once per dt.  Not available for models with block units.         */
  ARB_OPT_TIMING = 3         /* 1: bracket the cable-step launches and the epoch-boundary kernels of
                                every epoch with CUDA events on the model's stream (read them with
                                ARB_PROBE_TIMING); setting the option clears the accumulated times  */
};

/* The problem statement of PAPER.md section II as flat arrays.
 * Cells are trees of control volumes (CVs).  Per-cell fields use CSR offsets
 * over cells; CV and synapse indices inside a cell are cell-local. */
typedef struct {
  /* cells and compartments */
  int64_t n_cells;
  const int64_t* cv_off;    /* [n_cells+1], cv_off[0] = 0, every cell has >= 1 CV                 */
  const int32_t* cv_parent; /* [n_cv] local parent, -1 for CV 0 (root), otherwise 0 <= parent < i */
  const double* cv_area;    /* [n_cv] um^2  > 0   (S_i)                             */
  const double* cv_cm;      /* [n_cv] uF/cm^2 > 0 (c_i = cm * area)                               */
  const double* cv_raxial;  /* [n_cv] MOhm > 0, CV centre -> parent centre (1/sigma_ij); root ignored */
  const double* cv_vinit;   /* [n_cv] mV, or NULL => -65                                          */
  /* density mechanisms; all three hh arrays or none; a CV whose three hh
   * parameters are 0 has no HH; pas_g == 0 => no passive channel on that CV                    */
  const double *hh_gnabar, *hh_gkbar, *hh_gl; /* [n_cv] S/cm^2 or NULL                           */
  double hh_ena, hh_ek, hh_el;                /* mV                                               */
  const double *pas_g, *pas_e;                /* [n_cv] S/cm^2, mV; both or NULL                  */
  /* exponential synapses (point mechanisms) */
  const int64_t* syn_off;   /* [n_cells+1] or NULL when there are no synapses                    */
  const int32_t* syn_cv;    /* [n_syn] local CV                                                  */
  const double *syn_tau, *syn_e; /* [n_syn] ms (> 0), mV                                          */
  /* current clamps: amplitude > 0 depolarises, active for t0 <= t < t1 (t = step start)          */
  int64_t n_clamp;
  const int64_t* clamp_cell;
  const int32_t* clamp_cv;
  const double *clamp_t0, *clamp_t1, *clamp_amp; /* ms, ms, nA                                    */
  /* spike detectors, one per cell */
  const int32_t* det_cv;    /* [n_cells] local CV, or NULL => CV 0                               */
  double threshold;         /* mV                                                                */
  /* network: (source, destination, synapse, delay, weight)                         */
  int64_t n_conn;
  const int64_t *conn_src, *conn_dst; /* cells                                                   */
  const int32_t* conn_syn;            /* synapse index local to the destination cell             */
  const double *conn_delay, *conn_weight; /* ms (> 0, and >= dt at arb_advance), uS               */
  /* external events (kicks, pre-generated Poisson trains): g[syn] += weight at `time`            */
  int64_t n_ext;
  const int64_t* ext_cell;
  const int32_t* ext_syn;
  const double *ext_time, *ext_weight; /* ms (>= 0), uS                                           */
  /* Layout and capacity options; 0 = library default.  Part of the description, so that planning
   * and creation agree and the library keeps no process-wide state.
   *   layout_group_min_cells  cells with identical trees are laid out cell-interleaved in groups
   *                           (lane = cell) when their topology class has at least this many cells
   *                           (default 4; 1 = every cell in groups; >= 2^31 = no groups)
   *   layout_forest_cv        cells that do not share their tree are packed into forests of up to this
   *                           many control volumes, one CTA each (default: 2048, less for models of fewer than 1.2e6 such
   *                           control volumes so that they spread over the SMs, and never more than fits the
   *                           27 KB of shared memory of the smallest launch class; a larger cell is a
   *                           forest of its own)
   *   cap_spikes              entries of the device spike buffer.  arb_advance drains it into host
   *                           memory at least every 2,000 grid steps, so it bounds the spikes of
   *                           such a stretch, not of the run (default max(2^20, 64 n_cells))
   *   cap_events              entries of the pool of events in flight, i.e. generated by a spike
   *                           but due after the epoch being built (default n_conn * max(4,
   *                           ceil(max delay / 2 ms) + 1) + 1024)
   * Capacities: exceeding one makes arb_advance return ARB_E_OVERFLOW with the buffer named in
   * arb_last_error.  Events or spikes beyond the capacity are lost, so the model is unusable
   * afterwards (every later call returns the same error): create it again with a larger cap_*.
   * (reading R0 says why the state is not rolled back to the last epoch.) */
  int64_t layout_group_min_cells, layout_forest_cv, cap_spikes, cap_events;
  /* Sharding (cells are distributed over ranks, spikes are exchanged once per epoch).
   * shard_n_global == 0: the model is the whole network, conn_src are its own cells.
   * shard_n_global > 0: the model holds cells [shard_gid_base, shard_gid_base + n_cells) of a network of
   * shard_n_global cells; conn_dst stay local, conn_src are GLOBAL cell ids (the table holds every connection
   * whose destination is local); spikes of remote sources arrive through arb_apply_spike_blocks.           */
  int64_t shard_gid_base, shard_n_global;
  /* Cell kinds other than the multi-compartment cell ("leaky integrate and fire cells and cells
   * representing artificial spike sources"; the paper names them only, reading R20).
   * cell_kind[c]: 0 = multi-compartment cell, 1 = LIF cell, 2 = spike source; NULL => all 0.
   * A LIF / source cell owns exactly ONE control volume in the per-CV arrays (its geometry is ignored; the CV's
   * voltage is the LIF membrane potential, cv_vinit its initial value) and its synapse range is its event targets.
   * LIF (event-driven, exact): V relaxes to lif_e_l with lif_tau_m; an event of weight w (a charge, pC) adds
   * w / lif_c_m; V >= lif_v_th at an event emits a spike AT the event time, V <- lif_e_r, events are ignored for
   * lif_t_ref.  Spike source: emits the times src_time[src_off[c] .. src_off[c+1]) (ascending).
   * The lif_* arrays are [n_cells] (read for LIF cells only); src_off is [n_cells+1]; all NULL when cell_kind is. */
  const int32_t* cell_kind;
  const double *lif_tau_m, *lif_v_th, *lif_c_m, *lif_e_l, *lif_e_r, *lif_t_ref; /* ms, mV, nF, mV, mV, ms */
  const int64_t* src_off;
  const double* src_time;
} arb_desc;

typedef struct arb_model arb_model; /* opaque; lives in host memory, owned by the library */

/* Validate the description and report the device workspace size arb_create needs.  No device
 * work, no allocation kept.  ARB_E_INVALID: parent >= index or < -1, non-positive area / cm /
 * raxial / tau, CV / synapse / cell index out of range, delay <= 0, NaN / Inf, external event
 * earlier than t = 0, inconsistent NULLs. */
int arb_plan(const arb_desc* desc, size_t* workspace_bytes);

/* Build the model: lay the cells out (cell-interleaved groups for cells that share a tree, forests
 * with lane = control volume for the rest), upload to
 * `dev_workspace` (DEVICE pointer, 256-byte aligned, >= workspace_bytes from arb_plan) on
 * `cuda_stream` (a cudaStream_t; NULL = default stream), initialise state (V = vinit, gates at
 * steady state, g = 0, t = 0; reading R4).  Returns after the upload has completed. */
int arb_create(const arb_desc* desc, void* dev_workspace, size_t workspace_bytes, void* cuda_stream,
               arb_model** out);

/* Integrate from the model's current time t to t_end on the grid t_k = t + k*dt; a final shorter
 * step is taken when (t_end - t) is not a multiple of dt; grid steps are split at event times
 * (reading R9).  Kernels are queued on the model's stream; the call returns after
 * they have completed and the overflow flags have been checked.  ARB_E_INVALID: dt <= 0,
 * t_end < t, dt longer than the shortest connection delay.
 * Epochs: cells are independent for one minimum delay, so spikes become events
 * once per epoch of floor(min_delay / dt - 1e-6) grid steps (at least 1).  The 1e-6 guard keeps an
 * event that lands exactly on the epoch's last grid point out of the epoch that generates it: a
 * network with min_delay = 5 ms and dt = 0.025 ms runs epochs of 199 steps, one with
 * min_delay = 5.0001 ms epochs of 200.  Results do not depend on the epoch length. */
int arb_advance(arb_model* m, double t_end, double dt);

/* Spikes since creation (or since the last arb_clear_spikes).  Returns the count; fills min(cap,
 * count) entries sorted by (time, cell).  cell / time may be NULL when cap == 0.  Negative on
 * error.  The history lives in host memory (arb_advance drains the device buffer into it). */
int64_t arb_spikes(arb_model* m, int64_t* cell, double* time, int64_t cap);

/* Sharded networks (arb_desc.shard_*), one call pair per epoch between two arb_advance calls; the caller moves
 * the blocks between ranks (an all-gather: ncclAllGather / torch.distributed.all_gather_into_tensor).
 * arb_spike_block: writes the spikes this model has produced since the previous arb_spike_block call (or since
 * creation) into `dev_block`, a DEVICE buffer of (1 + 2 cap) 8-byte words: int64 count | int64 gid[cap] |
 * double time[cap], global cell ids.  Returns the count, ARB_E_OVERFLOW when it exceeds cap (nothing is lost:
 * call again with a larger block).
 * arb_apply_spike_blocks: `dev_blocks` holds n_blocks such blocks back to back (DEVICE memory); every spike of
 * every block except block `own_block` (this model's own: arb_advance has turned those into events already; pass
 * -1 to apply all) is pushed through the local connection table: events (spike time + delay, synapse, weight)
 * on the targets' queues, delivered by the following arb_advance calls.  Every epoch advanced between two exchanges
 * must be no longer than the shortest connection delay of the WHOLE network.                                  */
int64_t arb_spike_block(arb_model* m, void* dev_block, int64_t cap);
int arb_apply_spike_blocks(arb_model* m, const void* dev_blocks, int64_t n_blocks, int64_t cap, int64_t own_block);

/* Forget the spikes recorded so far (a caller that reads spikes after every epoch keeps the
 * history short this way).  Does not touch events already generated from them. */
int arb_clear_spikes(arb_model* m);

/* Membrane potential of every CV in the caller's CV order.  n_cv must equal cv_off[n_cells]. */
int arb_voltage(arb_model* m, double* out, int64_t n_cv);

/* ARB_PROBE_M/H/N: gate state per CV (0 where the CV has no HH), n = n_cv.
 * ARB_PROBE_SYN_G: synaptic conductance per synapse in the caller's order, n = n_syn.  (In a cell with >= 1,024
 *                  synapses the library integrates ONE conductance per run of synapses that sit on the same control
 *                  volume with the same tau and e - I = (sum g_j)(V - e) and the exponential decay are exact for the
 *                  sum - when that at least halves their number; every synapse keeps a record (g_j, time of last
 *                  event) from which this probe returns its own conductance, and arb_set_state rebuilds the sums.
 *                  DESIGN.md reading R22; 10,000 synapses on ~130 control volumes.)
 * ARB_PROBE_TIME:  out[0] = current time, n >= 1.
 * ARB_PROBE_NSTEPS: out[0] = grid steps so far, out[1] = cell sub-steps so far (>= cells*grid
 *                  steps; the excess comes from event-driven step splitting), n >= 2.
 * ARB_PROBE_STATS: out[0..7] = {units, slots (CVs incl. padding), branches, workspace bytes,
 *                  events delivered, kernel launches so far, epoch steps, bytes of the records one
 *                  grid step moves (all units and groups)}, n >= 8; when n >= 12 also {warp units,
 *                  warps per CTA and shared-memory bytes per warp of the last launch, distinct tree
 *                  records}; when n >= 16 also {cell groups, topology classes in groups, CTAs of a
 *                  cell-group launch, shared-memory bytes per CTA of the cell-group kernel}; when
 *                  n >= 20 also {forests, block units, CTAs of a forest launch, shared-memory bytes
 *                  per CTA of the forest kernel}.
 * ARB_PROBE_TIMING: out[0..3] = {ms spent in cable-step kernels, cable-step launches timed,
 *                  ms spent in epoch-boundary (spike -> event) kernels, their launches}, measured
 *                  with CUDA events while ARB_OPT_TIMING is on, n >= 4. */
int arb_probe(arb_model* m, int what, double* out, int64_t n);

/* arb_probe(ARB_PROBE_M / ARB_PROBE_H / ARB_PROBE_N) for callers that may not allocate device memory (code under CUDA
 * graph capture, serving loops, harnesses that forbid cudaMalloc): the per-CV staging buffer the gates are gathered
 * into is not part of a workspace but a static device array of arb_noalloc_max_cv() = 524,288 doubles (4 MiB, held by
 * every GPU that loads the library until the process exits).  Same arguments and result as arb_probe for the three gate
 * selectors: out[i] = the gate of control volume i, 0 where it carries no HH mechanism, n_cv = the model's CV count,
 * `out` is HOST memory, the call returns after the copy.  ARB_E_INVALID (with the limit in arb_last_error) when n_cv
 * exceeds the array; nothing is written then.  The call makes no cudaMalloc / cudaFree and no allocating library call.
 * All calls on a GPU share the array and it keeps the last call's contents: every call clears the part it uses first,
 * so calls in sequence are independent, but calls that OVERLAP on the GPU (two models on different streams) race -
 * serialise them. */
int arb_gates_noalloc(arb_model* m, int what, double* out, int64_t n_cv);
int64_t arb_noalloc_max_cv(void);

/* Overwrite state from host arrays in the caller's order (any pointer may be NULL = keep).
 * Detector history is reset to the new voltages.  Exists so that tests can start both
 * implementations from one state. */
int arb_set_state(arb_model* m, const double* v, const double* hh_m, const double* hh_h,
                  const double* hh_n, const double* syn_g);

int arb_set_option(arb_model* m, int key, int64_t value);

/* The mechanism catalogue (mechanisms and cell kinds "are referenced by name").  The library's
 * mechanisms are hand-written kernels; the catalogue is the table that names them, their kind and their parameters
 * (the arb_desc fields that carry them), so that a front end can look a mechanism up instead of hard-coding fields.
 * arb_catalogue_size: entries.  arb_catalogue_entry: name ("hh", "pas", "expsyn", "iclamp", "lif", "spike_source"),
 * kind (0 density mechanism, 1 point mechanism, 2 cell kind), number of parameters; returns ARB_E_INVALID beyond the
 * table.  arb_catalogue_param: name of the arb_desc field, unit and default value of one parameter.
 * arb_catalogue_find: index of a name, or -1. */
int arb_catalogue_size(void);
int arb_catalogue_entry(int index, const char** name, int* kind, int* n_params);
int arb_catalogue_param(int index, int param, const char** field, const char** unit, double* default_value);
int arb_catalogue_find(const char* name);

/* Measures the fp64 fused-multiply-add rate of the current device (independent DFMA chains in
 * registers, no memory traffic; kernel timed with CUDA events on `cuda_stream`, NULL = default
 * stream): the peak of the arithmetic bound of the roofline ("Roofline time per
 * step = max(bytes/BW, DP-instr/peak)").  *dfma_per_s receives DFMA instructions (thread level) per
 * second, *ms (may be NULL) the duration of the timed launch.  Needs no model. */
int arb_fp64_peak(void* cuda_stream, double* dfma_per_s, double* ms);

void arb_destroy(arb_model* m);

/* Text of the last error of this model, or of the last arb_plan / arb_create failure on this
 * thread when m == NULL.  Never NULL. */
const char* arb_last_error(const arb_model* m);

#ifdef __cplusplus
}
#endif
#endif
