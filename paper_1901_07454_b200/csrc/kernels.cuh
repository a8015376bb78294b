// kernels.cuh - device-side model view and kernel launchers (implemented in kernels.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "forest_layout.h"
#include "group_layout.h"
#include "unit_layout.h"

namespace arbb {

enum Counter {
  CNT_SPIKES = 0,       // spikes recorded since creation
  CNT_SPIKES_DONE = 1,  // spikes already turned into events
  CNT_POOL = 2,         // events waiting in the current pool
  CNT_POOL_NEXT = 3,    // events carried over into the other pool
  CNT_ERROR = 4,        // bit 0 spike overflow, bit 1 pool overflow, bit 2 epoch list overflow, bit 3 non-finite voltage
  CNT_SUBSTEPS = 5,     // cell sub-steps executed
  CNT_DELIVERED = 6,    // events delivered
  CNT_EVLIST = 7,       // size of the current epoch list
  CNT_GROUP0 = 8,       // group kernel: next unclaimed group of even / odd launches (dynamic
  CNT_GROUP1 = 9,       //   distribution of groups over the persistent CTAs)
  CNT_HOT0 = 10,        // group kernel: lengths of the three rotating "hot" lists (groups with an event in
  CNT_HOT1 = 11,        //   the next grid step, which are integrated first so that their longer
  CNT_HOT2 = 12,        //   event-split steps do not end up at the tail of the launch)
  CNT_POOL_PEAK = 13,   // largest number of events in flight asked of the pool so far (also beyond its capacity)
  CNT_COUNT = 14
};

struct EventPool { double* t; uint32_t* dst; uint32_t* gidx; double* w; };

struct DevModel {
  const UnitDesc* units;      // forests first, then block units
  int64_t n_units, n_forests, n_cells;
  ForestClass fcls[kForestClasses];   // forest launches by shared-memory need (forest_layout.h)
  uint8_t* fast;
  double* state;
  const double* gen;
  const uint8_t* topo;
  double* scratch;            // at header.scratch_base: block units contrib | dcontrib | xI | fgen | invdgen | run heads;
                              // forests fgen | invdgen | dcon (forest_layout.h)
  double* factor_dcontrib;    // [total branches], used by factor_kernel only
  const uint32_t* cell_orig;  // internal -> caller's cell id
  const uint32_t* cell_rt_idx;// internal cell -> state index of its runtime triple
  // epoch event list (CSR over internal cells)
  uint32_t* ev_off;           // [n_cells + 1]
  double* ev_t; uint32_t* ev_gidx; double* ev_w;
  uint32_t* ev_fill;          // [n_cells] fill cursors / counts
  int64_t ev_cap;
  // external events (CSR over internal cells, time sorted) and their cursors
  const uint32_t* ext_off; const double* ext_t; const uint32_t* ext_gidx; const double* ext_w;
  uint32_t* ext_cur;
  // network grouped by source cell (global ids when the model is a shard: local cell c is source gid_base + c)
  int64_t gid_base;
  const uint32_t* conn_off; const uint32_t* conn_dst; const uint32_t* conn_gidx;
  const double* conn_delay; const double* conn_w;
  EventPool pool[2];
  int64_t pool_cap;
  // spikes
  uint32_t* spike_cell; double* spike_t; int64_t spike_cap;
  unsigned long long* counters;
  uint32_t* scan_tmp;         // block sums for the offsets scan
  // synapse parameters when every synapse of the model has the same tau and e
  int syn_uniform;
  double syn_e_u, syn_tau_u, syn_decay_u;
  double ena, ek, el, theta;
  // cell groups (group_layout.h); cells of groups come first in the internal cell order
  const GroupDesc* groups;
  int64_t n_groups;
  GroupSmemPlan gplan;
  int l2_prefetch;            // group kernel: TMA-prefetch the next group's records into L2
  // point cells (LIF cells, spike sources): the last n_pcells cells of the internal order
  int64_t n_pcells, pc_first, pc_state_base;
  const int32_t* pc_kind; const double* pc_par; const uint32_t* pc_src_off; const double* pc_src_time; const uint32_t* pc_cv;
  int sm_count;               // SMs of the device the model lives on (grid sizing)
  int linearised;             // ARB_OPT_LINEARISED: conductance-linearised step
  // synapse runs (reading R22): lazy records (g_j | time of last touch | tau, 3 x lazy_n doubles) at state[lazy_base];
  // an event's target index inside that range names a record, lazy_run[record] the state index of the run it feeds
  uint32_t lazy_base, lazy_n;
  const uint32_t* lazy_run;
  const uint32_t* run_off; const uint32_t* run_gidx; int64_t n_runs;
  uint32_t* ghot;             // group kernel: three lists of n_groups entries (see CNT_HOT0)
  uint32_t* ghotflag;         // [2][n_groups], half launch_id & 1: launch_id of the launch whose hot list holds the group
};

struct StepArgs {
  double t0, dt, t_end;  // grid t_k = t0 + k*dt, t_nsteps = t_end
  int64_t k_first, nk, nsteps;
  int last_full;         // the last grid step has nominal length dt
  int parity;            // launch counter & 1 (group kernel: which work counter this launch claims from)
  uint32_t launch_id;    // group kernel: running number of the launch
  int hot_valid;         // the hot list of this launch was written by the launch before it
  int mark_hot;          // write the hot list of the next launch
};

// Where an event with target index gx adds its weight.  A target inside the lazy range is a synapse of a
// cell that keeps one conductance per run (R22): its own record is brought up to date at the delivery time t,
// g_j <- g_j exp(-(t - t_j) / tau) + w, and the weight goes to the run.
__device__ __forceinline__ uint32_t event_target(const DevModel& M, uint32_t gx, double t, double w) {
  if (gx - M.lazy_base < M.lazy_n) {                 // (unsigned: false for everything below lazy_base, and when lazy_n == 0)
    double* rec = M.state + gx;
    const double tau = rec[2 * (size_t)M.lazy_n], tl = rec[M.lazy_n];
    rec[0] = rec[0] * exp(-(t - tl) / tau) + w;
    rec[M.lazy_n] = t;
    return M.lazy_run[gx - M.lazy_base];
  }
  return gx;
}

// all launchers queue work on `s` and return the last CUDA error code
cudaError_t launch_factor(const DevModel& M, double dt, cudaStream_t s);
cudaError_t launch_init(const DevModel& M, cudaStream_t s);
// the cable step of the block units: one CTA per unit
cudaError_t launch_cable(const DevModel& M, const StepArgs& A, cudaStream_t s, int* launches);
// forests (forest_kernel.cu): one launch per shared-memory class
cudaError_t launch_forest_factor(const DevModel& M, double dt, cudaStream_t s);
cudaError_t launch_forest_init(const DevModel& M, cudaStream_t s);
cudaError_t launch_forest_cable(const DevModel& M, const StepArgs& A, int cls, cudaStream_t s, int* launches);
cudaError_t configure_forest_kernel(int max_optin_bytes);
cudaError_t launch_build_events(const DevModel& M, int cur_pool, double t_window_end, cudaStream_t s, int* launches);
cudaError_t launch_spikes_to_events(const DevModel& M, int cur_pool, cudaStream_t s, int* launches);
// sharded networks: push the spikes of `n_blocks` blocks (int64 count | int64 gid[cap] | double t[cap]) except block
// `own` through the connection table into the event pool
cudaError_t launch_remote_spikes_to_events(const DevModel& M, int cur_pool, const unsigned long long* blocks, int64_t n_blocks,
                                           int64_t cap, int64_t own, cudaStream_t s);
cudaError_t launch_gather(const double* state, const uint32_t* idx, int64_t n, double* out, cudaStream_t s);
// synaptic conductances at time t: lazy records (R22) are decayed from their time of last touch on the way out
cudaError_t launch_gather_syn(const DevModel& M, const uint32_t* idx, int64_t n, double t, double* out, cudaStream_t s);
// after new g_j were scattered into the lazy records: stamp them with t and rebuild every run's sum (index order)
cudaError_t launch_lazy_rebuild(const DevModel& M, double t, cudaStream_t s);
cudaError_t launch_scatter(double* state, const uint32_t* idx, int64_t n, const double* in, cudaStream_t s);
cudaError_t launch_gather_hh(const double* state, const uint32_t* m_idx, const uint32_t* stride, const uint32_t* cv,
                             int which, int64_t n_hh, double* out, cudaStream_t s);
cudaError_t launch_scatter_hh(double* state, const uint32_t* m_idx, const uint32_t* stride, const uint32_t* cv,
                              int which, int64_t n_hh, const double* in, cudaStream_t s);
cudaError_t launch_reset_detectors(const DevModel& M, cudaStream_t s);
// point cells: one epoch (events before t_win, scheduled spikes before t_win); read-back / state injection helpers
cudaError_t launch_point_cells(const DevModel& M, double t_win, cudaStream_t s, int* launches);
cudaError_t launch_lif_relax(const DevModel& M, double t, double* io, cudaStream_t s);
cudaError_t launch_point_reset(const DevModel& M, double t, cudaStream_t s);
// read-back without an allocation (no_alloc.cu): the staging buffer is a static device array of kNoAllocMaxCv doubles
constexpr int64_t kNoAllocMaxCv = 1 << 19;   // 4 MiB per GPU that loads the library
int64_t noalloc_max_cv();
cudaError_t noalloc_scratch(double** out);   // its device address on the current device (cudaGetSymbolAddress, once per device)
cudaError_t launch_noalloc_gates(const double* state, const uint32_t* m_idx, const uint32_t* stride, const uint32_t* cv, int which,
                                 int64_t n_hh, int64_t n_cv, double* host_out, cudaStream_t s);
// cell groups (group_kernel.cu)
cudaError_t launch_group_factor(const DevModel& M, double dt, uint32_t seg_cap, cudaStream_t s);
cudaError_t launch_group_init(const DevModel& M, cudaStream_t s);
cudaError_t launch_group_cable(const DevModel& M, const StepArgs& A, int grid, cudaStream_t s, int* launches);
int group_ctas_per_sm(uint32_t smem_bytes);   // resident CTAs of the group kernel per SM (0: does not fit)
// Opts the cable kernels into the device's full dynamic shared memory on the CURRENT device (the
// attribute is per function and device; called by every arb_create, nothing is cached).
cudaError_t configure_kernels();
cudaError_t configure_group_kernel(int max_optin_bytes);
int cable_smem_limit();       // bytes of dynamic shared memory a CTA may use (sm_100a opt-in maximum)

}  // namespace arbb
