// layout.hpp - host-side model builder: validation, branch decomposition, cell groups, forests, block units.
// Pure C++ (no CUDA): turns the caller's arb_desc into the pools described in group_layout.h,
// forest_layout.h and unit_layout.h.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/arbb200.h"
#include "forest_layout.h"
#include "group_layout.h"
#include "unit_layout.h"

namespace arbb {

struct BuildParams {
  bool forest_cv_auto = true;     // a small model gets smaller forests, so that it still spreads over the SMs: forests of
                                  // (control volumes in forests) / (4 x 148 SMs) control volumes, at least 384, at most forest_cv
  uint32_t forest_cv = 2048;      // cells are packed into forests of up to this many control volumes (larger cells
                                  // are a forest of their own)
  uint32_t forest_max_cv = 24000; // cells with more control volumes do not fit a CTA's shared memory: block units
  uint32_t forest_max_syn = 1024; // cells with at least this many synapses are block units (key reduction)
  uint32_t merge_min_syn = 1024;  // cells with at least this many synapses keep ONE conductance per run of synapses on the same
                                  // control volume with the same (tau, e) (second half); 0 = never
  uint32_t max_branch_len = 1024; // block units: longer unbranched chains are cut into pieces
  uint32_t group_min_cells = 4;   // a topology class with fewer cells is laid out as units; 0 = no groups
  uint32_t group_max_smem = 112 * 1024;  // shared memory a cell group may need (two CTAs per SM at least)
  uint32_t group_max_cv = 1536;   // cells with more control volumes are laid out as units (V of a
                                  // group must fit in shared memory: 8 * kG bytes per control volume)
};

constexpr int kPcDoubles = 8;         // a point cell's record in the state pool: V | runtime triple | t_last | t_ref_end |
                                      // schedule cursor | pad
constexpr int64_t kMaxGroupCtas = 148 * 16;   // upper bound of resident CTAs of the group kernel (scratch sizing)

struct UnitCounts {                   // everything the offset functions need
  uint32_t n_slot = 0, n_cv = 0, n_lane = 0, n_task = 0, n_level = 0, n_cell = 0, n_hh = 0, n_syn = 0,
           n_clamp = 0, n_child = 0;
  uint32_t flags = 0;
  int64_t cell_base = 0, lane_base = 0, hh_base = 0;
  int64_t fast_off = 0, state_base = 0, gen_base = 0, topo_off = 0, scratch_base = -1;
  uint32_t fast_bytes = 0, state_bytes = 0, topo_bytes = 0;
  int n_warp = 0;                     // forests: warps that sweep the unit (forest_layout.h)
};

struct HostModel {
  int64_t n_cells = 0, n_cv = 0, n_syn = 0, n_clamp = 0, n_conn = 0, n_ext = 0, n_hh = 0;
  // point cells (arb_desc.cell_kind != 0: LIF cells, spike sources): the last cells of the internal order
  int64_t n_sched = 0;                  // scheduled spikes of all sources
  int64_t n_pcells = 0, pc_first = 0, pc_state_base = 0;   // first internal index; double index of their records
  std::vector<int32_t> pc_kind;
  std::vector<double> pc_par;           // [n_pcells][6]: tau_m, v_th, c_m, e_l, e_r, t_ref
  std::vector<uint32_t> pc_src_off, pc_cv;   // schedule offsets [n_pcells + 1]; caller's CV index of every point cell
  std::vector<double> pc_src_time;
  // synapse runs (reading R22): synapses of merged cells keep a lazy record (g_j, time of last touch, tau) in the state pool
  // at [lazy_base, lazy_base + 3 n_lazy); syn_state_idx of such a synapse is its record, lazy_run the state index of its run
  int64_t n_lazy = 0, lazy_base = 0, n_runs = 0, n_syn_inst = 0;   // n_syn_inst: synapse instances the kernels integrate
  std::vector<uint32_t> lazy_run;       // [n_lazy]
  std::vector<uint32_t> run_off;        // [n_runs + 1]: lazy records of run r (contiguous)
  std::vector<uint32_t> run_gidx;       // [n_runs]: state index of the run's conductance
  int64_t gid_base = 0, n_src = 0;    // sharding: global id of local cell 0, cells of the whole network (= n_cells when unsharded)
  int64_t n_units = 0, n_forests = 0, n_lanes = 0;   // units: forests first, then block units
  int64_t fast_bytes = 0, state_doubles = 0, gen_doubles = 0, topo_bytes = 0, scratch_doubles = 0;
  int64_t topo_records = 0;           // distinct tree structures
  ForestClass fcls[kForestClasses];   // forest launches by shared-memory need
  uint32_t block_lane_cap = 0;
  bool syn_uniform = false;
  double syn_tau_u = 0, syn_e_u = 0;
  double min_delay = 0, max_delay = 0;
  double ena = 0, ek = 0, el = 0, threshold = 0;
  // cell groups: cells [0, n_group_cells) of the internal order
  int64_t n_groups = 0, n_group_cells = 0, n_classes = 0;
  GroupCaps gcaps = {0, 0, 0, 0, 0};
  uint32_t g_seg_cap = 0;
  std::vector<GroupDesc> gdescs;
  std::vector<UnitCounts> units;
  std::vector<uint32_t> cell_order;     // internal -> caller's cell id
  std::vector<uint32_t> cell_internal;  // caller's cell id -> internal
  // ---- filled only by build(..., fill = true) ----
  std::vector<uint8_t> fast, topo;
  std::vector<double> state, gen;
  std::vector<UnitDesc> descs;
  std::vector<uint32_t> cell_rt_idx;    // internal cell -> index of its runtime triple in the state pool
  std::vector<uint32_t> cv_state_idx;   // caller's CV -> index of its V in the state pool
  std::vector<uint32_t> syn_state_idx;  // caller's synapse -> index of its g in the state pool
  std::vector<uint32_t> hh_m_idx, hh_stride, hh_cv;  // per HH instance: index of m, distance to h, caller's CV
  // network, grouped by (caller's) source cell; external events grouped by internal cell, time-sorted
  std::vector<uint32_t> conn_off, conn_dst, conn_gidx;
  std::vector<double> conn_delay, conn_w;
  std::vector<uint32_t> ext_off, ext_gidx;
  std::vector<double> ext_t, ext_w;
};

// Returns ARB_OK or ARB_E_*; err receives text.
int validate(const arb_desc& d, std::string& err);
int build(const arb_desc& d, const BuildParams& p, bool fill, HostModel& out, std::string& err);

}  // namespace arbb
