// layout.hpp - host-side model builder: validation, branch decomposition, cell blocks.
// Pure C++ (no CUDA): turns the caller's arb_desc into the pools described in block_layout.h.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/arbb200.h"
#include "block_layout.h"

namespace arbb {

struct BuildParams {
  uint32_t target_slots = 2304;   // close a block once it holds this many CVs (on-chip budget)
  uint32_t max_cells = 64;        // cells per block
  uint32_t max_branch_len = 1024; // longer unbranched chains are cut into pieces
};

struct HostModel {
  int64_t n_cells = 0, n_cv = 0, n_syn = 0, n_clamp = 0, n_conn = 0, n_ext = 0, n_hh = 0;
  int64_t n_blocks = 0, n_lanes = 0;
  int64_t gen_doubles = 0, fast_doubles = 0, state_doubles = 0, meta_bytes = 0, scratch_doubles = 0;
  uint32_t max_block_slots = 0, max_block_lanes = 0, max_block_cells = 0;
  double min_delay = 0, max_delay = 0;
  double ena = 0, ek = 0, el = 0, threshold = 0;
  std::vector<BlockInfo> blocks;
  std::vector<uint32_t> cell_order;     // internal -> caller's cell id
  std::vector<uint32_t> cell_internal;  // caller's cell id -> internal
  std::vector<uint32_t> cell_block;     // internal -> block
  // ---- filled only by build(..., fill = true) ----
  std::vector<double> gen, fast, state;
  std::vector<uint8_t> meta;
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
