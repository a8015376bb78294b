// unit_layout.h - the in-HBM layout of one "cell unit", shared by the host builder and the kernels.
//
// A unit is the work of one CTA.  Two kinds share the record formats of this file:
//   forests      (forest_layout.h) one or several cells, lane = control volume, segmented warp scans:
//                every cell that does not share its tree with others and fits a CTA's shared memory
//   block units  (this file) one cell whose branches (maximal unbranched chains of control volumes)
//                are interleaved so that consecutive lanes touch consecutive addresses, lane = branch
//                ("SoA with interleaved branches", BASELINE.json north_star; the paper's own GPU layout
//                interleaves whole cells, one thread per cell, PAPER.md:220 - prior art), integrated
//                straight from global memory: cells too large for shared memory, and cells with
//                thousands of synapses (key reduction).
//
//   level l of the unit  = all branches whose distance (in branches) from their cell's root is l
//   task                 = up to 32 branches of one level, longest first; one warp, lane = branch
//   row k of a task      = the k-th control volume (k = 0 proximal) of every branch longer than k;
//                          rows are stored back to back and are RAGGED: row k holds cnt_k = #{lanes :
//                          len > k} slots, so a unit has exactly one slot per control volume
//   slot(task, k, lane)  = task.slot_off + sum_{j<k} cnt_j + lane
//
// Per unit there are four records in the device workspace:
//   fast  (bytes, constant per dt)  UnitHeader | f | invd | a | b | hh conductances | per-synapse
//                                   e, decay (only when synapses are not uniform) | clamps |
//                                   slot / cell indices of HH instances, synapses, clamps
//   state (doubles, mutable)        V | m | h | n | g | per-cell runtime triples
//   gen   (doubles, constant)       C | S | sigma | G | bg | syn_tau     (dt-independent; used by
//                                   the factorisation and by event-split sub-steps only)
//   topo  (bytes, constant)         tasks, levels, branch links - shared by all units with the same
//                                   tree structure (deduplicated); a warp keeps the record of its
//                                   current unit in shared memory and reloads it only on change
// The fast and state records are what a time step streams.
#pragma once
#include <stdint.h>

#if defined(__CUDACC__)
#define ARBB_HD __host__ __device__ __forceinline__
#else
#define ARBB_HD inline
#endif

namespace arbb {

constexpr uint32_t kNoSlot = 0xFFFFFFFFu;
constexpr uint32_t kBlockUnitMaxCells = 64;

struct Task {            // 16 bytes, one broadcast load
  uint32_t slot_off;     // slot of (k = 0, lane = 0)
  uint32_t nslots;       // sum of the branch lengths
  uint32_t lane_off;     // unit-local branch index of lane 0
  uint16_t nlanes;       // 1..32
  uint16_t maxlen_full;  // bits 0..14: length of lane 0 (the longest); bit 15: every lane has that length
};
constexpr uint16_t kTaskFull = 0x8000u;

struct LaneRec {         // 16 bytes per branch, one load per lane
  uint32_t pslot;        // slot of the parent control volume of the branch's first CV, or kNoSlot
  uint32_t cbeg;         // first entry of its child-branch list
  uint16_t len;          // control volumes in the branch
  uint16_t ccnt;         // child branches hanging off its last CV
  uint16_t cell;         // unit-local cell
  uint16_t pad;
};

enum : uint32_t { UNIT_BLOCK = 1u };   // processed by a whole CTA straight from global memory

struct UnitHeader {      // the first 128 bytes of a unit's fast record
  uint32_t n_slot;       // control volumes rounded up to even (one dead slot when odd)
  uint32_t n_lane, n_task, n_level;
  uint32_t n_cell, n_hh, n_syn, n_clamp;
  uint32_t n_child, flags, fast_bytes, state_bytes;
  int64_t topo_off;      // byte offset into the topo pool
  int64_t gen_base;      // double index into the gen pool
  int64_t state_base;    // double index into the state pool
  int64_t cell_base;     // internal index of the unit's first cell
  int64_t scratch_base;  // double index into the scratch pool (block units) or -1
  uint32_t pad[10];
};
static_assert(sizeof(UnitHeader) == 128, "UnitHeader must be 128 bytes");

struct UnitDesc {        // what a loader needs before the header has arrived; 32 bytes
  int64_t fast_off;      // byte offset into the fast pool (128-byte aligned)
  int64_t state_base;    // double index into the state pool (16-double aligned)
  uint32_t fast_bytes, state_bytes;   // multiples of 16
  uint32_t topo_off16, topo_bytes;    // forests: the tree record (byte offset / 16 into the topo pool, bytes), which
                                      // the kernel stages in shared memory; 0 for block units
};

ARBB_HD uint32_t align_up(uint32_t x, uint32_t a) { return (x + a - 1) / a * a; }

// Byte offsets inside the fast record (every section 16-byte aligned).
struct FastOff {
  uint32_t f, invd, a, b, hh_gna, hh_gk, hh_gl, syn_e, syn_decay, cl_t0, cl_t1, cl_amp,
      hh_slot, syn_slot, cl_slot, hh_cell, syn_cell, cl_cell, total;
};
ARBB_HD FastOff fast_offsets(uint32_t n_slot, uint32_t n_hh, uint32_t n_syn, uint32_t n_clamp, uint32_t n_cell,
                             bool syn_uniform) {
  FastOff o;
  uint32_t p = 128;
  auto sec = [&](uint32_t bytes) { uint32_t at = p; p = align_up(p + bytes, 16); return at; };
  o.f = sec(8 * n_slot); o.invd = sec(8 * n_slot); o.a = sec(8 * n_slot); o.b = sec(8 * n_slot);
  o.hh_gna = sec(8 * n_hh); o.hh_gk = sec(8 * n_hh); o.hh_gl = sec(8 * n_hh);
  o.syn_e = sec(syn_uniform ? 0 : 8 * n_syn); o.syn_decay = sec(syn_uniform ? 0 : 8 * n_syn);
  o.cl_t0 = sec(8 * n_clamp); o.cl_t1 = sec(8 * n_clamp); o.cl_amp = sec(8 * n_clamp);
  o.hh_slot = sec(4 * n_hh); o.syn_slot = sec(4 * n_syn); o.cl_slot = sec(4 * n_clamp);
  const bool multi = n_cell > 1;
  o.hh_cell = sec(multi ? 2 * n_hh : 0); o.syn_cell = sec(multi ? 2 * n_syn : 0); o.cl_cell = sec(multi ? 2 * n_clamp : 0);
  o.total = p;
  return o;
}

// Double offsets inside the state record (every section 16-byte aligned).
struct StateOff { uint32_t v, m, h, n, g, rt, total; };
ARBB_HD StateOff state_offsets(uint32_t n_slot, uint32_t n_hh, uint32_t n_syn, uint32_t n_cell) {
  StateOff o;
  uint32_t p = 0;
  auto sec = [&](uint32_t n) { uint32_t at = p; p = align_up(p + n, 2); return at; };
  o.v = sec(n_slot); o.m = sec(n_hh); o.h = sec(n_hh); o.n = sec(n_hh); o.g = sec(n_syn); o.rt = sec(3 * n_cell);
  o.total = p;
  return o;
}

// Per-cell runtime triple inside the state record:
//   rt[0] = time of the next undelivered event of the current epoch list (+inf: none)
//   rt[1] = (ev_end << 32) | ev_cur   cursor and end of the cell's segment of the epoch list
//   rt[2] = 1.0 when the threshold detector is armed (reading R10), else 0.0
constexpr int kRtDoubles = 3;

// Double offsets inside the gen record.
struct GenOff { uint32_t C, S, sig, G, b, syn_tau, total; };
ARBB_HD GenOff gen_offsets(uint32_t n_slot, uint32_t n_syn) {
  GenOff o;
  o.C = 0; o.S = n_slot; o.sig = 2 * n_slot; o.G = 3 * n_slot; o.b = 4 * n_slot; o.syn_tau = 5 * n_slot;
  o.total = align_up(5 * n_slot + n_syn, 2);
  return o;
}

// Byte offsets inside a topo record (every section 8-byte aligned).
struct TopoOff { uint32_t tasks, lanes, level_begin, child, cell_det, total; };
ARBB_HD TopoOff topo_offsets(uint32_t n_task, uint32_t n_level, uint32_t n_lane, uint32_t n_child, uint32_t n_cell) {
  TopoOff o;
  uint32_t p = 0;
  auto sec = [&](uint32_t bytes) { uint32_t at = p; p = align_up(p + bytes, 16); return at; };
  o.tasks = sec(n_task * (uint32_t)sizeof(Task));
  o.lanes = sec(n_lane * (uint32_t)sizeof(LaneRec));
  o.level_begin = sec((n_level + 1) * 4);
  o.child = sec(n_child * 4);
  o.cell_det = sec(n_cell * 4);
  o.total = p;
  return o;
}

// per-cell runtime of the (sub-)step in progress, in shared memory (device_common.cuh: CellS)
constexpr uint32_t kCellScratchBytes = 64;   // tcur, tnext, delta, vprev (doubles) + evcur, evend, armed, mode, wb, dirty (u32)

}  // namespace arbb
