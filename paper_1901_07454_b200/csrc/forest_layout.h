// forest_layout.h - the in-HBM layout of a "forest", shared by the host builder and the kernels.
//
// Cells whose tree is their own (no other cell of the model has the same parent array) cannot be
// interleaved cell by cell (group_layout.h).  They are packed into FORESTS: one or several whole cells
// that one CTA integrates together, LANE = CONTROL VOLUME.  Both sweeps of the Hines solve
// are first-order linear recurrences along a branch once the matrix is factorised
// (reading R1), so a warp runs them as segmented scans over 32 consecutive control volumes (affine
// maps compose) instead of walking a branch row by row: the serial depth of a step is the number of
// branch LEVELS of the deepest cell (<= 9 for BASELINE.json configs[4]), not its longest path in
// control volumes (321).  (The paper's GPU solver runs one thread per cell over interleaved matrices,
// PAPER.md:220, and names "a GPU solver for Hines matrices [that] exposes more fine-grained
// parallelism" as future work.)
//
//   branch   a maximal unbranched chain of control volumes; its slots are consecutive, proximal first
//   level    branches at the same distance (in branches) from their cell's root; levels of all cells of
//            the forest are aligned, __syncthreads separates levels
//   run      the branches of one level that one warp of the CTA sweeps; its slots are consecutive.  A forest of
//            few cells deals the branches of a level to the warps (whole branches, longest first to the least
//            loaded warp); a forest of many cells deals whole CELLS to the warps (UNIT_WARP_CELLS), so that a
//            warp never waits for another between levels
//   chunk    32 consecutive slots of a run = one warp-wide segmented scan; a branch longer than a chunk
//            carries its recurrence from one chunk of the run to the next in a register
// Slot order: level (root first) -> warp -> branch -> control volume, so the forward sweep walks
// ascending addresses and every load of a per-CV array is one coalesced 256-byte row.
//
// A forest reuses the unit records of unit_layout.h (UnitHeader, fast / state / gen records with the
// same offset functions); only the tree record differs (FTopoOff below):
//   n_lane = branches, n_task = chunks, n_level = levels of the deepest cell; pad[2] = warps that sweep the forest.
#pragma once
#include <stdint.h>

#include "unit_layout.h"

namespace arbb {

constexpr int kForestWarps = 4;                      // warps per CTA of the forest kernel: forests of launch class 0 ...
constexpr int kForestWarpsBig = 8;                   // ... and of the classes above it (one large cell each: twice the warps
                                                     // halve the serial part of its step; measured on C4: 338 -> 251 us)
constexpr int kForestMaxWarps = 8;
constexpr int kForestThreads = kForestWarps * 32;
constexpr uint32_t kForestMaxCells = 64;             // cells per forest (one thread per cell keeps its runtime)
constexpr uint32_t kForestMaxBranchLen = 32768;      // longer chains are cut (len is stored in 16 bits)
constexpr int kForestClasses = 4;                    // launches by shared-memory need: 8, 4, 2, 1 CTAs per SM

enum : uint32_t { UNIT_FOREST = 2u,                  // UnitHeader.flags
                  UNIT_POINT_DISJOINT = 4u,          // no two kinds of point mechanism share a control volume
                  UNIT_WARP_CELLS = 8u };            // every cell of the forest is swept by ONE warp (all its branches are
                                                     // in that warp's runs): levels need __syncwarp only
constexpr uint32_t kForestWarpCellsMin = 6;          // cells a forest needs before its cells are dealt to warps whole

struct FRun { uint32_t chunk_beg, chunk_end; };      // chunks [beg, end) of (level, warp); backward runs them end -> beg

struct FChunk {          // 16 bytes, one broadcast load
  uint32_t slot0;        // slot of lane 0
  uint32_t heads;        // bit l: lane l is the first (proximal) control volume of its branch
  uint32_t tails;        // bit l: lane l is the last (distal) control volume of its branch
  uint32_t br_n;         // (branch of lane 0) * 64 + number of valid lanes (1..32); lanes beyond carry both bits
};

struct FBranch {         // 16 bytes, in slot order
  uint32_t slot0;        // slot of its first control volume
  uint32_t pslot;        // slot of the parent control volume of slot0, or kNoSlot
  uint32_t cbeg;         // first entry of its child list; with kFBranchInlineFlag: child0 | child1 << 16
  uint16_t len;          // control volumes
  uint16_t ccnt;         // child branches hanging off its last control volume (| kFBranchInlineFlag)
};
constexpr uint32_t kFBranchInlineChildren = 2;
constexpr uint16_t kFBranchInlineFlag = 0x8000u;   // (a branch has fewer than 32,768 children)

// Byte offsets inside a forest's tree record (every section 16-byte aligned).
struct FTopoOff { uint32_t offs, runs, chunks, chunk_cells, branches, br_cell, child, cell_det, level_br, total; };
// The record starts with a table of the offsets a CTA needs (FOffs), filled by the host, so that the kernel reads
// them from shared memory instead of recomputing three dozen aligned sums per thread.
struct FOffs {
  uint32_t fast[18];     // bytes into the fast record, in the order of FastOff (f ... cl_cell)
  uint32_t state[6];     // doubles into the state record: v, m, h, n, g, rt
  uint32_t gen[6];       // doubles into the gen record: C, S, sig, G, b, syn_tau
  uint32_t topo[8];      // bytes into this record: runs, chunks, chunk_cells, branches, br_cell, child, cell_det, level_br
  uint32_t scratch[3];   // doubles into the scratch record: fgen, invdgen, dcon
  uint32_t pad[23];
};
static_assert(sizeof(FOffs) == 256, "FOffs must be 256 bytes");
ARBB_HD FTopoOff ftopo_offsets(uint32_t n_level, uint32_t n_chunk, uint32_t n_branch, uint32_t n_child, uint32_t n_cell, uint32_t n_warp) {
  FTopoOff o;
  uint32_t p = 0;
  auto sec = [&](uint32_t bytes) { uint32_t at = p; p = align_up(p + bytes, 16); return at; };
  o.offs = sec((uint32_t)sizeof(FOffs));
  o.runs = sec(n_level * n_warp * (uint32_t)sizeof(FRun));
  o.chunks = sec(n_chunk * (uint32_t)sizeof(FChunk));
  o.chunk_cells = sec(n_chunk * 8);                  // uint64: bit c = the chunk holds control volumes of cell c
  o.branches = sec(n_branch * (uint32_t)sizeof(FBranch));
  o.br_cell = sec(n_branch * 2);                     // uint16: forest-local cell of every branch
  o.child = sec(n_child * 4);                        // uint32: child branches
  o.cell_det = sec(n_cell * 4);                      // uint32: slot of every cell's detector
  o.level_br = sec((n_level + 1) * 4);               // uint32: first branch of every level
  o.total = p;
  return o;
}

// Shared memory of one CTA of the forest kernel: the state record (V | m | h | n | g | runtime), the tree
// record, the contributions of the branches to their parents, the point currents, per-cell scratch.
// Every CTA lays out its own forest; a launch reserves what the largest forest of its class needs.
struct ForestCaps { uint32_t state_bytes, topo_bytes, n_branch, n_spec, n_cell; };
struct ForestSmemPlan { uint32_t off_topo, off_con, off_xi, off_cell, bytes; };
ARBB_HD ForestSmemPlan forest_smem_plan(const ForestCaps& c) {
  ForestSmemPlan P;
  uint32_t p = align_up(c.state_bytes, 128);
  P.off_topo = p; p = align_up(p + c.topo_bytes, 16);
  P.off_con = p;  p = align_up(p + 8 * c.n_branch, 16);
  P.off_xi = p;   p = align_up(p + 16 * c.n_spec, 16);    // currents (sources | conductances when linearised)
  P.off_cell = p; p = align_up(p + kCellScratchBytes * (c.n_cell ? c.n_cell : 1u), 16);
  P.bytes = align_up(p, 128);
  return P;
}
// upper bound of a tree record's size from counts known before the forest is built (n_level: levels of its deepest cell;
// every (level, warp) run ends in at most one partly filled chunk)
ARBB_HD uint32_t ftopo_bound(uint32_t n_cv, uint32_t n_branch, uint32_t n_cell, uint32_t n_warp, uint32_t n_level) {
  const uint32_t n_chunk = n_cv / 32 + n_warp * n_level + 1;
  return ftopo_offsets(n_level, n_chunk, n_branch, n_branch, n_cell, n_warp).total;
}
// shared-memory budget of launch class k (bytes per CTA so that 8 >> k CTAs share an SM's 227 KB)
// (1 KB per CTA is reserved by the system; the kernel's static shared memory is below 1 KB)
ARBB_HD uint32_t forest_class_budget(int k) { return ((227u * 1024u) >> (3 - k)) - 2048u; }

struct ForestClass {     // one launch: forests [first, first + count) of the unit list
  int64_t first, count;
  int n_warp;            // warps per CTA of the launch
  ForestSmemPlan plan;
};

// Double offsets inside a forest's scratch record (global memory; event-split sub-steps and the
// factorisation only): factors for a sub-step's own step length, and what a branch's parent loses.
struct FScratchOff { uint32_t fgen, invdgen, dcon, total; };
ARBB_HD FScratchOff fscratch_offsets(uint32_t n_slot, uint32_t n_branch) {
  FScratchOff o;
  o.fgen = 0; o.invdgen = n_slot; o.dcon = 2 * n_slot;
  o.total = align_up(2 * n_slot + n_branch, 2);
  return o;
}

}  // namespace arbb
