// group_layout.h - the in-HBM layout of a "cell group", shared by the host builder and the kernels.
//
// Cells with identical trees (same parent array) form a topology CLASS.  A class is cut into
// GROUPS of kG cells; a group is stored CELL-INTERLEAVED: row s of an array holds the value of
// control volume `slot s` for the kG cells of the group (kG * 8 contiguous bytes), and the rows of
// one array are contiguous, so that kG consecutive lanes (one "lane group", lane = cell) read
// consecutive addresses while they walk the tree.  (The paper's GPU solver interleaves whole cell
// matrices with one thread per cell; here several lane groups and several warps walk
// different subtrees of the same cells at the same time.)
//
//   segment   a maximal unbranched chain of control volumes; its slots are consecutive
//             (slot0 = proximal end).  One lane group eliminates a segment serially, carrying the
//             recurrence in a register.
//   chunk     a connected set of segments that one lane group eliminates one after the other
//   stage     chunks that do not depend on each other; the CTA's lane groups run them
//             concurrently, __syncthreads separates stages.  Backward (leaves -> root) runs stages
//             0..n_stage-1, forward (root -> leaves) runs them in reverse, segments reversed.
//
// Per class there is one ClassRecord in the topo pool (the kernel keeps the current one in shared memory).
// Per group there are three records:
//   const (fast pool, bytes)   f | invd | a | b | hh gna, gk, gl | syn e, decay (non-uniform only) |
//                              clamp t0, t1, amp | hh_slot | syn_slot | cl_slot | det_slot
//   state (state pool, doubles) V | g | per-cell runtime triples [cell][3] | m | h | n
//   gen   (gen pool, doubles)   C | S | sigma | G | bg | syn_tau   (dt-independent; factorisation
//                              and event-split sub-steps only)
// Rows of per-instance arrays (HH, synapses, clamps): row j = the j-th instance of every cell in
// ascending (slot, caller's index) order; cells with fewer instances are padded with slot kNoSlot16.
#pragma once
#include <stdint.h>

#include "unit_layout.h"

namespace arbb {

constexpr int kG = 4;                         // cells per group = lanes per lane group (4, 8, 16 or 32)
constexpr int kLaneGroups = 32 / kG;          // lane groups per warp
constexpr int kGroupWarps = 4;                // warps per CTA of the group kernel
constexpr int kGroupThreads = kGroupWarps * 32;
constexpr int kGroupMinCtas = 4;              // resident CTAs per SM the kernel is compiled for
constexpr int kGroupSlots = kGroupWarps * kLaneGroups;   // chunks a stage can run concurrently
constexpr uint16_t kNoSlot16 = 0xFFFFu;
constexpr uint32_t kGroupMaxCv = 65000;       // slots are stored as uint16

// Position of element (slot, cell) inside a per-control-volume array of a group: the linear index
// slot * kG + cell with the 16-byte chunk index inside each 128-byte line XORed with the line index
// (the TMA "128B swizzle" pattern, applied to the HBM layout itself so that linear bulk copies keep
// it).  Lane groups that walk rows 8 apart then fall on different shared-memory banks.  An involution;
// all per-CV arrays of a group (V, f, 1/d, a, b, C, S, sigma, G, bg) use the same positions, so
// element-wise loops may run over raw positions.
ARBB_HD uint32_t gswz(uint32_t e) { return e ^ (((e >> 4) & 7u) << 1); }
ARBB_HD uint32_t gpos(uint32_t slot, uint32_t cell) { return gswz(slot * (uint32_t)kG + cell); }
// positions of a per-CV array: whole 128-byte lines (the swizzle permutes inside a line)
ARBB_HD uint32_t gcv_elems(uint32_t n_cv) { return align_up(n_cv * (uint32_t)kG, 16); }

constexpr uint32_t kSegInlineChildren = 2;   // a segment with at most this many children carries them in its record
struct SegRec {          // 16 bytes, one broadcast load per lane group
  uint32_t slot0;        // slot of the proximal control volume
  uint32_t pslot;        // slot of the parent control volume of slot0, or kNoSlot
  uint16_t len;          // control volumes in the segment
  uint16_t ccnt;         // child segments hanging off its last control volume
  uint32_t cbeg;         // ccnt <= kSegInlineChildren: child0 | child1 << 16; else first entry of its child list
};

struct ClassRecord {     // header of a class record; arrays follow at the byte offsets below
  uint32_t n_cv, n_seg, n_stage, n_child;
  uint32_t off_segs;     // SegRec[n_seg]
  uint32_t off_order;    // uint16[n_seg]: the identity (segments ARE numbered in backward processing order, grouped by
                         // (stage, slot)); kept for the record's readers on the host, the kernels do not load it
  uint32_t off_sched;    // uint16[n_stage * kGroupSlots + 1]: begin of each (stage, slot) range in order[]
  uint32_t off_child;    // uint16[n_child]: child segments
  uint32_t bytes;
  uint32_t n_block;      // stages [0, n_block) use lane groups of several warps (block barriers between
                         // them); stages [n_block, n_stage) only use the lane groups of warp 0
  uint32_t pad[6];
};
static_assert(sizeof(ClassRecord) == 64, "ClassRecord must be 64 bytes");

struct GroupDesc {       // 64 bytes
  int64_t const_off;     // byte offset into the fast pool (128-byte aligned)
  int64_t state_base;    // double index into the state pool (16-double aligned)
  int64_t gen_base;      // double index into the gen pool
  int64_t class_off;     // byte offset of the ClassRecord in the topo pool
  int64_t cell_base;     // internal index of the group's first cell
  uint32_t n_cv, n_cell, n_hh_rows, n_syn_rows, n_cl_rows;
  uint32_t flags;        // GROUP_*
};
enum : uint32_t {
  GROUP_POINT_DISJOINT = 1u   // no two kinds of point mechanism (HH, synapse, clamp) of a cell share a control
                              // volume: their currents can be subtracted without barriers in between
};
static_assert(sizeof(GroupDesc) == 64, "GroupDesc must be 64 bytes");

// Byte offsets inside a group's const record (every section 128-byte aligned).
struct GConstOff {
  uint32_t f, invd, a, b, hh_gna, hh_gk, hh_gl, syn_e, syn_decay, cl_t0, cl_t1, cl_amp,
      hh_slot, syn_slot, cl_slot, det_slot, total;
};
ARBB_HD GConstOff gconst_offsets(uint32_t n_cv, uint32_t n_hh, uint32_t n_syn, uint32_t n_cl, bool syn_uniform) {
  GConstOff o;
  uint32_t p = 0;
  auto sec = [&](uint32_t bytes) { uint32_t at = p; p = align_up(p + bytes, 128); return at; };
  const uint32_t row = 8 * kG, row16 = 2 * kG;
  const uint32_t cvb = 8 * gcv_elems(n_cv);
  o.f = sec(cvb); o.invd = sec(cvb); o.a = sec(cvb); o.b = sec(cvb);
  o.hh_gna = sec(row * n_hh); o.hh_gk = sec(row * n_hh); o.hh_gl = sec(row * n_hh);
  o.syn_e = sec(syn_uniform ? 0 : row * n_syn); o.syn_decay = sec(syn_uniform ? 0 : row * n_syn);
  o.cl_t0 = sec(row * n_cl); o.cl_t1 = sec(row * n_cl); o.cl_amp = sec(row * n_cl);
  o.hh_slot = sec(row16 * n_hh); o.syn_slot = sec(row16 * n_syn); o.cl_slot = sec(row16 * n_cl);
  o.det_slot = sec(row16);
  o.total = p;
  return o;
}

// Double offsets inside a group's state record (every section 16-double aligned).  V | g | rt are
// what a launch writes back with one bulk store; the gates m | h | n are written by their own threads.
struct GStateOff { uint32_t v, g, rt, m, h, n, total; };
ARBB_HD GStateOff gstate_offsets(uint32_t n_cv, uint32_t n_hh, uint32_t n_syn) {
  GStateOff o;
  uint32_t p = 0;
  auto sec = [&](uint32_t n) { uint32_t at = p; p = align_up(p + n, 16); return at; };
  o.v = sec(gcv_elems(n_cv)); o.g = sec(kG * n_syn); o.rt = sec(kRtDoubles * kG);
  o.m = sec(kG * n_hh); o.h = sec(kG * n_hh); o.n = sec(kG * n_hh);
  o.total = p;
  return o;
}

// Double offsets inside a group's gen record.
struct GGenOff { uint32_t C, S, sig, G, b, syn_tau, total; };
ARBB_HD GGenOff ggen_offsets(uint32_t n_cv, uint32_t n_syn) {
  GGenOff o;
  const uint32_t n = gcv_elems(n_cv);
  o.C = 0; o.S = n; o.sig = 2 * n; o.G = 3 * n; o.b = 4 * n; o.syn_tau = 5 * n;
  o.total = align_up(5 * n + kG * n_syn, 16);
  return o;
}

// Shared memory of one CTA of the group kernel:
//   state record (V | g | rt | m | h | n) | f | 1/d | tail of the const record (hh conductances ...
//   det_slot) | class record | buf (xI, then contrib) | per-cell scratch | mbarrier
// Caps are maxima over all groups / classes of the model.
struct GroupCaps { uint32_t slot_cap, state_bytes, tail_bytes, class_bytes, buf_rows; };
struct GroupSmemPlan { uint32_t slot_cap, off_f, off_i, off_tail, off_class, off_buf, off_cell, off_mbar, bytes; };
ARBB_HD GroupSmemPlan group_smem_plan(const GroupCaps& c) {
  GroupSmemPlan P;
  P.slot_cap = c.slot_cap;
  uint32_t p = align_up(c.state_bytes, 128);
  P.off_f = p;     p = align_up(p + 8 * gcv_elems(c.slot_cap), 128);
  P.off_i = p;     p = align_up(p + 8 * gcv_elems(c.slot_cap), 128);
  P.off_tail = p;  p = align_up(p + c.tail_bytes, 128);
  P.off_class = p; p = align_up(p + c.class_bytes, 128);
  P.off_buf = p;   p = align_up(p + 8 * kG * c.buf_rows, 128);
  P.off_cell = p;  p = align_up(p + kCellScratchBytes * kG, 128);
  P.off_mbar = p;  p += 16;
  P.bytes = align_up(p, 128);
  return P;
}

}  // namespace arbb
