// block_layout.h - the in-HBM layout of one "cell block", shared by the host builder and the kernels.
//
// A cell block is the unit of work of one CTA: a handful of cells whose branches (maximal
// unbranched chains of control volumes) are interleaved so that consecutive lanes of a warp read
// consecutive addresses ("SoA with interleaved branches", BASELINE.json north_star; the paper's
// own GPU layout interleaves whole cells, one thread per cell, PAPER.md:220 - prior art).
//
//   level l of the block   = all branches whose distance (in branches) from their cell's root is l
//   task                   = up to 32 branches of one level, sorted by length; one warp, lane = branch
//   slot(task, k, lane)    = task.slot_off + k * task.width + lane      k = 0 proximal .. len-1 distal
//
// Per block there are four contiguous records in the device workspace:
//   gen   (doubles, constant)  [Cg | Sg | sig | Gg | bg]              x n_slot   dt-independent
//   fast  (doubles, per dt)    [f | invd | a | b]                      x n_slot   written by factor_kernel
//         followed by          [hh_gna|hh_gk|hh_gl] x n_hh, [syn_e|syn_decay|syn_tau] x n_syn,
//                              [cl_t0|cl_t1|cl_amp] x n_clamp
//   state (doubles, mutable)   [V x n_slot | m | h | n x n_hh | g x n_syn]
//   meta  (bytes, constant)    tasks, level table, per-branch links, specials, ... (offsets below)
#pragma once
#include <stdint.h>

#if defined(__CUDACC__)
#define ARBB_HD __host__ __device__ __forceinline__
#else
#define ARBB_HD inline
#endif

namespace arbb {

constexpr uint32_t kNoSlot = 0xFFFFFFFFu;
constexpr int kWarp = 32;

struct Task {            // 16 bytes
  uint32_t slot_off;     // slot of (k = 0, lane = 0)
  uint32_t lane_off;     // block-local branch index of lane 0
  uint16_t width;        // row stride in slots (nlanes rounded up to 4)
  uint16_t nlanes;       // 1..32
  uint16_t maxlen;       // longest branch of the task
  uint16_t level;
};

struct BlockInfo {       // one per block, read by every thread of the CTA
  int64_t gen_base;      // double index into the gen pool
  int64_t fast_base;     // double index into the fast pool
  int64_t state_base;    // double index into the state pool
  int64_t meta_base;     // byte index into the meta pool (16-byte aligned)
  int64_t cell_base;     // internal index of the block's first cell
  int64_t scratch_base;  // double index into the scratch pool (2*n_slot + 2*n_lane doubles) or -1
  uint32_t n_slot, n_lane, n_task, n_level;
  uint32_t n_cell, n_hh, n_syn, n_sp;
  uint32_t n_clamp, n_child, meta_bytes, flags;
};

ARBB_HD uint32_t align_up(uint32_t x, uint32_t a) { return (x + a - 1) / a * a; }

// Byte offsets of the sections of a block's meta blob (every section 16-byte aligned).
struct MetaOff {
  uint32_t tasks, level_begin, br_pslot, br_cbeg, br_len, br_cell, br_ccnt, child, cell_det,
      hh_slot, hh_cell, syn_cell, sp_slot, sp_hh, sp_syn_beg, sp_cl_beg, sp_syn_cnt, sp_cl_cnt,
      sp_cell, total;
};

ARBB_HD MetaOff meta_offsets(const BlockInfo& b) {
  MetaOff o;
  uint32_t p = 0;
  auto sec = [&](uint32_t bytes) { uint32_t at = p; p = align_up(p + bytes, 16); return at; };
  o.tasks = sec(b.n_task * 16);
  o.level_begin = sec((b.n_level + 1) * 4);
  o.br_pslot = sec(b.n_lane * 4);
  o.br_cbeg = sec(b.n_lane * 4);
  o.br_len = sec(b.n_lane * 2);
  o.br_cell = sec(b.n_lane * 2);
  o.br_ccnt = sec(b.n_lane * 2);
  o.child = sec(b.n_child * 4);
  o.cell_det = sec(b.n_cell * 4);
  o.hh_slot = sec(b.n_hh * 4);
  o.hh_cell = sec(b.n_hh * 2);
  o.syn_cell = sec(b.n_syn * 2);
  o.sp_slot = sec(b.n_sp * 4);
  o.sp_hh = sec(b.n_sp * 4);
  o.sp_syn_beg = sec(b.n_sp * 4);
  o.sp_cl_beg = sec(b.n_sp * 4);
  o.sp_syn_cnt = sec(b.n_sp * 2);
  o.sp_cl_cnt = sec(b.n_sp * 2);
  o.sp_cell = sec(b.n_sp * 2);
  o.total = p;
  return o;
}

// double offsets inside the fast record
struct FastOff { uint32_t f, invd, a, b, hh_gna, hh_gk, hh_gl, syn_e, syn_decay, syn_tau, cl_t0, cl_t1, cl_amp, total; };
ARBB_HD FastOff fast_offsets(const BlockInfo& b) {
  FastOff o;
  uint32_t p = 0;
  auto sec = [&](uint32_t n) { uint32_t at = p; p = align_up(p + n, 2); return at; };  // 16-byte aligned
  o.f = sec(b.n_slot); o.invd = sec(b.n_slot); o.a = sec(b.n_slot); o.b = sec(b.n_slot);
  o.hh_gna = sec(b.n_hh); o.hh_gk = sec(b.n_hh); o.hh_gl = sec(b.n_hh);
  o.syn_e = sec(b.n_syn); o.syn_decay = sec(b.n_syn); o.syn_tau = sec(b.n_syn);
  o.cl_t0 = sec(b.n_clamp); o.cl_t1 = sec(b.n_clamp); o.cl_amp = sec(b.n_clamp);
  o.total = align_up(p, 16);
  return o;
}

// double offsets inside the state record
struct StateOff { uint32_t v, m, h, n, g, total; };
ARBB_HD StateOff state_offsets(const BlockInfo& b) {
  StateOff o;
  uint32_t p = 0;
  auto sec = [&](uint32_t n) { uint32_t at = p; p = align_up(p + n, 2); return at; };
  o.v = sec(b.n_slot); o.m = sec(b.n_hh); o.h = sec(b.n_hh); o.n = sec(b.n_hh); o.g = sec(b.n_syn);
  o.total = align_up(p, 16);
  return o;
}

// gen record: five arrays of n_slot doubles (n_slot is a multiple of 16)
struct GenOff { uint32_t C, S, sig, G, b, total; };
ARBB_HD GenOff gen_offsets(const BlockInfo& bi) {
  GenOff o;
  o.C = 0; o.S = bi.n_slot; o.sig = 2 * bi.n_slot; o.G = 3 * bi.n_slot; o.b = 4 * bi.n_slot;
  o.total = 5 * bi.n_slot;
  return o;
}

// Per-cell runtime state (internal cell order), kept in global memory between launches.
struct CellRt {
  uint32_t ev_cur;     // next undelivered event of the current epoch list
  uint32_t ev_end;     // end of this cell's segment in the epoch list
  uint32_t armed;      // threshold detector armed (reading R10)
  uint32_t pad;
};

}  // namespace arbb
