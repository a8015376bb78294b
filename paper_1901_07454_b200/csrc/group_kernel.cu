// group_kernel.cu - the cable step for cell groups (group_layout.h): cells of one topology class,
// stored cell-interleaved, lane = cell.
//
//   cable_group_kernel   persistent grid, one CTA integrates one group at a time, several CTAs per SM;
//                        groups are claimed from a work counter.  Everything a group-step touches lives
//                        in shared memory and arrives there by bulk-async copies (TMA, cp.async.bulk +
//                        mbarrier): the state record (V, synaptic g, per-cell runtime, gates), the tail
//                        of the const record (instance tables) and, in two coefficient buffers, first the
//                        rhs coefficients a, b and then - once the rhs is formed - the solver factors f,
//                        1/d (second pair of copies, from L2, where a TMA prefetch has put them).  V, g
//                        and the runtime leave by one bulk store.  The class record (segments, stages)
//                        is kept in shared memory.  The nominal step has no global loads.
//                        Per grid step (or fused run of steps): event delivery ->
//                        mechanism currents (eq 2a) -> rhs of the implicit Euler system
//                         -> Hines / branched Thomas sweeps: the class
//                        schedule cuts the tree into stages of independent chunks, the CTA's lane
//                        groups eliminate the chunks of a stage concurrently -> V <- V' -> gate and
//                        synapse state update with V' -> threshold test.
//                        The gate update (fp64 exp and divide chains) of a group's last step is
//                        carried in registers and overlaps the next group's copies.
//   group_factor_kernel  once per dt: eliminates the constant matrix (reading R1) of every group
//   group_init_kernel    gates at their steady state for the initial voltage (reading R4)
//
// HBM-bound by design: 48 B per control volume and step (V in + out, a, b, f, 1/d) against ~6 fp64
// instructions.  No tensor cores: nothing here is a dense contraction.
#include "device_common.cuh"
#include "group_layout.h"
#include "kernels.cuh"

namespace arbb {

namespace {

constexpr int kT = kGroupThreads;
constexpr int kCUnroll = 4;               // unrolling of the rhs loop (phase C)
constexpr int kRows = 8;                  // rows of a segment a lane group loads ahead of the recurrence


// Pointers of one group.  "s" pointers address the CTA's shared memory, "g" pointers global memory.
// Rarely used arrays (clamps, non-uniform synapse parameters, the dt-independent "gen" arrays of
// event-split sub-steps) are derived on demand, which keeps the kernel's register count down.
struct GView {
  uint32_t n_cv, n_cell, n_hh, n_syn, n_cl;          // rows
  uint32_t n_stage, n_block, flags;
  uint32_t hh_cs, hh_ss;                             // doubles between gna|gk|gl and between m|h|n
  int syn_uniform;
  const uint8_t* tail;                               // const record from hh_gna on
  const double* gen;                                 // global: gen record
  const double *a, *b;                               // global
  const double* hh_gna;
  const uint16_t *hh_slot, *syn_slot, *det_slot;
  double *sm, *sg, *srt;                             // gates m (h, n follow), g, runtime: working copy
  double* gm;                                        // global: gates m (h, n follow)
  const SegRec* segs;                                // class record
  const uint16_t *order, *sched, *child;
  int64_t cell_base;

  __device__ __forceinline__ GConstOff co() const { return gconst_offsets(n_cv, n_hh, n_syn, n_cl, syn_uniform != 0); }
  __device__ __forceinline__ const uint8_t* tl(uint32_t off) const { return tail + (off - co().hh_gna); }
  __device__ __forceinline__ const double* syn_e() const { return (const double*)tl(co().syn_e); }
  __device__ __forceinline__ const double* syn_decay() const { return (const double*)tl(co().syn_decay); }
  __device__ __forceinline__ const double* cl_t0() const { return (const double*)tl(co().cl_t0); }
  __device__ __forceinline__ const double* cl_t1() const { return (const double*)tl(co().cl_t1); }
  __device__ __forceinline__ const double* cl_amp() const { return (const double*)tl(co().cl_amp); }
  __device__ __forceinline__ const uint16_t* cl_slot() const { return (const uint16_t*)tl(co().cl_slot); }
  __device__ __forceinline__ const double* C() const { return gen + ggen_offsets(n_cv, n_syn).C; }
  __device__ __forceinline__ const double* S() const { return gen + ggen_offsets(n_cv, n_syn).S; }
  __device__ __forceinline__ const double* sig() const { return gen + ggen_offsets(n_cv, n_syn).sig; }
  __device__ __forceinline__ const double* G() const { return gen + ggen_offsets(n_cv, n_syn).G; }
  __device__ __forceinline__ const double* bg() const { return gen + ggen_offsets(n_cv, n_syn).b; }
  __device__ __forceinline__ const double* syn_tau() const { return gen + ggen_offsets(n_cv, n_syn).syn_tau; }
};

// `state`, `tail`, `cls`: where the group's state record, const-record tail and class record are
// (shared memory in the cable kernel, global memory in the factor / init kernels).
__device__ __forceinline__ void make_gview(GView& U, const DevModel& M, const GroupDesc& D, double* state, const uint8_t* tail,
                                           const uint8_t* cls) {
  U.n_cv = D.n_cv; U.n_cell = D.n_cell; U.n_hh = D.n_hh_rows; U.n_syn = D.n_syn_rows; U.n_cl = D.n_cl_rows;
  U.flags = D.flags;
  U.syn_uniform = M.syn_uniform;
  const GConstOff co = gconst_offsets(D.n_cv, D.n_hh_rows, D.n_syn_rows, D.n_cl_rows, M.syn_uniform != 0);
  const uint8_t* cb = M.fast + D.const_off;
  U.tail = tail;
  U.a = (const double*)(cb + co.a); U.b = (const double*)(cb + co.b);
  U.hh_gna = (const double*)tail; U.hh_cs = (co.hh_gk - co.hh_gna) / 8;
  U.hh_slot = (const uint16_t*)(tail + (co.hh_slot - co.hh_gna)); U.syn_slot = (const uint16_t*)(tail + (co.syn_slot - co.hh_gna));
  U.det_slot = (const uint16_t*)(tail + (co.det_slot - co.hh_gna));
  const GStateOff so = gstate_offsets(D.n_cv, D.n_hh_rows, D.n_syn_rows);
  U.sm = state + so.m; U.hh_ss = so.h - so.m; U.sg = state + so.g; U.srt = state + so.rt;
  U.gm = M.state + D.state_base + so.m;
  U.gen = M.gen + D.gen_base;
  const ClassRecord* R = (const ClassRecord*)cls;
  U.n_stage = R->n_stage; U.n_block = R->n_block;
  U.segs = (const SegRec*)(cls + R->off_segs);
  U.order = (const uint16_t*)(cls + R->off_order);
  U.sched = (const uint16_t*)(cls + R->off_sched);
  U.child = (const uint16_t*)(cls + R->off_child);
  U.cell_base = D.cell_base;
}

__device__ __forceinline__ SegRec load_seg(const SegRec* p) {
  const uint4 q = *(const uint4*)p;
  SegRec s;
  s.slot0 = q.x; s.pslot = q.y; s.len = (uint16_t)(q.z & 0xFFFFu); s.ccnt = (uint16_t)(q.z >> 16); s.cbeg = q.w;
  return s;
}
// j-th child segment of a segment (in the order a leaves -> root elimination meets them): out of the record itself
// when there are at most two (group_layout.h), else out of the class record's child list.
__device__ __forceinline__ uint32_t seg_child(const GView& U, const SegRec& sg, uint32_t j) {
  return sg.ccnt <= kSegInlineChildren ? (sg.cbeg >> (16u * j)) & 0xFFFFu : (uint32_t)U.child[sg.cbeg + j];
}

// ------------------------------------------------------------------------------------------
// Elimination of the diagonal of one segment for step length delta (factorisation; event-split
// sub-steps):  d_k = C_k/delta + S_k - sum_children sigma_c^2 / d_c ;  f_k = -sigma_k / d_k.
// dcon[segment] = sigma_0^2 / d_0 is what the parent control volume loses.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void eliminate_seg(const GView& U, const SegRec& sg, uint32_t seg_idx, int c, double delta,
                                              double* fout, double* invdout, double* dcon) {
  const double *C = U.C(), *S = U.S(), *sig = U.sig();
  constexpr int kB = 8;                   // rows whose C, S, sigma are requested together (global memory)
  uint32_t lin = (sg.slot0 + sg.len - 1) * kG + c;
  double carry = 0.0;                     // f_{k+1} * sigma_{k+1}: what row k loses to its child in the segment
  for (uint32_t j = 0; j < sg.ccnt; ++j) carry -= dcon[seg_child(U, sg, j) * kG + c];
  double fk = 0.0, sk = 0.0;
  int left = sg.len;
  while (left > 0) {
    double cr[kB], sr[kB], gr[kB];
    uint32_t p[kB];
#pragma unroll
    for (int j = 0; j < kB; ++j)
      if (j < left) { p[j] = gswz(lin - j * kG); cr[j] = C[p[j]]; sr[j] = S[p[j]]; gr[j] = sig[p[j]]; }
#pragma unroll
    for (int j = 0; j < kB; ++j)
      if (j < left) {
        const double d = (cr[j] / delta + sr[j]) + carry;
        const double invd = 1.0 / d;
        sk = gr[j];
        fk = -sk * invd;
        fout[p[j]] = fk;
        invdout[p[j]] = invd;
        carry = fk * sk;                  // d_p -= f*u with u = -sigma
      }
    lin -= kB * kG;
    left -= kB;
  }
  dcon[seg_idx * kG + c] = -fk * sk;
}

// Re-elimination for an event-split sub-step of length delta = dt / r, out of shared memory and
// without the dt-independent arrays: F, I hold this cell's NOMINAL f_k, 1/d_k and are replaced by the
// ones for delta.  With sigma_k = -f_k d_k and q_c = sigma_c (1 + f_c) for the children c of k,
//     C_k/dt = d_k - sigma_k - sum_c q_c      and      d'_k = r C_k/dt + sigma_k + sum_c q'_c,
// so   d'_k = r (d_k - sigma_k) + sigma_k + sum_c z_c   with   z_c = q'_c - r q_c ,
// which only needs one number per child (carried along a segment, zcon[] across segments).
__device__ __forceinline__ void eliminate_seg_smem(const GView& U, const SegRec& sg, uint32_t seg_idx, int c, double r,
                                                   double* F, double* I, double* zcon) {
  uint32_t lin = (sg.slot0 + sg.len - 1) * kG + c;
  double z = 0.0;
  for (uint32_t j = 0; j < sg.ccnt; ++j) z += zcon[seg_child(U, sg, j) * kG + c];
#pragma unroll 2
  for (int left = sg.len; left > 0; --left, lin -= kG) {
    const uint32_t p = gswz(lin);
    const double f0 = F[p], d0 = 1.0 / I[p];
    const double sk = -f0 * d0;
    const double d1 = fma(r, d0 - sk, sk) + z;
    const double invd = 1.0 / d1;
    const double f1 = -sk * invd;
    F[p] = f1;
    I[p] = invd;
    z = sk * ((1.0 + f1) - r * (1.0 + f0));
  }
  zcon[seg_idx * kG + c] = z;
}

// Elimination for the conductance-linearised step (PAPER.md:152-156 with the membrane
// conductances on the diagonal): F holds the assembled diagonal C/delta + sum(sigma) + sum(g) of this cell, I its
// link conductances sigma; both are replaced by f_k = -sigma_k / d_k and 1 / d_k.  The same recurrence as the
// oracle's Hines elimination: d_parent -= sigma_c^2 / d_c.
__device__ __forceinline__ void eliminate_seg_lin(const GView& U, const SegRec& sg, uint32_t seg_idx, int c, double* F, double* I, double* dcon) {
  uint32_t lin = (sg.slot0 + sg.len - 1) * kG + c;
  double carry = 0.0;                     // f_{k+1} sigma_{k+1}: what row k loses to its child in the segment
  for (uint32_t j = 0; j < sg.ccnt; ++j) carry -= dcon[seg_child(U, sg, j) * kG + c];
  double fk = 0.0, sk = 0.0;
#pragma unroll 2
  for (int left = sg.len; left > 0; --left, lin -= kG) {
    const uint32_t p = gswz(lin);
    const double invd = 1.0 / (F[p] + carry);
    sk = I[p];
    fk = -sk * invd;
    F[p] = fk;
    I[p] = invd;
    carry = fk * sk;
  }
  dcon[seg_idx * kG + c] = -fk * sk;
}

// ------------------------------------------------------------------------------------------
// Backward (leaves -> root) sweep of one segment on the rhs held in Vs:
//   rhs_{k-1} -= f_k rhs_k along the segment; the parent control volume loses con[segment] = f_0 rhs_0;
// every control volume is left holding rhs_k / d_k, which is what the forward sweep needs.
// F, I: the factors f and 1/d (shared memory; the cell's own re-elimination on event-split sub-steps).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void backward_seg(const GView& U, const SegRec& sg, uint32_t seg_idx, int c,
                                             const double* __restrict__ F, const double* __restrict__ I,
                                             double* Vs, double* con) {
  uint32_t s = (sg.slot0 + sg.len - 1) * kG + c;
  double fp = 0.0, rp = 0.0;
  int left = sg.len;
  bool first = true;
  while (left >= kRows) {                 // whole blocks: no predication
    double fr[kRows], ir[kRows], vr[kRows];
    uint32_t p[kRows];
#pragma unroll
    for (int j = 0; j < kRows; ++j) { p[j] = gswz(s - j * kG); fr[j] = F[p[j]]; ir[j] = I[p[j]]; vr[j] = Vs[p[j]]; }
    if (first) {
#pragma unroll 1
      for (uint32_t j = 0; j < sg.ccnt; ++j) vr[0] -= con[seg_child(U, sg, j) * kG + c];
      first = false;
    }
#pragma unroll
    for (int j = 0; j < kRows; ++j) {
      const double r = fma(-fp, rp, vr[j]);
      Vs[p[j]] = r * ir[j];
      fp = fr[j]; rp = r;
    }
    s -= kRows * kG;
    left -= kRows;
  }
#pragma unroll 1
  for (; left > 0; --left, s -= kG) {
    const uint32_t p = gswz(s);
    double v = Vs[p];
    if (first) {
#pragma unroll 1
      for (uint32_t j = 0; j < sg.ccnt; ++j) v -= con[seg_child(U, sg, j) * kG + c];
      first = false;
    }
    const double r = fma(-fp, rp, v);
    Vs[p] = r * I[p];
    fp = F[p]; rp = r;
  }
  con[seg_idx * kG + c] = fp * rp;
}

// Forward (root -> leaves) substitution of one segment: V'_k = rhs_k/d_k - f_k V'_{k-1}; V <- V'.
__device__ __forceinline__ void forward_seg(const SegRec& sg, int c, const double* __restrict__ F, double* Vs) {
  double vp = sg.pslot != kNoSlot ? Vs[gpos(sg.pslot, c)] : 0.0;
  uint32_t s = sg.slot0 * kG + c;
  int left = sg.len;
  while (left >= kRows) {
    double fr[kRows], vr[kRows];
    uint32_t p[kRows];
#pragma unroll
    for (int j = 0; j < kRows; ++j) { p[j] = gswz(s + j * kG); fr[j] = F[p[j]]; vr[j] = Vs[p[j]]; }
#pragma unroll
    for (int j = 0; j < kRows; ++j) {
      vp = fma(-fr[j], vp, vr[j]);
      Vs[p[j]] = vp;
    }
    s += kRows * kG;
    left -= kRows;
  }
#pragma unroll 1
  for (; left > 0; --left, s += kG) {
    const uint32_t p = gswz(s);
    vp = fma(-F[p], vp, Vs[p]);
    Vs[p] = vp;
  }
}

__device__ __forceinline__ void backward_stage(const GView& U, uint32_t st, int h, int c, bool on, const double* F,
                                               const double* I, double* Vs, double* con) {
  const uint32_t beg = U.sched[st * kGroupSlots + h], end = U.sched[st * kGroupSlots + h + 1];
  if (on)
    for (uint32_t q = beg; q < end; ++q) {
      const uint32_t si = q;
      backward_seg(U, load_seg(U.segs + si), si, c, F, I, Vs, con);
    }
}
__device__ __forceinline__ void forward_stage(const GView& U, uint32_t st, int h, int c, bool on, const double* F, double* Vs) {
  const uint32_t beg = U.sched[st * kGroupSlots + h], end = U.sched[st * kGroupSlots + h + 1];
  if (on)
    for (uint32_t q = end; q-- > beg;) forward_seg(load_seg(U.segs + q), c, F, Vs);
}

// Both sweeps.  Stages [0, n_block) hold chunks on lane groups of several warps: block barriers.
// Stages [n_block, n_stage) only use the lane groups of warp 0: it runs them back to back, backward
// and then forward, with warp barriers only.
__device__ __forceinline__ void sweeps(const GView& U, int h, int c, bool on, const double* F, const double* I,
                                       double* Vs, double* con) {
  const uint32_t n_stage = U.n_stage, n_block = U.n_block;
  for (uint32_t st = 0; st < n_block; ++st) {
    backward_stage(U, st, h, c, on, F, I, Vs, con);
    __syncthreads();
  }
  if (threadIdx.x < 32) {
    for (uint32_t st = n_block; st < n_stage; ++st) {
      backward_stage(U, st, h, c, on, F, I, Vs, con);
      __syncwarp();
    }
    for (uint32_t st = n_stage; st-- > n_block;) {
      forward_stage(U, st, h, c, on, F, Vs);
      __syncwarp();
    }
  }
  for (uint32_t st = n_block; st-- > 0;) {
    __syncthreads();
    forward_stage(U, st, h, c, on, F, Vs);
  }
}

// ------------------------------------------------------------------------------------------
// HH gate update x <- x_inf(V') + (x - x_inf) exp(-delta (alpha + beta)) (reading R5),
// deferred: phase F only captures (V', delta, m, h, n) in registers; the exp / divide chains run
// later, off the critical path of the CTA.
// ------------------------------------------------------------------------------------------
constexpr int kHHDefer = 1;       // HH instances per thread that can be deferred

struct HHDefer {
  double v[kHHDefer], delta[kHHDefer], m[kHHDefer], h[kHHDefer], n[kHHDefer];
  uint32_t e[kHHDefer];           // kNoSlot: empty
};
__device__ __forceinline__ void clear(HHDefer& d) {
#pragma unroll
  for (int i = 0; i < kHHDefer; ++i) d.e[i] = kNoSlot;
}

// not inlined: the exp / expm1 / divide chains are ~1,000 instructions and there are several call sites
__device__ __noinline__ void hh_gates(double v, double delta, double& m, double& h, double& n) {
  const Rates r = hh_rates(v);
  double inf = r.am / (r.am + r.bm);
  m = inf + (m - inf) * exp(-delta * (r.am + r.bm));
  inf = r.ah / (r.ah + r.bh);
  h = inf + (h - inf) * exp(-delta * (r.ah + r.bh));
  inf = r.an / (r.an + r.bn);
  n = inf + (n - inf) * exp(-delta * (r.an + r.bn));
}

// run the deferred updates; results go to dst0 and (when not null) dst1: m at [e], h and n at +ss, +2 ss
__device__ __forceinline__ void run_deferred(HHDefer& dh, double* dst0, double* dst1, uint32_t ss) {
#pragma unroll
  for (int i = 0; i < kHHDefer; ++i)
    if (dh.e[i] != kNoSlot) {
      double m = dh.m[i], h = dh.h[i], n = dh.n[i];
      hh_gates(dh.v[i], dh.delta[i], m, h, n);
      double* p = dst0 + dh.e[i];
      p[0] = m; p[ss] = h; p[2 * ss] = n;
      if (dst1) { p = dst1 + dh.e[i]; p[0] = m; p[ss] = h; p[2 * ss] = n; }
      dh.e[i] = kNoSlot;
    }
}

// ------------------------------------------------------------------------------------------
// One (sub-)step of every active cell of the group (phases B..F; phase A, event delivery and the
// choice of the sub-step, is in the kernel body).  Point-mechanism instances are dealt to threads
// from the END of the CTA (thread kT-1 first) so that they do not land on warp 0, which owns the
// serial parts (phase A, the narrow stages).  The HH gate updates come back deferred in `dh`.
// ------------------------------------------------------------------------------------------
// kLin: the conductance-linearised step (ARB_OPT_LINEARISED).  The four coefficient arrays of the const record then
// hold C/dt, G e, C/dt + sum(sigma) + G and sigma (group_factor_kernel): phase B computes every point mechanism's
// conductance and source g E instead of its current, the sources are added to the rhs, the conductances to the
// diagonal, and every cell's matrix is eliminated in shared memory before the sweeps.
template <bool kGen, bool kLin>
__device__ __forceinline__ void group_substep(const DevModel& M, const GView& U, double* Vs, const double* Fs, const double* Is,
                                              double* buf, const CellS& cs, double dt, HHDefer& dh, double vprev, double tstart,
                                              const uint8_t* fg, uint32_t vbytes, uint64_t* mbarB, uint32_t& parB) {
  const int tid = threadIdx.x, c = tid % kG, h = tid / kG;
  const int rtid = kT - 1 - tid, rc = rtid % kG;      // reversed dealing of instances; cell of those
  const uint32_t nE_cv = gcv_elems(U.n_cv), nE_hh = U.n_hh * kG, nE_syn = U.n_syn * kG, nE_cl = U.n_cl * kG;
  const uint32_t md = kGen ? cs.mode[c] : 1u, rmd = kGen ? cs.mode[rc] : 1u;
  const double rdelta = kGen ? cs.delta[rc] : dt;
  // ---- B: currents of HH, synapses and clamps from V(t); the passive current is
  // folded into a, b.  Items of one cell on one CV form a run; its first item sums it in index order.
  double* xI = buf;
#pragma unroll 1
  for (uint32_t e = rtid; e < nE_hh; e += kT) {
    const uint32_t slot = U.hh_slot[e];
    if (slot == kNoSlot16 || !rmd) continue;
    const double v = Vs[gpos(slot, rc)];
    const double m = U.sm[e], hh = U.sm[e + U.hh_ss], n = U.sm[e + 2 * U.hh_ss];
    if (!kLin) {
      xI[e] = U.hh_gna[e] * m * m * m * hh * (v - M.ena) + U.hh_gna[e + U.hh_cs] * n * n * n * n * (v - M.ek) +
              U.hh_gna[e + 2 * U.hh_cs] * (v - M.el);
    } else {
      const double gna = U.hh_gna[e] * m * m * m * hh, gk = U.hh_gna[e + U.hh_cs] * n * n * n * n, gl = U.hh_gna[e + 2 * U.hh_cs];
      xI[e] = gna * M.ena + gk * M.ek + gl * M.el;
    }
  }
#pragma unroll 1
  for (uint32_t e = rtid; e < nE_syn; e += kT) {
    const uint32_t slot = U.syn_slot[e];
    if (slot == kNoSlot16 || !rmd) continue;
    if (e >= (uint32_t)kG && U.syn_slot[e - kG] == slot) continue;
    const double v = Vs[gpos(slot, rc)];
    double I = 0.0;
    uint32_t j = e;
    do {
      const double es = M.syn_uniform ? M.syn_e_u : U.syn_e()[j];
      if (!kLin) I += U.sg[j] * (v - es);
      else I += U.sg[j] * es;
      j += kG;
    } while (j < nE_syn && U.syn_slot[j] == slot);
    xI[nE_hh + e] = I;
  }
  if (nE_cl) {
    const double t = kGen ? cs.tcur[rc] : tstart;
    const uint16_t* cl_slot = U.cl_slot();
    const double *cl_t0 = U.cl_t0(), *cl_t1 = U.cl_t1(), *cl_amp = U.cl_amp();
    for (uint32_t e = rtid; e < nE_cl; e += kT) {
      const uint32_t slot = cl_slot[e];
      if (slot == kNoSlot16 || !rmd) continue;
      if (e >= (uint32_t)kG && cl_slot[e - kG] == slot) continue;
      double I = 0.0;
      uint32_t j = e;
      do {
        if (cl_t0[j] <= t && t < cl_t1[j]) I -= cl_amp[j];
        j += kG;
      } while (j < nE_cl && cl_slot[j] == slot);
      xI[nE_hh + nE_syn + e] = kLin ? -I : I;          // kLin: sources are ADDED to the rhs
    }
  }
  __syncthreads();

  // ---- C: rhs_i = (C_i/delta - G_i) V_i + G_i e_i - I_i, in place of V; positions, not
  // (slot, cell) pairs: every per-CV array of the group uses the same positions
  // (a, b sit in the two coefficient buffers, Fs and Is, until the rhs is formed)
  if (!kGen) {
#pragma unroll kCUnroll
    for (uint32_t p = tid; p < nE_cv; p += kT) Vs[p] = fma(Fs[p], Vs[p], Is[p]);
  } else {
    // every position p = tid + j * kT a thread visits belongs to the same cell: kT is a multiple of
    // 128 positions, the period of the swizzle
    static_assert(kT % 128 == 0, "element-wise loops assume one cell per thread");
    const uint32_t pcell = gswz((uint32_t)tid) % kG, pmd = cs.mode[pcell];
    double* __restrict__ Vr = Vs;                            // no aliasing: the loads may run ahead of the stores
    if (pmd == 1u) {
      const double* __restrict__ ar = Fs; const double* __restrict__ br = Is;
#pragma unroll 4
      for (uint32_t p = tid; p < nE_cv; p += kT) Vr[p] = fma(ar[p], Vr[p], br[p]);
    } else if (pmd == 2u) {
      // (C/delta - G) V + G e  with  C/delta - G = a + (r - 1) C/dt  and  G e = b   (kLin: a = C/dt, C/delta = r a)
      const double* __restrict__ ar = Fs; const double* __restrict__ br = Is; const double* __restrict__ C = U.C();
      const double rm1 = dt / cs.delta[pcell] - 1.0;
#pragma unroll 4
      for (uint32_t p = tid; p < nE_cv; p += kT) Vr[p] = fma(fma(rm1, C[p] / dt, ar[p]), Vr[p], br[p]);
    }
  }
  __syncthreads();
  // a, b are dead: the same two buffers now receive the solver factors f, 1/d (L2, prefetched) while
  // the point currents are subtracted
  if (tid == 0) {
    fence_proxy_async();
    mbar_expect_tx(mbarB, 2u * vbytes);
    bulk_g2s((void*)Fs, fg, vbytes, mbarB);
    bulk_g2s((void*)Is, fg + vbytes, vbytes, mbarB);
  }
  // HH, synapse and clamp currents of a cell may meet on a control volume: barriers in between, unless
  // the host found that they never do in this group
  const bool disjoint = (U.flags & GROUP_POINT_DISJOINT) != 0;
  if (nE_hh) {
  #pragma unroll 1
  for (uint32_t e = rtid; e < nE_hh; e += kT) {
      const uint32_t slot = U.hh_slot[e];
      if (slot == kNoSlot16 || !rmd) continue;
      if (!kLin) Vs[gpos(slot, rc)] -= xI[e]; else Vs[gpos(slot, rc)] += xI[e];
    }
    if (!disjoint) __syncthreads();
  }
  if (nE_syn) {
  #pragma unroll 1
  for (uint32_t e = rtid; e < nE_syn; e += kT) {
      const uint32_t slot = U.syn_slot[e];
      if (slot == kNoSlot16 || !rmd) continue;
      if (e >= (uint32_t)kG && U.syn_slot[e - kG] == slot) continue;
      if (!kLin) Vs[gpos(slot, rc)] -= xI[nE_hh + e]; else Vs[gpos(slot, rc)] += xI[nE_hh + e];
    }
    if (!disjoint) __syncthreads();
  }
  if (nE_cl) {
    const uint16_t* cl_slot = U.cl_slot();
    for (uint32_t e = rtid; e < nE_cl; e += kT) {
      const uint32_t slot = cl_slot[e];
      if (slot == kNoSlot16 || !rmd) continue;
      if (e >= (uint32_t)kG && cl_slot[e - kG] == slot) continue;
      if (!kLin) Vs[gpos(slot, rc)] -= xI[nE_hh + nE_syn + e]; else Vs[gpos(slot, rc)] += xI[nE_hh + nE_syn + e];
    }
    if (!disjoint) __syncthreads();
  }
  if (disjoint && (nE_hh | nE_syn | nE_cl)) __syncthreads();
  mbar_wait(mbarB, parB);
  parB ^= 1u;
  if (kLin) {
    // the coefficient buffers now hold the assembled diagonal without the point mechanisms and sigma: add the
    // conductances (recomputed from the gates and the synaptic g, which phase B left untouched; different kinds may
    // share a control volume: in turn), on event-split sub-steps the larger C/delta, then eliminate every cell's
    // matrix, stage by stage
    double* F = const_cast<double*>(Fs);
    double* I = const_cast<double*>(Is);
#pragma unroll 1
    for (uint32_t e = rtid; e < nE_hh; e += kT) {
      const uint32_t slot = U.hh_slot[e];
      if (slot == kNoSlot16 || !rmd) continue;
      const double m = U.sm[e], hh = U.sm[e + U.hh_ss], n = U.sm[e + 2 * U.hh_ss];
      F[gpos(slot, rc)] += (U.hh_gna[e] * m * m * m * hh + U.hh_gna[e + U.hh_cs] * n * n * n * n) + U.hh_gna[e + 2 * U.hh_cs];
    }
    __syncthreads();
#pragma unroll 1
    for (uint32_t e = rtid; e < nE_syn; e += kT) {
      const uint32_t slot = U.syn_slot[e];
      if (slot == kNoSlot16 || !rmd) continue;
      if (e >= (uint32_t)kG && U.syn_slot[e - kG] == slot) continue;
      double G = 0.0;
      uint32_t j = e;
      do { G += U.sg[j]; j += kG; } while (j < nE_syn && U.syn_slot[j] == slot);
      F[gpos(slot, rc)] += G;
    }
    if (kGen) {
      __syncthreads();
      const uint32_t pcell = gswz((uint32_t)tid) % kG;
      if (cs.mode[pcell] == 2u) {
        const double* __restrict__ C = U.C();
        const double rm1 = dt / cs.delta[pcell] - 1.0;
        for (uint32_t p = tid; p < nE_cv; p += kT) F[p] = fma(rm1, C[p] / dt, F[p]);
      }
    }
    __syncthreads();
    for (uint32_t st = 0; st < U.n_stage; ++st) {
      const uint32_t beg = U.sched[st * kGroupSlots + h], end = U.sched[st * kGroupSlots + h + 1];
      if (!kGen || md != 0u)
        for (uint32_t q = beg; q < end; ++q) {
          const uint32_t si = q;
          eliminate_seg_lin(U, load_seg(U.segs + si), si, c, F, I, buf);
        }
      __syncthreads();
    }
  }
  // ---- event-split sub-steps: this cell's matrix is re-eliminated for its own delta (reading R9); its
  // column of the shared-memory factors is overwritten (every (sub-)step copies them afresh)
  if (kGen && !kLin) {
    double* F = const_cast<double*>(Fs);
    double* I = const_cast<double*>(Is);
    for (uint32_t st = 0; st < U.n_stage; ++st) {
      const uint32_t beg = U.sched[st * kGroupSlots + h], end = U.sched[st * kGroupSlots + h + 1];
      if (md == 2u)
        for (uint32_t q = beg; q < end; ++q) {
          const uint32_t si = q;
          eliminate_seg_smem(U, load_seg(U.segs + si), si, c, dt / cs.delta[c], F, I, buf);
        }
      __syncthreads();
    }
  }

  // ---- D: backward sweep, stage by stage; E: forward substitution, stages reversed; V <- V'
  sweeps(U, h, c, kGen ? md != 0u : true, Fs, Is, Vs, buf);   // buf: xI is dead, it now holds the contributions
  __syncthreads();

  // ---- F: state update with V', threshold test
  {
    uint32_t e = rtid;
#pragma unroll
    for (int i = 0; i < kHHDefer; ++i, e += kT) {
      dh.e[i] = kNoSlot;
      if (e < nE_hh) {
        const uint32_t slot = U.hh_slot[e];
        if (slot != kNoSlot16 && rmd) {
          dh.v[i] = Vs[gpos(slot, rc)]; dh.delta[i] = rdelta; dh.e[i] = e;
          dh.m[i] = U.sm[e]; dh.h[i] = U.sm[e + U.hh_ss]; dh.n[i] = U.sm[e + 2 * U.hh_ss];
        }
      }
    }
    for (; e < nE_hh; e += kT) {          // more instances than can be deferred: update in place
      const uint32_t slot = U.hh_slot[e];
      if (slot == kNoSlot16 || !rmd) continue;
      double m = U.sm[e], hh = U.sm[e + U.hh_ss], n = U.sm[e + 2 * U.hh_ss];
      hh_gates(Vs[gpos(slot, rc)], rdelta, m, hh, n);
      U.sm[e] = m; U.sm[e + U.hh_ss] = hh; U.sm[e + 2 * U.hh_ss] = n;
      U.gm[e] = m; U.gm[e + U.hh_ss] = hh; U.gm[e + 2 * U.hh_ss] = n;
    }
  }
  if (rmd) {
    double decay_u = M.syn_decay_u;
    if (kGen && rmd == 2u && M.syn_uniform) decay_u = exp(-rdelta / M.syn_tau_u);
  #pragma unroll 1
  for (uint32_t e = rtid; e < nE_syn; e += kT) {
      if (U.syn_slot[e] == kNoSlot16) continue;
      double decay = decay_u;
      if (!M.syn_uniform) decay = (!kGen || rmd == 1u) ? U.syn_decay()[e] : exp(-rdelta / U.syn_tau()[e]);
      U.sg[e] *= decay;
    }
  }
  if (tid < kG && md) {
    const double vd = Vs[gpos(U.det_slot[tid], tid)], vp = kGen ? cs.vprev[tid] : vprev;
    if ((uint32_t)tid < U.n_cell) {
      if (!isfinite(vd)) atomicOr(&M.counters[CNT_ERROR], 8ull);
      if (vp < M.theta && M.theta <= vd && cs.armed[tid]) {
        const double ts = (kGen ? cs.tcur[tid] : tstart) + (kGen ? cs.delta[tid] : dt) * (M.theta - vp) / (vd - vp);
        const unsigned long long pos = atomicAdd(&M.counters[CNT_SPIKES], 1ull);
        if ((int64_t)pos < M.spike_cap) { M.spike_cell[pos] = M.cell_orig[U.cell_base + tid]; M.spike_t[pos] = ts; }
        else atomicOr(&M.counters[CNT_ERROR], 1ull);
        cs.armed[tid] = 0;
      }
      if (vd < M.theta && !cs.armed[tid]) cs.armed[tid] = 1;
    }
    if (kGen) cs.tcur[tid] = cs.tnext[tid];
  }
}

// Work item -> group.  Items [0, n_hot) are the groups of this launch's hot list (an event falls into
// the coming grid step: their event-split steps take longer, so they go first); items n_hot + g are
// the groups in index order, minus the hot ones.  Returns n_groups past the end, -1 for "skip".
__device__ __forceinline__ int64_t map_item(const DevModel& M, const StepArgs& A, uint32_t n_hot, unsigned long long i) {
  if (i < n_hot) return (int64_t)M.ghot[(size_t)(A.launch_id % 3u) * (size_t)M.n_groups + i];
  const int64_t g = (int64_t)(i - n_hot);
  if (g >= M.n_groups) return M.n_groups;
  if (n_hot != 0 && M.ghotflag[(size_t)(A.launch_id & 1u) * (size_t)M.n_groups + g] == A.launch_id) return -1;
  return g;
}

// ------------------------------------------------------------------------------------------
// The cable step for cell groups.
// ------------------------------------------------------------------------------------------
// kLin: the conductance-linearised step (ARB_OPT_LINEARISED) is an instantiation of its own, so that its code costs the
// explicit step nothing (measured: 1.5 % when both live in one kernel).
template <bool kLin>
__global__ void __launch_bounds__(kGroupThreads, kGroupMinCtas) cable_group_kernel(DevModel M, StepArgs A) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ GroupDesc sD[2];            // this group's and the next group's descriptors
  __shared__ uint32_t flags[3];
  const GroupSmemPlan P = M.gplan;
  double* Ss = (double*)smem;            // state record; V first
  double* Vs = Ss;
  const double* Fs = (const double*)(smem + P.off_f);
  const double* Is = (const double*)(smem + P.off_i);
  const uint8_t* tail = smem + P.off_tail;
  uint8_t* cls = smem + P.off_class;
  double* buf = (double*)(smem + P.off_buf);
  const CellS cs = carve_cells(smem + P.off_cell, kG);
  uint64_t* mbar = (uint64_t*)(smem + P.off_mbar);
  const int tid = threadIdx.x;
  if (tid == 0) { mbar_init(mbar, 1); mbar_init(mbar + 1, 1); fence_mbar_init(); }
  __shared__ int64_t sG[2];
  __shared__ uint32_t sNHot;
  if (tid == 0) {
    // Groups are claimed dynamically (group-steps differ in length): item blockIdx.x first, further
    // items from this launch's work counter, which the previous launch has reset to gridDim.x; this
    // launch resets the other one and clears the hot list after the next
    const uint32_t n_hot = A.hot_valid ? (uint32_t)M.counters[CNT_HOT0 + A.launch_id % 3u] : 0u;
    sNHot = n_hot;
    if (blockIdx.x == 0) {
      M.counters[CNT_GROUP0 + (A.parity ^ 1)] = gridDim.x;
      M.counters[CNT_HOT0 + (A.launch_id + 2u) % 3u] = 0ull;
    }
    int64_t g0 = map_item(M, A, n_hot, blockIdx.x);
    while (g0 < 0) g0 = map_item(M, A, n_hot, atomicAdd(&M.counters[CNT_GROUP0 + A.parity], 1ull));
    sG[0] = g0;
  }
  __syncthreads();
  if (tid < 16 && sG[0] < M.n_groups) ((uint32_t*)&sD[0])[tid] = ((const uint32_t*)&M.groups[sG[0]])[tid];
  __syncthreads();
  unsigned n_sub = 0, n_del = 0;
  uint32_t it = 0, par2 = 0;
  bool ab_ready = false;                 // the coefficient buffers hold a, b (else f, 1/d of the last (sub-)step)
  int64_t cached_class = -1;
  HHDefer dh;
  clear(dh);
  double* dh_gm = nullptr;               // where the carried gate update of the previous group goes
  uint32_t dh_ss = 0;
  for (int64_t g = sG[0]; g < M.n_groups; g = sG[(++it) & 1u]) {
    const GroupDesc& D = sD[it & 1u];
    const GConstOff co = gconst_offsets(D.n_cv, D.n_hh_rows, D.n_syn_rows, D.n_cl_rows, M.syn_uniform != 0);
    const GStateOff so = gstate_offsets(D.n_cv, D.n_hh_rows, D.n_syn_rows);
    const uint32_t vbytes = 8u * gcv_elems(D.n_cv);
    // a further (sub-)step of the same residency: a, b back into the coefficient buffers (L2)
    auto reload_ab = [&]() {
      if (tid == 0) {
        const uint8_t* cb = M.fast + D.const_off;
        fence_proxy_async();
        mbar_expect_tx(mbar + 1, 2u * vbytes);
        bulk_g2s((void*)Fs, cb + co.a, vbytes, mbar + 1);
        bulk_g2s((void*)Is, cb + co.b, vbytes, mbar + 1);
      }
      mbar_wait(mbar + 1, par2);
      par2 ^= 1u;
    };
    if (tid == 0) {
      // state record, a, b and the const tail of the group -> shared memory (one barrier)
      const uint8_t* cb = M.fast + D.const_off;
      const uint32_t tbytes = co.total - co.hh_gna;
      fence_proxy_async();
      mbar_expect_tx(mbar, 8u * so.total + 2u * vbytes + tbytes);
      bulk_g2s(Ss, M.state + D.state_base, 8u * so.total, mbar);
      bulk_g2s((void*)Fs, cb + co.a, vbytes, mbar);           // a, b first: the two coefficient buffers hold
      bulk_g2s((void*)Is, cb + co.b, vbytes, mbar);           // them until the rhs is formed, then f, 1/d
      bulk_g2s((void*)tail, cb + co.hh_gna, tbytes, mbar);
      if (M.l2_prefetch) bulk_prefetch_l2(cb + co.f, co.a - co.f);          // f, 1/d of this group -> L2
    } else if (tid >= 32 && tid < 64) {     // warp 1 claims the next group and fetches its descriptor
      long long gn = 0;
      if (tid == 32) {
        do gn = map_item(M, A, sNHot, atomicAdd(&M.counters[CNT_GROUP0 + A.parity], 1ull)); while (gn < 0);
        sG[(it + 1) & 1u] = gn;
      }
      gn = __shfl_sync(kFull, gn, 0);
      if (tid < 48 && gn < M.n_groups) ((uint32_t*)&sD[(it + 1) & 1u])[tid - 32] = ((const uint32_t*)&M.groups[gn])[tid - 32];
    }
    if (D.class_off != cached_class) {   // tree structure differs from the previous group's
      const ClassRecord* R = (const ClassRecord*)(M.topo + D.class_off);
      const uint32_t n16 = R->bytes / 16;
      const uint4* src = (const uint4*)R;
      for (uint32_t i = tid; i < n16; i += kT) ((uint4*)cls)[i] = src[i];
      cached_class = D.class_off;
      __syncthreads();
    }
    ab_ready = true;                     // a, b are on their way into the coefficient buffers
    GView U;
    make_gview(U, M, D, Ss, tail, cls);
    // the previous group's last gate update: registers -> global m, h, n, while the copies are in flight
    run_deferred(dh, dh_gm, nullptr, dh_ss);
    dh_gm = U.gm; dh_ss = U.hh_ss;
    mbar_wait(mbar, it & 1u);
    if (tid < kG) {
      const unsigned long long pk = (unsigned long long)__double_as_longlong(U.srt[kRtDoubles * tid + 1]);
      cs.evcur[tid] = (uint32_t)pk; cs.evend[tid] = (uint32_t)(pk >> 32);
      cs.armed[tid] = U.srt[kRtDoubles * tid + 2] != 0.0 ? 1u : 0u;
    }
    __syncthreads();

    for (int64_t k = A.k_first; k < A.k_first + A.nk; ++k) {
      const double ta = (k == 0) ? A.t0 : __dadd_rn(A.t0, __dmul_rn((double)k, A.dt));
      const double tb = (k + 1 == A.nsteps) ? A.t_end : __dadd_rn(A.t0, __dmul_rn((double)(k + 1), A.dt));
      const bool nominal = (k + 1 < A.nsteps) || A.last_full;
      // fast check: no cell has an event before the end of this nominal step -> one nominal step of the
      // whole group, with the cells' runtime in registers (the common case; reading R9 otherwise)
      double vprev = 0.0;
      if (tid < 32) {
        bool fast = true;
        if (tid < kG) {
          fast = nominal && !(U.srt[kRtDoubles * tid] < tb);
          vprev = Vs[gpos(U.det_slot[tid], tid)];
        }
        const int all_fast = __all_sync(kFull, fast);
        if (tid == 0) flags[0] = (uint32_t)all_fast;
      }
      __syncthreads();
      if (flags[0]) {
        if ((uint32_t)tid < U.n_cell) ++n_sub;
        run_deferred(dh, U.sm, U.gm, U.hh_ss);
        if (!ab_ready) reload_ab();
        ab_ready = false;
        group_substep<false, kLin>(M, U, Vs, Fs, Is, buf, cs, A.dt, dh, vprev, ta, M.fast + D.const_off + co.f, vbytes, mbar + 1, par2);
        __syncthreads();                  // flags are rewritten by the next grid step
        continue;
      }
      __syncthreads();                    // everyone has read flags[0]
      if (tid < kG) cs.tcur[tid] = ta;
      for (;;) {
        // ---- A: deliver the events due now, choose each cell's (sub-)step (R9)
        if (tid < 32) {
          bool active = false, gen = false, split = false;
          if (tid < kG) {
            const double t = cs.tcur[tid];
            uint32_t md = 0;
            if (t < tb) {
              double tn = U.srt[kRtDoubles * tid];
              if (tn <= t) {
                uint32_t cur = cs.evcur[tid];
                const uint32_t end = cs.evend[tid];
                while (cur < end && M.ev_t[cur] <= t) { Ss[event_target(M, M.ev_gidx[cur], t, M.ev_w[cur]) - (uint32_t)D.state_base] += M.ev_w[cur]; ++cur; ++n_del; }
                tn = cur < end ? M.ev_t[cur] : CUDART_INF;
                cs.evcur[tid] = cur; U.srt[kRtDoubles * tid] = tn;
              }
              const double next = tn < tb ? tn : tb;
              const bool fast = nominal && t == ta && next == tb;
              cs.delta[tid] = fast ? A.dt : next - t;
              md = fast ? 1u : 2u;
              if (!fast && M.l2_prefetch) bulk_prefetch_l2(U.C(), 8u * gcv_elems(U.n_cv));   // C for the general rhs
              cs.tnext[tid] = next;
              cs.vprev[tid] = Vs[gpos(U.det_slot[tid], tid)];
              active = true;
              if ((uint32_t)tid < U.n_cell) ++n_sub;
            }
            cs.mode[tid] = md;
            gen = md != 1u; split = md == 2u;
          }
          const unsigned ba = __ballot_sync(kFull, active), bg = __ballot_sync(kFull, gen), bs = __ballot_sync(kFull, split);
          if (tid == 0) { flags[0] = ba; flags[1] = bg; flags[2] = bs; }
        }
        __syncthreads();                  // also orders the delivered g += w before phase B
        if (!flags[0]) break;
        // another (sub-)step follows: the gates of the previous one are needed now (working copy and global)
        run_deferred(dh, U.sm, U.gm, U.hh_ss);
        if (!ab_ready) reload_ab();
        ab_ready = false;
        {                                 // (all cells nominal only after events delivered exactly at the step start)
          group_substep<true, kLin>(M, U, Vs, Fs, Is, buf, cs, A.dt, dh, 0.0, 0.0, M.fast + D.const_off + co.f, vbytes, mbar + 1, par2);
        }
        __syncthreads();
      }
      __syncthreads();                    // flags are rewritten by the next grid step
    }

    // ---- V', g, per-cell runtime -> HBM (one bulk store); the gates follow from registers
    if (tid < kG) {
      const unsigned long long pk = ((unsigned long long)cs.evend[tid] << 32) | cs.evcur[tid];
      U.srt[kRtDoubles * tid + 1] = __longlong_as_double((long long)pk);
      U.srt[kRtDoubles * tid + 2] = cs.armed[tid] ? 1.0 : 0.0;
    }
    if (A.mark_hot && tid < 32) {         // does an event of this group fall into the next grid step?
      const double t_hot = A.t0 + (double)(A.k_first + A.nk + 1) * A.dt;
      const bool hot = (uint32_t)tid < U.n_cell && U.srt[kRtDoubles * (tid < kG ? tid : 0)] < t_hot;
      if (__any_sync(kFull, hot) && tid == 0) {
        const uint32_t nxt = A.launch_id + 1u;
        const unsigned long long pos = atomicAdd(&M.counters[CNT_HOT0 + nxt % 3u], 1ull);
        M.ghot[(size_t)(nxt % 3u) * (size_t)M.n_groups + pos] = (uint32_t)g;
        M.ghotflag[(size_t)(nxt & 1u) * (size_t)M.n_groups + g] = nxt;   // (this launch may still look at the other half)
      }
    }
    fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
      bulk_s2g(M.state + D.state_base, Ss, 8u * so.m);
      bulk_commit();
      if (M.l2_prefetch && sG[(it + 1) & 1u] < M.n_groups) {   // next group's records -> L2
        const GroupDesc& Dn = sD[(it + 1) & 1u];
        const GConstOff con = gconst_offsets(Dn.n_cv, Dn.n_hh_rows, Dn.n_syn_rows, Dn.n_cl_rows, M.syn_uniform != 0);
        bulk_prefetch_l2(M.fast + Dn.const_off + con.a, con.total - con.a);      // a, b and the tables
        bulk_prefetch_l2(M.state + Dn.state_base, 8u * gstate_offsets(Dn.n_cv, Dn.n_hh_rows, Dn.n_syn_rows).total);
      }
      bulk_wait_read0();
    }
    __syncthreads();                      // shared memory may be overwritten by the next group's copies
  }
  run_deferred(dh, dh_gm, nullptr, dh_ss);
  if (tid < 32) {
    for (int o = 16; o; o >>= 1) { n_sub += __shfl_xor_sync(kFull, n_sub, o); n_del += __shfl_xor_sync(kFull, n_del, o); }
    if (tid == 0) {
      if (n_sub) atomicAdd(&M.counters[CNT_SUBSTEPS], (unsigned long long)n_sub);
      if (n_del) atomicAdd(&M.counters[CNT_DELIVERED], (unsigned long long)n_del);
    }
  }
}

// ------------------------------------------------------------------------------------------
// Once per dt: f, 1/d, a, b (and per-synapse decay factors) of every group.  One CTA per group;
// dynamic shared memory: n_seg * kG doubles.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kGroupThreads) group_factor_kernel(DevModel M, double dt) {
  extern __shared__ __align__(128) uint8_t smem[];
  double* dcon = (double*)smem;
  const GroupDesc D = M.groups[blockIdx.x];
  const GConstOff co = gconst_offsets(D.n_cv, D.n_hh_rows, D.n_syn_rows, D.n_cl_rows, M.syn_uniform != 0);
  uint8_t* cb = M.fast + D.const_off;
  GView U;
  make_gview(U, M, D, M.state + D.state_base, cb + co.hh_gna, M.topo + D.class_off);
  const int tid = threadIdx.x, c = tid % kG, h = tid / kG;
  double* f = (double*)(cb + co.f);
  double* invd = (double*)(cb + co.invd);
  double* a = (double*)(cb + co.a);
  double* b = (double*)(cb + co.b);
  const double *C = U.C(), *G = U.G(), *bg = U.bg();
  if (!M.linearised) {
    for (uint32_t st = 0; st < U.n_stage; ++st) {
      const uint32_t beg = U.sched[st * kGroupSlots + h], end = U.sched[st * kGroupSlots + h + 1];
      for (uint32_t q = beg; q < end; ++q) {
        const uint32_t si = q;
        eliminate_seg(U, load_seg(U.segs + si), si, c, dt, f, invd, dcon);
      }
      __syncthreads();
    }
    for (uint32_t e = tid; e < gcv_elems(U.n_cv); e += kT) {
      a[e] = C[e] / dt - G[e];
      b[e] = bg[e];
    }
  } else {
    // conductance-linearised step: rhs = (C/dt) V + G e + ..., diagonal C/dt + sum(sigma) + G + ..., sigma
    const double *S = U.S(), *sig = U.sig();
    for (uint32_t e = tid; e < gcv_elems(U.n_cv); e += kT) {
      const double cdt = C[e] / dt;
      a[e] = cdt;
      b[e] = bg[e];
      f[e] = (cdt + S[e]) + G[e];
      invd[e] = sig[e];
    }
  }
  if (!M.syn_uniform) {
    double* decay = (double*)(cb + co.syn_decay);
    const double* tau = U.syn_tau();
    for (uint32_t e = tid; e < U.n_syn * kG; e += kT) decay[e] = exp(-dt / tau[e]);
  }
}

// R4: gates start at their steady state for the initial voltage.
__global__ void __launch_bounds__(kGroupThreads) group_init_kernel(DevModel M) {
  const GroupDesc D = M.groups[blockIdx.x];
  const GConstOff co = gconst_offsets(D.n_cv, D.n_hh_rows, D.n_syn_rows, D.n_cl_rows, M.syn_uniform != 0);
  double* st = M.state + D.state_base;
  GView U;
  make_gview(U, M, D, st, M.fast + D.const_off + co.hh_gna, M.topo + D.class_off);
  const int c = threadIdx.x % kG;
  for (uint32_t e = threadIdx.x; e < U.n_hh * kG; e += kT) {
    const uint32_t slot = U.hh_slot[e];
    if (slot == kNoSlot16) continue;
    const Rates r = hh_rates(st[gpos(slot, c)]);
    U.gm[e] = r.am / (r.am + r.bm);
    U.gm[e + U.hh_ss] = r.ah / (r.ah + r.bh);
    U.gm[e + 2 * U.hh_ss] = r.an / (r.an + r.bn);
  }
}

}  // namespace

// Resident CTAs of the group kernel per SM for `smem_bytes` of dynamic shared memory (asks the
// runtime; configure_kernels() has opted the kernel in).  0: does not fit / no device.
cudaError_t configure_group_kernel(int max_optin_bytes) {
  for (const void* k : {(const void*)cable_group_kernel<false>, (const void*)cable_group_kernel<true>}) {
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, k);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, max_optin_bytes - (int)fa.sharedSizeBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

int group_ctas_per_sm(uint32_t smem_bytes) {
  if (smem_bytes + 1024u > (uint32_t)cable_smem_limit()) return 0;
  int n = 0;
  int nl = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, cable_group_kernel<false>, kGroupThreads, smem_bytes) != cudaSuccess) return 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nl, cable_group_kernel<true>, kGroupThreads, smem_bytes) != cudaSuccess) return 0;
  return n < nl ? n : nl;
}

cudaError_t launch_group_factor(const DevModel& M, double dt, uint32_t seg_cap, cudaStream_t s) {
  if (M.n_groups == 0) return cudaSuccess;
  group_factor_kernel<<<(unsigned)M.n_groups, kGroupThreads, seg_cap * kG * 8, s>>>(M, dt);
  return cudaGetLastError();
}

cudaError_t launch_group_init(const DevModel& M, cudaStream_t s) {
  if (M.n_groups == 0) return cudaSuccess;
  group_init_kernel<<<(unsigned)M.n_groups, kGroupThreads, 0, s>>>(M);
  return cudaGetLastError();
}

cudaError_t launch_group_cable(const DevModel& M, const StepArgs& A, int grid, cudaStream_t s, int* launches) {
  if (M.n_groups == 0) return cudaSuccess;
  const int smem = (int)M.gplan.bytes;          // group_ctas_per_sm() has opted the kernel in
  if (!M.linearised) cable_group_kernel<false><<<(unsigned)grid, kGroupThreads, smem, s>>>(M, A);
  else cable_group_kernel<true><<<(unsigned)grid, kGroupThreads, smem, s>>>(M, A);
  if (launches) ++*launches;
  return cudaGetLastError();
}

}  // namespace arbb
