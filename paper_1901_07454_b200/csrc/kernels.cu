// kernels.cu - hand-written fp64 CUDA kernels for sm_100a: the whole hot path of arbb200.
//
//   cable_block_kernel  the cable step for block units (unit_layout.h): cells too large for a CTA's shared
//                       memory, or with thousands of synapses.  One CTA per unit, working straight out of
//                       global memory (L1/L2), lane = branch, __syncthreads between tree levels.  Per grid
//                       step (or fused run of steps): event delivery -> mechanism currents
//                       (eq 2a; synapse currents summed by a warp-level key reduction,
//                       PAPER.md:218) -> rhs of the implicit Euler system -> branched Thomas /
//                       Hines sweeps over tasks of interleaved branches -> V <- V' -> gate /
//                       synapse state update with V' -> threshold test.
//                       (Cells that share a tree run in group_kernel.cu, all other cells in forest_kernel.cu.)
//   factor_kernel       once per dt: eliminates the (constant, reading R1) matrix of every block unit
//   ev_* / spikes_to_events   once per min-delay epoch
//
// No tensor cores: nothing here is a dense contraction.
#include "kernels.cuh"
#include "device_common.cuh"

namespace arbb {

namespace {

constexpr int kPcRecord = 8;         // doubles of a point cell's record (layout.hpp: kPcDoubles)
constexpr int kBlockThreads = 128;              // cable_block_kernel, factor_kernel, init_kernel
constexpr int kBlockWarps = kBlockThreads / 32;
constexpr uint32_t kSynKeyReduceMin = 1024;     // block units with at least this many synapses reduce currents by key

// a block unit is integrated by one CTA
struct S {
  static constexpr int size = kBlockThreads, warps = kBlockWarps;
  static __device__ __forceinline__ int tid() { return threadIdx.x; }
  static __device__ __forceinline__ int warp() { return threadIdx.x >> 5; }
  static __device__ __forceinline__ void sync() { __syncthreads(); }
  static __device__ __forceinline__ bool any(bool p) { return __syncthreads_or(p) != 0; }
};

// Pointers of one unit; everything addresses global memory.
struct UnitView {
  uint32_t n_slot, n_lane, n_task, n_level, n_cell, n_hh, n_syn, n_clamp;
  const double *f, *invd, *a, *b, *hh_gna, *hh_gk, *hh_gl, *syn_e, *syn_decay, *cl_t0, *cl_t1, *cl_amp;
  const uint32_t *hh_slot, *syn_slot, *cl_slot;
  const uint16_t *hh_cell, *syn_cell, *cl_cell;
  double *V, *m, *h, *n, *g, *rt;
  uint32_t g_gidx0;                 // state-pool index of g[0]
  const Task* tasks; const LaneRec* lanes; const uint32_t *level_begin, *child, *cell_det;
  const double *C, *S, *sig, *G, *bg, *syn_tau;
  double *contrib, *dcontrib, *xI, *fgen, *invdgen;
  uint32_t* heads;              // block units: heads[0] = runs in the synapse list, heads[1..] = their first synapse
  int64_t cell_base;
};

__device__ __forceinline__ void make_view(UnitView& U, const DevModel& M, const UnitHeader& H, uint8_t* fastw, double* statew,
                                          const uint8_t* topow) {
  U.n_slot = H.n_slot; U.n_lane = H.n_lane; U.n_task = H.n_task; U.n_level = H.n_level;
  U.n_cell = H.n_cell; U.n_hh = H.n_hh; U.n_syn = H.n_syn; U.n_clamp = H.n_clamp;
  const FastOff fo = fast_offsets(H.n_slot, H.n_hh, H.n_syn, H.n_clamp, H.n_cell, M.syn_uniform != 0);
  U.f = (const double*)(fastw + fo.f); U.invd = (const double*)(fastw + fo.invd);
  U.a = (const double*)(fastw + fo.a); U.b = (const double*)(fastw + fo.b);
  U.hh_gna = (const double*)(fastw + fo.hh_gna); U.hh_gk = (const double*)(fastw + fo.hh_gk); U.hh_gl = (const double*)(fastw + fo.hh_gl);
  U.syn_e = (const double*)(fastw + fo.syn_e); U.syn_decay = (const double*)(fastw + fo.syn_decay);
  U.cl_t0 = (const double*)(fastw + fo.cl_t0); U.cl_t1 = (const double*)(fastw + fo.cl_t1); U.cl_amp = (const double*)(fastw + fo.cl_amp);
  U.hh_slot = (const uint32_t*)(fastw + fo.hh_slot); U.syn_slot = (const uint32_t*)(fastw + fo.syn_slot); U.cl_slot = (const uint32_t*)(fastw + fo.cl_slot);
  U.hh_cell = (const uint16_t*)(fastw + fo.hh_cell); U.syn_cell = (const uint16_t*)(fastw + fo.syn_cell); U.cl_cell = (const uint16_t*)(fastw + fo.cl_cell);
  const StateOff so = state_offsets(H.n_slot, H.n_hh, H.n_syn, H.n_cell);
  U.V = statew + so.v; U.m = statew + so.m; U.h = statew + so.h; U.n = statew + so.n; U.g = statew + so.g; U.rt = statew + so.rt;
  U.g_gidx0 = (uint32_t)(H.state_base + so.g);
  const TopoOff to = topo_offsets(H.n_task, H.n_level, H.n_lane, H.n_child, H.n_cell);
  U.tasks = (const Task*)(topow + to.tasks); U.lanes = (const LaneRec*)(topow + to.lanes);
  U.level_begin = (const uint32_t*)(topow + to.level_begin); U.child = (const uint32_t*)(topow + to.child);
  U.cell_det = (const uint32_t*)(topow + to.cell_det);
  const GenOff go = gen_offsets(H.n_slot, H.n_syn);
  const double* gen = M.gen + H.gen_base;
  U.C = gen + go.C; U.S = gen + go.S; U.sig = gen + go.sig; U.G = gen + go.G; U.bg = gen + go.b; U.syn_tau = gen + go.syn_tau;
  U.cell_base = H.cell_base;
}

struct TaskCtx { Task T; LaneRec R; };
__device__ __forceinline__ TaskCtx load_ctx(const UnitView& U, uint32_t ti, int lane) {
  TaskCtx c;
  c.T = U.tasks[ti];
  c.R = U.lanes[c.T.lane_off + ((uint32_t)lane < c.T.nlanes ? lane : 0)];
  return c;
}

// ------------------------------------------------------------------------------------------
// Elimination of the diagonal for one step length (factorisation, and event-split sub-steps).
// For a branch (lane) with CVs k = 0..len-1:
//   d_k = C_k/delta + S_k - sum_children sigma_c^2 / d_c ;  f_k = -sigma_k / d_k = u_k / d_k
// fout/invdout receive f and 1/d; dcontrib[branch] = f_0 * u_0 is what the parent's last CV loses.
// Every lane of the warp must call it (ragged rows are counted with ballots); `on` selects the
// lanes that take part.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void eliminate_task(const UnitView& U, const TaskCtx& X, int lane, bool on, double delta,
                                               double* fout, double* invdout, double* dcontrib) {
  const Task& T = X.T;
  const bool in = (uint32_t)lane < T.nlanes;
  const uint32_t len = in ? X.R.len : 0u;
  const uint32_t maxlen = T.maxlen_full & 0x7FFFu;
  const bool full = (T.maxlen_full & kTaskFull) != 0;
  const uint32_t tl = T.lane_off + lane;
  uint32_t row = T.slot_off + T.nslots;
  double fp = 0.0, sgp = 0.0;
  for (int k = (int)maxlen - 1; k >= 0; --k) {
    const bool act = (uint32_t)k < len;
    const uint32_t cnt = full ? T.nlanes : (uint32_t)__popc(__ballot_sync(kFull, act));
    row -= cnt;
    if (act && on) {
      const uint32_t s = row + lane;
      double d = U.C[s] / delta + U.S[s];
      if ((uint32_t)k == len - 1) {
        for (uint32_t j = 0; j < X.R.ccnt; ++j) d -= dcontrib[U.child[X.R.cbeg + j]];
      } else {
        d = fma(fp, sgp, d);                 // d_p -= f*u with u = -sigma
      }
      const double invd = 1.0 / d;
      const double sg = U.sig[s];
      const double fk = -sg * invd;
      fout[s] = fk;
      invdout[s] = invd;
      fp = fk; sgp = sg;
      if (k == 0) dcontrib[tl] = -fk * sg;   // f*u
    }
  }
}

// ------------------------------------------------------------------------------------------
// Backward (leaves -> root) sweep of one task on the rhs held in U.V:
//   rhs_{k-1} -= f_k rhs_k along the branch, the parent's last CV loses contrib[child] = f_0 rhs_0;
// every CV is left holding rhs_k / d_k, which is what the forward sweep needs.
// kGen: cells of the unit may be inactive (mode 0) or on an event-split sub-step (mode 2).
// ------------------------------------------------------------------------------------------
template <bool kGen>
__device__ __forceinline__ void backward_task(const UnitView& U, const CellS& cs, const TaskCtx& X, int lane) {
  const Task& T = X.T;
  const bool in = (uint32_t)lane < T.nlanes;
  const uint32_t len = in ? X.R.len : 0u;
  const uint32_t maxlen = T.maxlen_full & 0x7FFFu;
  const bool full = (T.maxlen_full & kTaskFull) != 0;
  const uint32_t tl = T.lane_off + lane;
  uint32_t md = in ? 1u : 0u;
  if (kGen) {
    double delta = 0.0;
    if (in) { md = cs.mode[X.R.cell]; delta = cs.delta[X.R.cell]; }
    if (__any_sync(kFull, md == 2u)) eliminate_task(U, X, lane, md == 2u, delta, U.fgen, U.invdgen, U.dcontrib);
  }
  if (!kGen && full) {
    // every row is full and every lane takes a nominal step: rows are prefetched four at a time so
    // that only the dependent fma chain is exposed
    if (!in) return;
    const uint32_t w = T.nlanes;
    uint32_t s = T.slot_off + T.nslots - w + lane;
    double r = U.V[s];
    for (uint32_t j = 0; j < X.R.ccnt; ++j) r -= U.contrib[U.child[X.R.cbeg + j]];
    double fc = U.f[s], ic = U.invd[s];
    uint32_t k = maxlen - 1;
    while (k >= 4) {
      const uint32_t s1 = s - w, s2 = s1 - w, s3 = s2 - w, s4 = s3 - w;
      const double r1 = U.V[s1], r2 = U.V[s2], r3 = U.V[s3], r4 = U.V[s4];
      const double f1 = U.f[s1], f2 = U.f[s2], f3 = U.f[s3], f4 = U.f[s4];
      const double i1 = U.invd[s1], i2 = U.invd[s2], i3 = U.invd[s3], i4 = U.invd[s4];
      U.V[s] = r * ic;   r = fma(-fc, r, r1);
      U.V[s1] = r * i1;  r = fma(-f1, r, r2);
      U.V[s2] = r * i2;  r = fma(-f2, r, r3);
      U.V[s3] = r * i3;  r = fma(-f3, r, r4);
      fc = f4; ic = i4; s = s4; k -= 4;
    }
    while (k >= 1) {
      const uint32_t s1 = s - w;
      const double r1 = U.V[s1], f1 = U.f[s1], i1 = U.invd[s1];
      U.V[s] = r * ic;   r = fma(-fc, r, r1);
      fc = f1; ic = i1; s = s1; --k;
    }
    U.V[s] = r * ic;
    U.contrib[tl] = fc * r;
    return;
  }
  uint32_t row = T.slot_off + T.nslots;
  double r = 0.0, fp = 0.0;
  for (int k = (int)maxlen - 1; k >= 0; --k) {
    const bool act = (uint32_t)k < len;
    const uint32_t cnt = full ? T.nlanes : (uint32_t)__popc(__ballot_sync(kFull, act));
    row -= cnt;
    if (act && md) {
      const uint32_t s = row + lane;
      double rk = U.V[s];
      if ((uint32_t)k == len - 1) {
        for (uint32_t j = 0; j < X.R.ccnt; ++j) rk -= U.contrib[U.child[X.R.cbeg + j]];
      } else {
        rk = fma(-fp, r, rk);
      }
      double fk, ik;
      if (kGen && md == 2u) { fk = U.fgen[s]; ik = U.invdgen[s]; }
      else { fk = U.f[s]; ik = U.invd[s]; }
      U.V[s] = rk * ik;
      r = rk; fp = fk;
      if (k == 0) U.contrib[tl] = fk * rk;
    }
  }
}

// Forward (root -> leaves) substitution of one task: V'_k = rhs_k/d_k - f_k V'_{k-1}; V <- V'.
template <bool kGen>
__device__ __forceinline__ void forward_task(const UnitView& U, const CellS& cs, const TaskCtx& X, int lane) {
  const Task& T = X.T;
  const bool in = (uint32_t)lane < T.nlanes;
  const uint32_t len = in ? X.R.len : 0u;
  const uint32_t maxlen = T.maxlen_full & 0x7FFFu;
  const bool full = (T.maxlen_full & kTaskFull) != 0;
  uint32_t md = in ? 1u : 0u;
  if (kGen && in) md = cs.mode[X.R.cell];
  double vp = 0.0;
  if (in && md && X.R.pslot != kNoSlot) vp = U.V[X.R.pslot];
  if (!kGen && full) {
    if (!in) return;
    const uint32_t w = T.nlanes;
    uint32_t s = T.slot_off + lane;
    uint32_t k = maxlen;
    while (k >= 4) {
      const uint32_t s1 = s + w, s2 = s1 + w, s3 = s2 + w;
      const double f0 = U.f[s], f1 = U.f[s1], f2 = U.f[s2], f3 = U.f[s3];
      const double q0 = U.V[s], q1 = U.V[s1], q2 = U.V[s2], q3 = U.V[s3];
      const double v0 = fma(-f0, vp, q0), v1 = fma(-f1, v0, q1), v2 = fma(-f2, v1, q2), v3 = fma(-f3, v2, q3);
      U.V[s] = v0; U.V[s1] = v1; U.V[s2] = v2; U.V[s3] = v3;
      vp = v3; s = s3 + w; k -= 4;
    }
    while (k >= 1) {
      vp = fma(-U.f[s], vp, U.V[s]);
      U.V[s] = vp;
      s += w; --k;
    }
    return;
  }
  uint32_t row = T.slot_off;
  for (uint32_t k = 0; k < maxlen; ++k) {
    const bool act = k < len;
    const uint32_t cnt = full ? T.nlanes : (uint32_t)__popc(__ballot_sync(kFull, act));
    if (act && md) {
      const uint32_t s = row + lane;
      const double fk = (kGen && md == 2u) ? U.fgen[s] : U.f[s];
      vp = fma(-fk, vp, U.V[s]);
      U.V[s] = vp;
    }
    row += cnt;
  }
}

// rhs_i = (C_i/delta - G_i) V_i + G_i e_i in place of V, one task (general path only)
__device__ __forceinline__ void rhs_task(const UnitView& U, const CellS& cs, const TaskCtx& X, int lane) {
  const Task& T = X.T;
  const bool in = (uint32_t)lane < T.nlanes;
  const uint32_t len = in ? X.R.len : 0u;
  const uint32_t maxlen = T.maxlen_full & 0x7FFFu;
  const bool full = (T.maxlen_full & kTaskFull) != 0;
  uint32_t md = 0;
  double delta = 0.0;
  if (in) { md = cs.mode[X.R.cell]; delta = cs.delta[X.R.cell]; }
  uint32_t row = T.slot_off;
  for (uint32_t k = 0; k < maxlen; ++k) {
    const bool act = k < len;
    const uint32_t cnt = full ? T.nlanes : (uint32_t)__popc(__ballot_sync(kFull, act));
    if (act && md) {
      const uint32_t s = row + lane;
      if (md == 1u) U.V[s] = fma(U.a[s], U.V[s], U.b[s]);
      else U.V[s] = fma(U.C[s] / delta - U.G[s], U.V[s], U.bg[s]);
    }
    row += cnt;
  }
}

// ------------------------------------------------------------------------------------------
// One (sub-)step of every active cell of a unit, phases B..F of the step (phase A, event delivery
// and the choice of the sub-step, is in run_unit).
// ------------------------------------------------------------------------------------------
template <bool kGen>
__device__ __forceinline__ void substep(const DevModel& M, const UnitView& U, const CellS& cs, double dt) {
  const int tid = S::tid(), lane = threadIdx.x & 31;
  const bool multi = U.n_cell > 1;
  const uint32_t n_hh = U.n_hh, n_syn = U.n_syn, n_cl = U.n_clamp;

  // ---- B: currents of HH, synapses and clamps from V(t); the passive current is
  // folded into a, b.  Items on one CV form a run; the first lane of a run sums it in index order.
  for (uint32_t i = tid; i < n_hh; i += S::size) {
    if (kGen && !cs.mode[multi ? U.hh_cell[i] : 0]) continue;
    const double v = U.V[U.hh_slot[i]];
    const double m = U.m[i], h = U.h[i], n = U.n[i];
    U.xI[i] = U.hh_gna[i] * m * m * m * h * (v - M.ena) + U.hh_gk[i] * n * n * n * n * (v - M.ek) + U.hh_gl[i] * (v - M.el);
  }
  if (n_syn >= kSynKeyReduceMin) {
    // Many synapses per control volume (the paper's ring cell): a run head summing its
    // run alone would leave the other lanes idle.  Each warp takes 32 consecutive synapses (coalesced),
    // reduces them by key = control volume with shuffles (the "key reduction" of PAPER.md:218; runs are
    // contiguous), and the first lane of every key inside the chunk stores a partial sum; in phase C the run
    // heads add the partials of the chunks their run extends into, in index order (no atomics).
    constexpr int kCh = 2;               // chunks per warp and trip: independent loads in flight
    for (uint32_t base = (uint32_t)S::warp() * 32u * kCh; base < n_syn; base += (uint32_t)S::warps * 32u * kCh) {
      uint32_t slot[kCh];
      double term[kCh];
#pragma unroll
      for (int q = 0; q < kCh; ++q) {
        const uint32_t i = base + q * 32u + lane;
        slot[q] = i < n_syn ? U.syn_slot[i] : 0xFFFFFFFFu;
      }
#pragma unroll
      for (int q = 0; q < kCh; ++q) {
        const uint32_t i = base + q * 32u + lane;
        term[q] = 0.0;
        if (i < n_syn && !(kGen && !cs.mode[multi ? U.syn_cell[i] : 0])) {
          const double gi = U.g[i];
          term[q] = gi * (U.V[slot[q]] - (M.syn_uniform ? M.syn_e_u : U.syn_e[i]));
          // nominal step: the decay over dt does not depend on V', so g is updated while it is here
          if (!kGen) U.g[i] = gi * (M.syn_uniform ? M.syn_decay_u : U.syn_decay[i]);
        }
      }
#pragma unroll
      for (int q = 0; q < kCh; ++q) {
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const double t = __shfl_down_sync(kFull, term[q], o);
          const uint32_t k = __shfl_down_sync(kFull, slot[q], o);
          if (lane + o < 32 && k == slot[q]) term[q] += t;
        }
        const uint32_t prev = __shfl_up_sync(kFull, slot[q], 1);
        const uint32_t i = base + q * 32u + lane;
        if (i < n_syn && (lane == 0 || prev != slot[q])) U.xI[n_hh + i] = term[q];
      }
    }
  } else
  for (uint32_t i = tid; i < n_syn; i += S::size) {
    const uint32_t slot = U.syn_slot[i];
    if (i > 0 && U.syn_slot[i - 1] == slot) continue;
    if (kGen && !cs.mode[multi ? U.syn_cell[i] : 0]) continue;
    const double v = U.V[slot];
    double I = 0.0;
    uint32_t j = i;
    do {
      I += U.g[j] * (v - (M.syn_uniform ? M.syn_e_u : U.syn_e[j]));
      ++j;
    } while (j < n_syn && U.syn_slot[j] == slot);
    U.xI[n_hh + i] = I;
  }
  for (uint32_t i = tid; i < n_cl; i += S::size) {
    const uint32_t slot = U.cl_slot[i];
    if (i > 0 && U.cl_slot[i - 1] == slot) continue;
    const uint32_t c = multi ? U.cl_cell[i] : 0;
    if (kGen && !cs.mode[c]) continue;
    const double t = cs.tcur[c];
    double I = 0.0;
    uint32_t j = i;
    do {
      if (U.cl_t0[j] <= t && t < U.cl_t1[j]) I -= U.cl_amp[j];
      ++j;
    } while (j < n_cl && U.cl_slot[j] == slot);
    U.xI[n_hh + n_syn + i] = I;
  }
  S::sync();

  // ---- C: rhs_i = (C_i/delta - G_i) V_i + G_i e_i - I_i, in place of V
  if (!kGen) {
    const uint32_t n = U.n_slot;
#pragma unroll 4
    for (uint32_t s = tid; s < n; s += S::size) U.V[s] = fma(U.a[s], U.V[s], U.b[s]);
  } else {
    for (uint32_t ti = S::warp(); ti < U.n_task; ti += S::warps) rhs_task(U, cs, load_ctx(U, ti, lane), lane);
  }
  S::sync();
  if (n_hh) {
    for (uint32_t i = tid; i < n_hh; i += S::size) {
      if (kGen && !cs.mode[multi ? U.hh_cell[i] : 0]) continue;
      U.V[U.hh_slot[i]] -= U.xI[i];
    }
    S::sync();
  }
  if (n_syn >= kSynKeyReduceMin) {
    // run heads (listed once per dt by factor_kernel) add the partial sums of the chunks their run
    // extends into, in index order
    const uint32_t nh = U.heads[0];
    for (uint32_t h = tid; h < nh; h += S::size) {
      const uint32_t i = U.heads[1 + h];
      const uint32_t slot = U.syn_slot[i];
      if (kGen && !cs.mode[multi ? U.syn_cell[i] : 0]) continue;
      double I = U.xI[n_hh + i];
      for (uint32_t j = (i & ~31u) + 32u; j < n_syn && U.syn_slot[j] == slot; j += 32u) I += U.xI[n_hh + j];
      U.V[slot] -= I;
    }
    S::sync();
  } else if (n_syn) {
    for (uint32_t i = tid; i < n_syn; i += S::size) {
      const uint32_t slot = U.syn_slot[i];
      if (i > 0 && U.syn_slot[i - 1] == slot) continue;
      if (kGen && !cs.mode[multi ? U.syn_cell[i] : 0]) continue;
      U.V[slot] -= U.xI[n_hh + i];
    }
    S::sync();
  }
  if (n_cl) {
    for (uint32_t i = tid; i < n_cl; i += S::size) {
      const uint32_t slot = U.cl_slot[i];
      if (i > 0 && U.cl_slot[i - 1] == slot) continue;
      if (kGen && !cs.mode[multi ? U.cl_cell[i] : 0]) continue;
      U.V[slot] -= U.xI[n_hh + n_syn + i];
    }
    S::sync();
  }

  // ---- D: backward sweep, deepest level first; E: forward substitution, root first; V <- V'
  {
    const int warp = S::warp();
    for (int lvl = (int)U.n_level - 1; lvl >= 0; --lvl) {
      for (uint32_t ti = U.level_begin[lvl] + warp; ti < U.level_begin[lvl + 1]; ti += S::warps)
        backward_task<kGen>(U, cs, load_ctx(U, ti, lane), lane);
      __syncthreads();
    }
    for (uint32_t lvl = 0; lvl < U.n_level; ++lvl) {
      for (uint32_t ti = U.level_begin[lvl] + warp; ti < U.level_begin[lvl + 1]; ti += S::warps)
        forward_task<kGen>(U, cs, load_ctx(U, ti, lane), lane);
      __syncthreads();
    }
  }

  // ---- F: state update with V', threshold test
  for (uint32_t i = tid; i < n_hh; i += S::size) {
    const uint32_t c = (kGen && multi) ? U.hh_cell[i] : 0;
    if (kGen && !cs.mode[c]) continue;
    const double delta = kGen ? cs.delta[c] : dt;
    const Rates r = hh_rates(U.V[U.hh_slot[i]]);
    double inf = r.am / (r.am + r.bm);
    const double m = inf + (U.m[i] - inf) * exp(-delta * (r.am + r.bm));
    inf = r.ah / (r.ah + r.bh);
    const double h = inf + (U.h[i] - inf) * exp(-delta * (r.ah + r.bh));
    inf = r.an / (r.an + r.bn);
    const double n = inf + (U.n[i] - inf) * exp(-delta * (r.an + r.bn));
    U.m[i] = m; U.h[i] = h; U.n[i] = n;
  }
  if (!kGen && n_syn >= kSynKeyReduceMin) {
    // done in phase B
  } else
  for (uint32_t i = tid; i < n_syn; i += S::size) {
    const uint32_t c = (kGen && multi) ? U.syn_cell[i] : 0;
    const uint32_t md = kGen ? cs.mode[c] : 1u;
    if (!md) continue;
    double decay;
    if (md == 1u) decay = M.syn_uniform ? M.syn_decay_u : U.syn_decay[i];
    else decay = exp(-cs.delta[c] / (M.syn_uniform ? M.syn_tau_u : U.syn_tau[i]));
    U.g[i] *= decay;
  }
  if ((uint32_t)tid < U.n_cell && (!kGen || cs.mode[tid])) {
    const double vd = U.V[U.cell_det[tid]], vp = cs.vprev[tid];
    if (!isfinite(vd)) atomicOr(&M.counters[CNT_ERROR], 8ull);
    if (cs.armed[tid] && vp < M.theta && M.theta <= vd) {
      const double ts = cs.tcur[tid] + cs.delta[tid] * (M.theta - vp) / (vd - vp);
      const unsigned long long pos = atomicAdd(&M.counters[CNT_SPIKES], 1ull);
      if ((int64_t)pos < M.spike_cap) { M.spike_cell[pos] = M.cell_orig[U.cell_base + tid]; M.spike_t[pos] = ts; }
      else atomicOr(&M.counters[CNT_ERROR], 1ull);
      cs.armed[tid] = 0; cs.dirty[tid] = 1;
    }
    if (vd < M.theta && !cs.armed[tid]) { cs.armed[tid] = 1; cs.dirty[tid] = 1; }
    cs.tcur[tid] = cs.tnext[tid];
  }
  S::sync();
}

// ------------------------------------------------------------------------------------------
// A.nk grid steps of one unit.  Phase A: deliver the events due now and choose each cell's
// sub-step (reading R9), then the step itself.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void run_unit(const DevModel& M, const StepArgs& A, const UnitView& U, const CellS& cs,
                                         unsigned& n_sub, unsigned& n_del) {
  const int tid = S::tid();
  const uint32_t n_cell = U.n_cell;
  if ((uint32_t)tid < n_cell) {
    const unsigned long long pk = (unsigned long long)__double_as_longlong(U.rt[kRtDoubles * tid + 1]);
    cs.evcur[tid] = (uint32_t)pk; cs.evend[tid] = (uint32_t)(pk >> 32);
    cs.armed[tid] = U.rt[kRtDoubles * tid + 2] != 0.0 ? 1u : 0u;
    cs.dirty[tid] = 0;
  }
  for (int64_t k = A.k_first; k < A.k_first + A.nk; ++k) {
    const double ta = (k == 0) ? A.t0 : __dadd_rn(A.t0, __dmul_rn((double)k, A.dt));
    const double tb = (k + 1 == A.nsteps) ? A.t_end : __dadd_rn(A.t0, __dmul_rn((double)(k + 1), A.dt));
    const bool nominal = (k + 1 < A.nsteps) || A.last_full;
    if ((uint32_t)tid < n_cell) cs.tcur[tid] = ta;
    S::sync();
    for (;;) {
      bool active = false, plain = true;
      if ((uint32_t)tid < n_cell) {
        const double t = cs.tcur[tid];
        uint32_t md = 0;
        if (t < tb) {
          double tn = U.rt[kRtDoubles * tid];
          if (tn <= t) {
            uint32_t cur = cs.evcur[tid];
            const uint32_t end = cs.evend[tid];
            while (cur < end && M.ev_t[cur] <= t) { U.g[event_target(M, M.ev_gidx[cur], t, M.ev_w[cur]) - U.g_gidx0] += M.ev_w[cur]; ++cur; ++n_del; }
            tn = cur < end ? M.ev_t[cur] : CUDART_INF;
            cs.evcur[tid] = cur; U.rt[kRtDoubles * tid] = tn; cs.dirty[tid] = 1;
          }
          const double next = tn < tb ? tn : tb;
          const bool fast = nominal && t == ta && next == tb;
          cs.delta[tid] = fast ? A.dt : next - t;
          md = fast ? 1u : 2u;
          cs.tnext[tid] = next;
          cs.vprev[tid] = U.V[U.cell_det[tid]];
          active = true;
          ++n_sub;
        }
        cs.mode[tid] = md;
        plain = md == 1u;
      }
      if (!S::any(active)) break;
      const bool general = S::any(!plain);
      S::sync();
      if (general) substep<true>(M, U, cs, A.dt);
      else substep<false>(M, U, cs, A.dt);
    }
  }
  if ((uint32_t)tid < n_cell && cs.dirty[tid]) {
    double* rt = U.rt + kRtDoubles * tid;
    const unsigned long long pk = ((unsigned long long)cs.evend[tid] << 32) | cs.evcur[tid];
    rt[1] = __longlong_as_double((long long)pk);
    rt[2] = cs.armed[tid] ? 1.0 : 0.0;
  }
}

__device__ __forceinline__ void flush_stats(const DevModel& M, unsigned n_sub, unsigned n_del) {
  for (int o = 16; o; o >>= 1) { n_sub += __shfl_xor_sync(kFull, n_sub, o); n_del += __shfl_xor_sync(kFull, n_del, o); }
  if ((threadIdx.x & 31) == 0) {
    if (n_sub) atomicAdd(&M.counters[CNT_SUBSTEPS], (unsigned long long)n_sub);
    if (n_del) atomicAdd(&M.counters[CNT_DELIVERED], (unsigned long long)n_del);
  }
}

// ------------------------------------------------------------------------------------------
// The cable step for block units: one CTA per unit, working copy = the records in global memory.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void block_view(UnitView& U, const DevModel& M, const UnitHeader& H, const UnitDesc& d) {
  make_view(U, M, H, M.fast + d.fast_off, M.state + d.state_base, M.topo + H.topo_off);
  double* sc = M.scratch + H.scratch_base;
  const uint32_t nl = align_up(H.n_lane, 2), ns = align_up(H.n_hh + H.n_syn + H.n_clamp, 2);
  U.contrib = sc; U.dcontrib = sc + nl; U.xI = sc + 2 * (size_t)nl;
  U.fgen = U.xI + ns; U.invdgen = U.fgen + H.n_slot;
  U.heads = (uint32_t*)(U.invdgen + H.n_slot);
}

constexpr int kBlockMinCtas = 16;   // latency-bound out of L2: full occupancy beats registers (measured 1..16 x 64..256 threads)
__global__ void __launch_bounds__(kBlockThreads, kBlockMinCtas) cable_block_kernel(DevModel M, StepArgs A) {
  __shared__ UnitHeader H;
  __shared__ __align__(16) uint8_t cell_mem[kCellScratchBytes * kBlockUnitMaxCells];
  const UnitDesc d = M.units[M.n_forests + blockIdx.x];
  if (threadIdx.x < sizeof(UnitHeader) / 4) ((uint32_t*)&H)[threadIdx.x] = ((const uint32_t*)(M.fast + d.fast_off))[threadIdx.x];
  __syncthreads();
  UnitView U;
  block_view(U, M, H, d);
  const CellS cs = carve_cells(cell_mem, kBlockUnitMaxCells);
  unsigned n_sub = 0, n_del = 0;
  run_unit(M, A, U, cs, n_sub, n_del);
  flush_stats(M, n_sub, n_del);
}

// ------------------------------------------------------------------------------------------
// Once per dt: f, 1/d, a, b (and per-synapse decay factors) of every block unit.  One CTA per unit.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBlockThreads) factor_kernel(DevModel M, double dt) {
  __shared__ UnitHeader H;
  const UnitDesc d = M.units[M.n_forests + blockIdx.x];
  if (threadIdx.x < sizeof(UnitHeader) / 4) ((uint32_t*)&H)[threadIdx.x] = ((const uint32_t*)(M.fast + d.fast_off))[threadIdx.x];
  __syncthreads();
  UnitView U;
  make_view(U, M, H, M.fast + d.fast_off, M.state + d.state_base, M.topo + H.topo_off);
  const int64_t lane_base = (int64_t)(((uint64_t)H.pad[1] << 32) | H.pad[0]);
  double* dcontrib = M.factor_dcontrib + lane_base;
  double* f = const_cast<double*>(U.f);
  double* invd = const_cast<double*>(U.invd);
  double* a = const_cast<double*>(U.a);
  double* b = const_cast<double*>(U.b);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int lvl = (int)U.n_level - 1; lvl >= 0; --lvl) {
    for (uint32_t ti = U.level_begin[lvl] + warp; ti < U.level_begin[lvl + 1]; ti += kBlockWarps)
      eliminate_task(U, load_ctx(U, ti, lane), lane, true, dt, f, invd, dcontrib);
    __syncthreads();
  }
  for (uint32_t s = threadIdx.x; s < U.n_slot; s += kBlockThreads) {
    a[s] = U.C[s] / dt - U.G[s];
    b[s] = U.bg[s];
  }
  if (!M.syn_uniform) {
    double* decay = const_cast<double*>(U.syn_decay);
    for (uint32_t i = threadIdx.x; i < U.n_syn; i += kBlockThreads) decay[i] = exp(-dt / U.syn_tau[i]);
  }
  if (U.n_syn >= kSynKeyReduceMin) {   // run heads of the synapse list (order irrelevant)
    __shared__ uint32_t n_heads;
    uint32_t* heads = (uint32_t*)(M.scratch + H.scratch_base + 2 * (size_t)align_up(H.n_lane, 2) +
                                  align_up(H.n_hh + H.n_syn + H.n_clamp, 2) + 2 * (size_t)H.n_slot);
    if (threadIdx.x == 0) n_heads = 0;
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < U.n_syn; i += kBlockThreads)
      if (i == 0 || U.syn_slot[i - 1] != U.syn_slot[i]) heads[1 + atomicAdd(&n_heads, 1u)] = i;
    __syncthreads();
    if (threadIdx.x == 0) heads[0] = n_heads;
  }
}

// R4: gates start at their steady state for the initial voltage.
__global__ void __launch_bounds__(kBlockThreads) init_kernel(DevModel M) {
  __shared__ UnitHeader H;
  const UnitDesc d = M.units[M.n_forests + blockIdx.x];
  if (threadIdx.x < sizeof(UnitHeader) / 4) ((uint32_t*)&H)[threadIdx.x] = ((const uint32_t*)(M.fast + d.fast_off))[threadIdx.x];
  __syncthreads();
  UnitView U;
  make_view(U, M, H, M.fast + d.fast_off, M.state + d.state_base, M.topo + H.topo_off);
  for (uint32_t i = threadIdx.x; i < U.n_hh; i += kBlockThreads) {
    const Rates r = hh_rates(U.V[U.hh_slot[i]]);
    U.m[i] = r.am / (r.am + r.bm);
    U.h[i] = r.ah / (r.ah + r.bh);
    U.n[i] = r.an / (r.an + r.bn);
  }
}

__global__ void reset_detectors_kernel(DevModel M) {
  int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c < M.n_cells) M.state[M.cell_rt_idx[c] + 2] = 1.0;
}

// ------------------------------------------------------------------------------------------
// Epoch boundary: spikes -> events -> per-cell time-sorted lists.
// ------------------------------------------------------------------------------------------
// one warp per new spike walks the out-edges of its source (connection table grouped by source)
__global__ void __launch_bounds__(256) spikes_to_events_kernel(DevModel M, int cur) {
  const unsigned long long n_sp = M.counters[CNT_SPIKES] < (unsigned long long)M.spike_cap ? M.counters[CNT_SPIKES] : (unsigned long long)M.spike_cap;
  const unsigned long long first = M.counters[CNT_SPIKES_DONE];
  const int lane = threadIdx.x & 31;
  const int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = (gridDim.x * (int64_t)blockDim.x) >> 5;
  const EventPool P = M.pool[cur];
  for (unsigned long long s = first + warp; s < n_sp; s += n_warps) {
    const int64_t src = M.gid_base + M.spike_cell[s];
    const double ts = M.spike_t[s];
    for (uint32_t e = M.conn_off[src] + lane; e < M.conn_off[src + 1]; e += 32) {
      const unsigned long long pos = atomicAdd(&M.counters[CNT_POOL], 1ull);
      if ((int64_t)pos < M.pool_cap) {
        P.t[pos] = ts + M.conn_delay[e]; P.dst[pos] = M.conn_dst[e]; P.gidx[pos] = M.conn_gidx[e]; P.w[pos] = M.conn_w[e];
      } else {
        atomicOr(&M.counters[CNT_ERROR], 2ull);
      }
    }
  }
}

// sharded networks: the spikes of the other ranks, gathered into blocks, walk the same table
__global__ void __launch_bounds__(256) remote_spikes_to_events_kernel(DevModel M, int cur, const unsigned long long* blocks, int64_t n_blocks,
                                                                      int64_t cap, int64_t own) {
  const int lane = threadIdx.x & 31;
  const int64_t warp = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = (gridDim.x * (int64_t)blockDim.x) >> 5;
  const EventPool P = M.pool[cur];
  const int64_t stride = 1 + 2 * cap;
  for (int64_t b = 0; b < n_blocks; ++b) {
    if (b == own) continue;
    const unsigned long long* blk = blocks + b * stride;
    const int64_t n = (int64_t)blk[0] < cap ? (int64_t)blk[0] : cap;
    for (int64_t s = warp; s < n; s += n_warps) {
      const int64_t src = (int64_t)blk[1 + s];
      const double ts = __longlong_as_double((long long)blk[1 + cap + s]);
      for (uint32_t e = M.conn_off[src] + lane; e < M.conn_off[src + 1]; e += 32) {
        const unsigned long long pos = atomicAdd(&M.counters[CNT_POOL], 1ull);
        if ((int64_t)pos < M.pool_cap) {
          P.t[pos] = ts + M.conn_delay[e]; P.dst[pos] = M.conn_dst[e]; P.gidx[pos] = M.conn_gidx[e]; P.w[pos] = M.conn_w[e];
        } else {
          atomicOr(&M.counters[CNT_ERROR], 2ull);
        }
      }
    }
  }
}

__global__ void spikes_done_kernel(DevModel M) {
  if (M.counters[CNT_POOL] > M.counters[CNT_POOL_PEAK]) M.counters[CNT_POOL_PEAK] = M.counters[CNT_POOL];
  M.counters[CNT_SPIKES_DONE] = M.counters[CNT_SPIKES] < (unsigned long long)M.spike_cap ? M.counters[CNT_SPIKES] : (unsigned long long)M.spike_cap;
  if (M.counters[CNT_POOL] > (unsigned long long)M.pool_cap) M.counters[CNT_POOL] = (unsigned long long)M.pool_cap;
}

// count per cell: external events before the window end, pool events before the window end
__global__ void ev_count_ext_kernel(DevModel M, double t_win) {
  int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= M.n_cells) return;
  uint32_t p = M.ext_cur[c];
  const uint32_t e = M.ext_off[c + 1];
  uint32_t n = 0;
  while (p + n < e && M.ext_t[p + n] < t_win) ++n;
  M.ev_fill[c] = n;
}

__global__ void ev_count_pool_kernel(DevModel M, int cur, double t_win) {
  const unsigned long long n = M.counters[CNT_POOL];
  const EventPool P = M.pool[cur];
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n; i += gridDim.x * (unsigned long long)blockDim.x)
    if (P.t[i] < t_win) atomicAdd(&M.ev_fill[P.dst[i]], 1u);
}

// exclusive scan of ev_fill[0..n) into ev_off[0..n], three small kernels
constexpr int kScanBlock = 1024;
__global__ void __launch_bounds__(kScanBlock) scan_local_kernel(const uint32_t* in, uint32_t* out, uint32_t* sums, int64_t n) {
  __shared__ uint32_t sh[kScanBlock];
  int64_t i = blockIdx.x * (int64_t)kScanBlock + threadIdx.x;
  uint32_t v = i < n ? in[i] : 0;
  sh[threadIdx.x] = v;
  __syncthreads();
  for (int off = 1; off < kScanBlock; off <<= 1) {
    uint32_t add = threadIdx.x >= off ? sh[threadIdx.x - off] : 0;
    __syncthreads();
    sh[threadIdx.x] += add;
    __syncthreads();
  }
  if (i < n) out[i] = sh[threadIdx.x] - v;
  if (threadIdx.x == kScanBlock - 1) sums[blockIdx.x] = sh[threadIdx.x];
}

__global__ void scan_sums_kernel(uint32_t* sums, int64_t nb, DevModel M, int64_t n) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    unsigned long long acc = 0;
    for (int64_t b = 0; b < nb; ++b) { uint32_t v = sums[b]; sums[b] = (uint32_t)acc; acc += v; }
    if ((int64_t)acc > M.ev_cap) { atomicOr(&M.counters[CNT_ERROR], 4ull); }
    M.ev_off[n] = (uint32_t)(acc > 0xFFFFFFFFull ? 0xFFFFFFFFull : acc);
    M.counters[CNT_EVLIST] = acc;
  }
}

// finish the scan, publish each cell's segment, copy its external events, leave the fill cursor
// behind them
__global__ void ev_place_kernel(DevModel M, double t_win) {
  int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= M.n_cells) return;
  const bool ok = (int64_t)M.counters[CNT_EVLIST] <= M.ev_cap;
  uint32_t off = M.ev_off[c] + M.scan_tmp[c / kScanBlock];
  M.ev_off[c] = off;
  uint32_t p = M.ext_cur[c];
  const uint32_t e = M.ext_off[c + 1];
  uint32_t q = off;
  if (ok) {
    while (p < e && M.ext_t[p] < t_win) { M.ev_t[q] = M.ext_t[p]; M.ev_gidx[q] = M.ext_gidx[p]; M.ev_w[q] = M.ext_w[p]; ++p; ++q; }
    M.ext_cur[c] = p;
  }
  const uint32_t total = M.ev_fill[c];
  M.ev_fill[c] = q;
  const unsigned long long pk = ((unsigned long long)(ok ? off + total : off) << 32) | off;
  M.state[M.cell_rt_idx[c] + 1] = __longlong_as_double((long long)pk);
}

__global__ void ev_scatter_pool_kernel(DevModel M, int cur, double t_win) {
  const unsigned long long n = M.counters[CNT_POOL];
  const EventPool P = M.pool[cur], Q = M.pool[cur ^ 1];
  const bool ok = (int64_t)M.counters[CNT_EVLIST] <= M.ev_cap;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n; i += gridDim.x * (unsigned long long)blockDim.x) {
    const double t = P.t[i];
    if (t < t_win) {
      if (ok) { uint32_t q = atomicAdd(&M.ev_fill[P.dst[i]], 1u); M.ev_t[q] = t; M.ev_gidx[q] = P.gidx[i]; M.ev_w[q] = P.w[i]; }
    } else {
      unsigned long long q = atomicAdd(&M.counters[CNT_POOL_NEXT], 1ull);
      Q.t[q] = t; Q.dst[q] = P.dst[i]; Q.gidx[q] = P.gidx[i]; Q.w[q] = P.w[i];   // q < n <= pool_cap
    }
  }
}

// per cell: order by (time, synapse, weight) - lists are a handful of events long - and publish the
// time of the first one
__global__ void ev_sort_kernel(DevModel M) {
  int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= M.n_cells) return;
  double* rt = M.state + M.cell_rt_idx[c];
  const unsigned long long pk = (unsigned long long)__double_as_longlong(rt[1]);
  const uint32_t b = (uint32_t)pk, e = (uint32_t)(pk >> 32);
  for (uint32_t i = b + 1; i < e; ++i) {
    const double t = M.ev_t[i], w = M.ev_w[i];
    const uint32_t g = M.ev_gidx[i];
    uint32_t j = i;
    while (j > b) {
      const double tj = M.ev_t[j - 1];
      const uint32_t gj = M.ev_gidx[j - 1];
      const bool greater = tj > t || (tj == t && (gj > g || (gj == g && M.ev_w[j - 1] > w)));
      if (!greater) break;
      M.ev_t[j] = tj; M.ev_gidx[j] = gj; M.ev_w[j] = M.ev_w[j - 1];
      --j;
    }
    M.ev_t[j] = t; M.ev_gidx[j] = g; M.ev_w[j] = w;
  }
  rt[0] = b < e ? M.ev_t[b] : CUDART_INF;
}

__global__ void pool_swap_kernel(DevModel M) {
  M.counters[CNT_POOL] = M.counters[CNT_POOL_NEXT];
  M.counters[CNT_POOL_NEXT] = 0;
}

// ------------------------------------------------------------------------------------------
// Point cells (reading R20), one thread per cell, once per epoch: a LIF cell walks its
// epoch's events (time-sorted) - exact relaxation between events, V += w / C_m, spike AT the event that reaches
// the threshold, reset, refractory period; a spike source emits its schedule.
// Record in the state pool: V | runtime triple | t_last | t_ref_end | schedule cursor | pad.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void emit_spike(const DevModel& M, int64_t internal, double t) {
  const unsigned long long pos = atomicAdd(&M.counters[CNT_SPIKES], 1ull);
  if ((int64_t)pos < M.spike_cap) { M.spike_cell[pos] = M.cell_orig[internal]; M.spike_t[pos] = t; }
  else atomicOr(&M.counters[CNT_ERROR], 1ull);
}

__global__ void __launch_bounds__(128) point_cells_kernel(DevModel M, double t_win) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= M.n_pcells) return;
  double* st = M.state + M.pc_state_base + kPcRecord * i;
  const unsigned long long pk = (unsigned long long)__double_as_longlong(st[2]);
  uint32_t cur = (uint32_t)pk;
  const uint32_t end = (uint32_t)(pk >> 32);
  unsigned n_del = 0;
  if (M.pc_kind[i] == 1) {
    const double* par = M.pc_par + 6 * i;
    const double tau = par[0], vth = par[1], cm = par[2], el = par[3], er = par[4], tref = par[5];
    double v = st[0], tl = st[4], tre = st[5];
    for (; cur < end; ++cur) {
      const double te = M.ev_t[cur];
      ++n_del;
      if (te < tre) continue;                              // refractory: the event is lost
      v = el + (v - el) * exp(-(te - tl) / tau);
      tl = te;
      v += M.ev_w[cur] / cm;
      if (v >= vth) {
        emit_spike(M, M.pc_first + i, te);
        v = er; tre = te + tref; tl = tre;
      }
    }
    st[0] = v; st[4] = tl; st[5] = tre;
  } else {
    uint32_t q = M.pc_src_off[i] + (uint32_t)st[6];
    const uint32_t qe = M.pc_src_off[i + 1];
    for (; q < qe && M.pc_src_time[q] < t_win; ++q) emit_spike(M, M.pc_first + i, M.pc_src_time[q]);
    st[6] = (double)(q - M.pc_src_off[i]);
    n_del = end - cur;                                     // events on a source have no effect
    cur = end;
  }
  st[1] = CUDART_INF;
  st[2] = __longlong_as_double((long long)(((unsigned long long)end << 32) | cur));
  if (n_del) atomicAdd(&M.counters[CNT_DELIVERED], (unsigned long long)n_del);
}

// arb_voltage: a LIF cell's potential relaxed from the time of its last event to the current time
__global__ void lif_relax_kernel(DevModel M, double t, double* io) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= M.n_pcells || M.pc_kind[i] != 1) return;
  const double* st = M.state + M.pc_state_base + kPcRecord * i;
  const double* par = M.pc_par + 6 * i;
  if (t > st[4]) io[M.pc_cv[i]] = par[3] + (st[0] - par[3]) * exp(-(t - st[4]) / par[0]);
}

// arb_set_state: the injected V of a LIF cell is its potential at the current time, outside any refractory period
__global__ void point_reset_kernel(DevModel M, double t) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= M.n_pcells) return;
  double* st = M.state + M.pc_state_base + kPcRecord * i;
  st[4] = t; st[5] = -CUDART_INF;
}

// ------------------------------------------------------------------------------------------
// read-back / state injection helpers
// ------------------------------------------------------------------------------------------
__global__ void gather_kernel(const double* state, const uint32_t* idx, int64_t n, double* out) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) out[i] = state[idx[i]];
}
__global__ void gather_syn_kernel(DevModel M, const uint32_t* idx, int64_t n, double t, double* out) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t gx = idx[i];
  double g = M.state[gx];
  if (gx - M.lazy_base < M.lazy_n && g != 0.0) g *= exp(-(t - M.state[gx + M.lazy_n]) / M.state[gx + 2 * (size_t)M.lazy_n]);
  out[i] = g;
}
__global__ void lazy_rebuild_kernel(DevModel M, double t) {
  int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (r >= M.n_runs) return;
  double sum = 0.0;
  for (uint32_t l = M.run_off[r]; l < M.run_off[r + 1]; ++l) { sum += M.state[M.lazy_base + l]; M.state[M.lazy_base + M.lazy_n + l] = t; }
  M.state[M.run_gidx[r]] = sum;
}
__global__ void scatter_kernel(double* state, const uint32_t* idx, int64_t n, const double* in) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) state[idx[i]] = in[i];
}
__global__ void gather_hh_kernel(const double* state, const uint32_t* m_idx, const uint32_t* stride, const uint32_t* cv,
                                 int which, int64_t n, double* out) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) out[cv[i]] = state[m_idx[i] + (uint32_t)which * stride[i]];
}
__global__ void scatter_hh_kernel(double* state, const uint32_t* m_idx, const uint32_t* stride, const uint32_t* cv,
                                  int which, int64_t n, const double* in) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) state[m_idx[i] + (uint32_t)which * stride[i]] = in[cv[i]];
}

inline unsigned grid_for(int64_t n, int block) { return (unsigned)((n + block - 1) / block); }

}  // namespace

int cable_smem_limit() { return 227 * 1024; }   // sm_100a: opt-in maximum of dynamic shared memory per CTA

cudaError_t configure_kernels() {
  int dev = 0, optin = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (e != cudaSuccess) return e;
  e = configure_forest_kernel(optin);
  if (e != cudaSuccess) return e;
  return configure_group_kernel(optin);
}

cudaError_t launch_factor(const DevModel& M, double dt, cudaStream_t s) {
  if (M.n_units == M.n_forests) return cudaSuccess;
  factor_kernel<<<(unsigned)(M.n_units - M.n_forests), kBlockThreads, 0, s>>>(M, dt);
  return cudaGetLastError();
}

cudaError_t launch_init(const DevModel& M, cudaStream_t s) {
  if (M.n_units == M.n_forests) return cudaSuccess;
  init_kernel<<<(unsigned)(M.n_units - M.n_forests), kBlockThreads, 0, s>>>(M);
  return cudaGetLastError();
}

cudaError_t launch_reset_detectors(const DevModel& M, cudaStream_t s) {
  reset_detectors_kernel<<<grid_for(M.n_cells, 256), 256, 0, s>>>(M);
  return cudaGetLastError();
}

cudaError_t launch_cable(const DevModel& M, const StepArgs& A, cudaStream_t s, int* launches) {
  if (M.n_units > M.n_forests) {
    cable_block_kernel<<<(unsigned)(M.n_units - M.n_forests), kBlockThreads, 0, s>>>(M, A);
    if (launches) ++*launches;
  }
  return cudaGetLastError();
}

cudaError_t launch_build_events(const DevModel& M, int cur, double t_win, cudaStream_t s, int* launches) {
  const unsigned gc = grid_for(M.n_cells, 256);
  const int64_t nb = (M.n_cells + kScanBlock - 1) / kScanBlock;
  ev_count_ext_kernel<<<gc, 256, 0, s>>>(M, t_win);
  const unsigned gp = (unsigned)(4 * M.sm_count);      // grid-stride loops over the pool: four CTAs per SM
  ev_count_pool_kernel<<<gp, 256, 0, s>>>(M, cur, t_win);
  scan_local_kernel<<<(unsigned)nb, kScanBlock, 0, s>>>(M.ev_fill, M.ev_off, M.scan_tmp, M.n_cells);
  scan_sums_kernel<<<1, 32, 0, s>>>(M.scan_tmp, nb, M, M.n_cells);
  ev_place_kernel<<<gc, 256, 0, s>>>(M, t_win);
  ev_scatter_pool_kernel<<<gp, 256, 0, s>>>(M, cur, t_win);
  ev_sort_kernel<<<gc, 256, 0, s>>>(M);
  pool_swap_kernel<<<1, 1, 0, s>>>(M);
  if (launches) *launches += 8;
  return cudaGetLastError();
}

cudaError_t launch_spikes_to_events(const DevModel& M, int cur, cudaStream_t s, int* launches) {
  spikes_to_events_kernel<<<(unsigned)(2 * M.sm_count), 256, 0, s>>>(M, cur);
  spikes_done_kernel<<<1, 1, 0, s>>>(M);
  if (launches) *launches += 2;
  return cudaGetLastError();
}

cudaError_t launch_remote_spikes_to_events(const DevModel& M, int cur, const unsigned long long* blocks, int64_t n_blocks, int64_t cap,
                                           int64_t own, cudaStream_t s) {
  remote_spikes_to_events_kernel<<<(unsigned)(2 * M.sm_count), 256, 0, s>>>(M, cur, blocks, n_blocks, cap, own);
  spikes_done_kernel<<<1, 1, 0, s>>>(M);            // records the pool demand and clamps the counter
  return cudaGetLastError();
}

cudaError_t launch_point_cells(const DevModel& M, double t_win, cudaStream_t s, int* launches) {
  if (M.n_pcells == 0) return cudaSuccess;
  point_cells_kernel<<<grid_for(M.n_pcells, 128), 128, 0, s>>>(M, t_win);
  if (launches) ++*launches;
  return cudaGetLastError();
}
cudaError_t launch_lif_relax(const DevModel& M, double t, double* io, cudaStream_t s) {
  if (M.n_pcells == 0) return cudaSuccess;
  lif_relax_kernel<<<grid_for(M.n_pcells, 128), 128, 0, s>>>(M, t, io);
  return cudaGetLastError();
}
cudaError_t launch_point_reset(const DevModel& M, double t, cudaStream_t s) {
  if (M.n_pcells == 0) return cudaSuccess;
  point_reset_kernel<<<grid_for(M.n_pcells, 128), 128, 0, s>>>(M, t);
  return cudaGetLastError();
}

cudaError_t launch_gather(const double* state, const uint32_t* idx, int64_t n, double* out, cudaStream_t s) {
  if (n > 0) gather_kernel<<<grid_for(n, 256), 256, 0, s>>>(state, idx, n, out);
  return cudaGetLastError();
}
cudaError_t launch_gather_syn(const DevModel& M, const uint32_t* idx, int64_t n, double t, double* out, cudaStream_t s) {
  if (n > 0) gather_syn_kernel<<<grid_for(n, 256), 256, 0, s>>>(M, idx, n, t, out);
  return cudaGetLastError();
}
cudaError_t launch_lazy_rebuild(const DevModel& M, double t, cudaStream_t s) {
  if (M.n_runs > 0) lazy_rebuild_kernel<<<grid_for(M.n_runs, 256), 256, 0, s>>>(M, t);
  return cudaGetLastError();
}
cudaError_t launch_scatter(double* state, const uint32_t* idx, int64_t n, const double* in, cudaStream_t s) {
  if (n > 0) scatter_kernel<<<grid_for(n, 256), 256, 0, s>>>(state, idx, n, in);
  return cudaGetLastError();
}
cudaError_t launch_gather_hh(const double* state, const uint32_t* m_idx, const uint32_t* stride, const uint32_t* cv,
                             int which, int64_t n, double* out, cudaStream_t s) {
  if (n > 0) gather_hh_kernel<<<grid_for(n, 256), 256, 0, s>>>(state, m_idx, stride, cv, which, n, out);
  return cudaGetLastError();
}
cudaError_t launch_scatter_hh(double* state, const uint32_t* m_idx, const uint32_t* stride, const uint32_t* cv,
                              int which, int64_t n, const double* in, cudaStream_t s) {
  if (n > 0) scatter_hh_kernel<<<grid_for(n, 256), 256, 0, s>>>(state, m_idx, stride, cv, which, n, in);
  return cudaGetLastError();
}

}  // namespace arbb
