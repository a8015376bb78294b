// forest_kernel.cu - the cable step for forests (forest_layout.h): cells with a tree of their own,
// LANE = CONTROL VOLUME.
//
//   cable_forest_kernel  one CTA per forest (the hardware scheduler deals the CTAs, largest forests
//                        first).  The forest's state record (V, gates, synaptic g, per-cell runtime)
//                        arrives in shared memory by one bulk-async copy (TMA, cp.async.bulk + mbarrier)
//                        and leaves by one bulk store; the coefficient arrays (a, b, f, 1/d) are read
//                        straight from global memory, one coalesced 256-byte row per warp and array,
//                        after a TMA prefetch has pulled the forest's records into L2.
//                        Per grid step (or fused run of steps): event delivery ->
//                        mechanism currents (eq 2a) -> rhs of the implicit Euler system
//                         -> Hines / branched Thomas sweeps as SEGMENTED
//                        WARP SCANS: with the matrix factorised (reading R1) the backward sweep is
//                        r_k = rhs_k - f_{k+1} r_{k+1} and the forward sweep V'_k = r_k/d_k - f_k V'_{k-1},
//                        first-order linear recurrences along a branch; affine maps compose, so 32
//                        consecutive control volumes are swept in five shuffle steps, branch ends
//                        cut the scan by a zero multiplier, a branch longer than 32 carries its
//                        recurrence in a register, and __syncthreads separates the branch LEVELS of
//                        the tree -> V <- V' -> gate and synapse state update with V'
//                        -> threshold test.
//   forest_factor_kernel once per dt: eliminates the constant matrix of every forest
//   forest_init_kernel   gates at their steady state for the initial voltage (reading R4)
//
// HBM-bound by design: 48 B per control volume and step against ~25 fp64 instructions.  No tensor
// cores: nothing here is a dense contraction.
#include "device_common.cuh"
#include "forest_layout.h"
#include "kernels.cuh"

namespace arbb {

namespace {

constexpr int kT = kForestThreads;
constexpr int kW = kForestWarps;

// Pointers of one forest.  V, gates, g, runtime, con, xI address shared memory in the cable kernel
// (global memory in the factor / init kernels); everything else is global.
struct FView {
  uint32_t n_slot, n_branch, n_chunk, n_level, n_cell, n_hh, n_syn, n_clamp, flags;
  const double *f, *invd, *a, *b, *hh_gna, *hh_gk, *hh_gl, *syn_e, *syn_decay, *cl_t0, *cl_t1, *cl_amp;
  const uint32_t *hh_slot, *syn_slot, *cl_slot;
  const uint16_t *hh_cell, *syn_cell, *cl_cell;
  double *V, *m, *h, *n, *g, *rt;
  uint32_t g_gidx0;                 // state-pool index of g[0]
  const FRun* runs; const FChunk* chunks; const FBranch* br; const uint16_t* br_cell;
  const uint32_t *child, *cell_det, *level_br;
  const double *C, *S, *sig, *G, *bg, *syn_tau;
  double *con, *xI;                 // per branch: what its parent loses; per point-mechanism instance: its current
  double *fgen, *invdgen, *dcon;    // global scratch of the forest (event-split sub-steps, factorisation)
  int64_t cell_base;
};

__device__ __forceinline__ void make_fview(FView& U, const DevModel& M, const UnitHeader& H, uint8_t* fast, double* statew) {
  U.n_slot = H.n_slot; U.n_branch = H.n_lane; U.n_chunk = H.n_task; U.n_level = H.n_level;
  U.n_cell = H.n_cell; U.n_hh = H.n_hh; U.n_syn = H.n_syn; U.n_clamp = H.n_clamp; U.flags = H.flags;
  const FastOff fo = fast_offsets(H.n_slot, H.n_hh, H.n_syn, H.n_clamp, H.n_cell, M.syn_uniform != 0);
  U.f = (const double*)(fast + fo.f); U.invd = (const double*)(fast + fo.invd);
  U.a = (const double*)(fast + fo.a); U.b = (const double*)(fast + fo.b);
  U.hh_gna = (const double*)(fast + fo.hh_gna); U.hh_gk = (const double*)(fast + fo.hh_gk); U.hh_gl = (const double*)(fast + fo.hh_gl);
  U.syn_e = (const double*)(fast + fo.syn_e); U.syn_decay = (const double*)(fast + fo.syn_decay);
  U.cl_t0 = (const double*)(fast + fo.cl_t0); U.cl_t1 = (const double*)(fast + fo.cl_t1); U.cl_amp = (const double*)(fast + fo.cl_amp);
  U.hh_slot = (const uint32_t*)(fast + fo.hh_slot); U.syn_slot = (const uint32_t*)(fast + fo.syn_slot); U.cl_slot = (const uint32_t*)(fast + fo.cl_slot);
  U.hh_cell = (const uint16_t*)(fast + fo.hh_cell); U.syn_cell = (const uint16_t*)(fast + fo.syn_cell); U.cl_cell = (const uint16_t*)(fast + fo.cl_cell);
  const StateOff so = state_offsets(H.n_slot, H.n_hh, H.n_syn, H.n_cell);
  U.V = statew + so.v; U.m = statew + so.m; U.h = statew + so.h; U.n = statew + so.n; U.g = statew + so.g; U.rt = statew + so.rt;
  U.g_gidx0 = (uint32_t)(H.state_base + so.g);
  const uint8_t* tp = M.topo + H.topo_off;
  const FTopoOff to = ftopo_offsets(H.n_level, H.n_task, H.n_lane, H.n_child, H.n_cell);
  U.runs = (const FRun*)(tp + to.runs); U.chunks = (const FChunk*)(tp + to.chunks); U.br = (const FBranch*)(tp + to.branches);
  U.br_cell = (const uint16_t*)(tp + to.br_cell); U.child = (const uint32_t*)(tp + to.child);
  U.cell_det = (const uint32_t*)(tp + to.cell_det); U.level_br = (const uint32_t*)(tp + to.level_br);
  const GenOff go = gen_offsets(H.n_slot, H.n_syn);
  const double* gen = M.gen + H.gen_base;
  U.C = gen + go.C; U.S = gen + go.S; U.sig = gen + go.sig; U.G = gen + go.G; U.bg = gen + go.b; U.syn_tau = gen + go.syn_tau;
  const FScratchOff sc = fscratch_offsets(H.n_slot, H.n_lane);
  double* scr = M.scratch + H.scratch_base;
  U.fgen = scr + sc.fgen; U.invdgen = scr + sc.invdgen; U.dcon = scr + sc.dcon;
  U.cell_base = H.cell_base;
}

__device__ __forceinline__ FChunk load_chunk(const FChunk* p) {
  const uint4 q = __ldg((const uint4*)p);
  FChunk c;
  c.slot0 = q.x; c.heads = q.y; c.tails = q.z; c.br_n = q.w;
  return c;
}
__device__ __forceinline__ FBranch load_branch(const FBranch* p) {
  const uint4 q = __ldg((const uint4*)p);
  FBranch b;
  b.slot0 = q.x; b.pslot = q.y; b.cbeg = q.z; b.len = (uint16_t)(q.w & 0xFFFFu); b.ccnt = (uint16_t)(q.w >> 16);
  return b;
}
// branch of `lane` inside a chunk: the branch of lane 0 plus the branch heads met on the way
__device__ __forceinline__ uint32_t branch_of(const FChunk& ck, int lane) {
  const uint32_t upto = 0xFFFFFFFFu >> (31 - lane);
  return (ck.br_n >> 6) + (uint32_t)__popc(ck.heads & upto) - (ck.heads & 1u);
}

// ------------------------------------------------------------------------------------------
// Elimination of the diagonal for one step length, serial along a branch, one
// thread per branch, level by level:  d_k = C_k/delta + S_k - sum_children sigma_c^2 / d_c,
// f_k = -sigma_k / d_k.  Used once per dt for every cell (cs == nullptr) and, on event-split
// sub-steps (reading R9), for the cells that take a step of their own length.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void eliminate_forest(const FView& U, const CellS* cs, double dt, double* fout, double* invdout) {
  constexpr int kB = 8;                   // rows whose C, S, sigma are requested together
  for (int lvl = (int)U.n_level - 1; lvl >= 0; --lvl) {
    const uint32_t b0 = U.level_br[lvl], b1 = U.level_br[lvl + 1];
    for (uint32_t bi = b0 + threadIdx.x; bi < b1; bi += kT) {
      double delta = dt;
      if (cs) {
        const uint32_t c = U.br_cell[bi];
        if (cs->mode[c] != 2u) continue;
        delta = cs->delta[c];
      }
      const FBranch B = load_branch(U.br + bi);
      double carry = 0.0;                 // f_{k+1} sigma_{k+1}: what row k loses to its child in the branch
      for (uint32_t j = 0; j < B.ccnt; ++j) carry -= U.dcon[U.child[B.cbeg + j]];
      double fk = 0.0, sk = 0.0;
      int left = B.len;
      uint32_t s = B.slot0 + B.len - 1;
      while (left > 0) {
        double cr[kB], sr[kB], gr[kB];
#pragma unroll
        for (int j = 0; j < kB; ++j)
          if (j < left) { cr[j] = U.C[s - j]; sr[j] = U.S[s - j]; gr[j] = U.sig[s - j]; }
#pragma unroll
        for (int j = 0; j < kB; ++j)
          if (j < left) {
            const double d = (cr[j] / delta + sr[j]) + carry;
            const double invd = 1.0 / d;
            sk = gr[j];
            fk = -sk * invd;
            fout[s - j] = fk;
            invdout[s - j] = invd;
            carry = fk * sk;              // d_p -= f*u with u = -sigma
          }
        s -= kB;
        left -= kB;
      }
      U.dcon[bi] = -fk * sk;
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------
// Backward (leaves -> root) sweep of one chunk on the rhs held in V:
//   r_k = rhs_k - f_{k+1} r_{k+1} along a branch (suffix scan of affine maps), the last control volume
//   of a branch first loses con[child] = f_0 r_0 of every child branch; every control volume is left
//   holding r_k / d_k, which is what the forward sweep needs.
// cf, cr: f and r of the slot that follows the chunk (the previous chunk of the run), for a branch that
// continues there.
// ------------------------------------------------------------------------------------------
template <bool kGen>
__device__ __forceinline__ void backward_chunk(const FView& U, const CellS& cs, const FChunk& ck, int lane, double& cf, double& cr) {
  const int n = (int)(ck.br_n & 63u);
  const bool valid = lane < n;
  const uint32_t s = ck.slot0 + lane;
  const bool head = (ck.heads >> lane) & 1u, tail = (ck.tails >> lane) & 1u;
  const uint32_t br = branch_of(ck, lane);
  uint32_t md = 1u;
  double r = 0.0, f = 0.0, invd = 0.0;
  if (valid) {
    if (kGen) md = cs.mode[U.br_cell[br]];
    r = U.V[s];
    if (kGen && md == 2u) { f = U.fgen[s]; invd = U.invdgen[s]; }
    else { f = __ldg(U.f + s); invd = __ldg(U.invd + s); }
    if (tail) {
      const FBranch B = load_branch(U.br + br);
      for (uint32_t j = 0; j < B.ccnt; ++j) r -= U.con[__ldg(U.child + B.cbeg + j)];
    }
  }
  const double fnext = __shfl_down_sync(kFull, f, 1);
  double a = 0.0;                              // multiplier of r_{k+1} in r_k; 0 cuts the chain
  if (valid && !tail) {
    if (lane == n - 1) r = fma(-cf, cr, r);    // the branch continues in the chunk swept before this one
    else a = -fnext;
  }
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const double a2 = __shfl_down_sync(kFull, a, d);
    const double r2 = __shfl_down_sync(kFull, r, d);
    if (lane + d < 32) { r = fma(a, r2, r); a *= a2; }
  }
  if (valid && md) {
    U.V[s] = r * invd;
    if (head) U.con[br] = f * r;
  }
  cf = __shfl_sync(kFull, f, 0);
  cr = __shfl_sync(kFull, r, 0);
}

// Forward (root -> leaves) substitution of one chunk: V'_k = r_k/d_k - f_k V'_{k-1}; V <- V'.
// cv: V' of the slot before the chunk (the chunk of the run swept before this one).
template <bool kGen>
__device__ __forceinline__ void forward_chunk(const FView& U, const CellS& cs, const FChunk& ck, int lane, double& cv) {
  const int n = (int)(ck.br_n & 63u);
  const bool valid = lane < n;
  const uint32_t s = ck.slot0 + lane;
  const bool head = (ck.heads >> lane) & 1u;
  const uint32_t br = branch_of(ck, lane);
  uint32_t md = 1u;
  double a = 0.0, b = 0.0;
  if (valid) {
    if (kGen) md = cs.mode[U.br_cell[br]];
    const double q = U.V[s];
    const double f = (kGen && md == 2u) ? U.fgen[s] : __ldg(U.f + s);
    if (head) {
      const uint32_t ps = __ldg(&U.br[br].pslot);
      b = ps != kNoSlot ? fma(-f, U.V[ps], q) : q;
    } else if (lane == 0) {
      b = fma(-f, cv, q);
    } else {
      a = -f; b = q;
    }
  }
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const double a2 = __shfl_up_sync(kFull, a, d);
    const double b2 = __shfl_up_sync(kFull, b, d);
    if (lane >= d) { b = fma(a, b2, b); a *= a2; }
  }
  if (valid && md) U.V[s] = b;
  cv = __shfl_sync(kFull, b, n - 1);
}

// ------------------------------------------------------------------------------------------
// One (sub-)step of every active cell of the forest, phases B..F (phase A, event delivery and the choice
// of the sub-step, is in run_forest).  kGen: cells may be inactive (mode 0) or on an event-split
// sub-step of their own length (mode 2).
// ------------------------------------------------------------------------------------------
template <bool kGen>
__device__ __forceinline__ void forest_substep(const DevModel& M, const FView& U, const CellS& cs, double dt) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool multi = U.n_cell > 1;
  const uint32_t n_hh = U.n_hh, n_syn = U.n_syn, n_cl = U.n_clamp;

  // event-split sub-steps: those cells' matrices are eliminated for their own step length (reading R9)
  if (kGen) {
    bool split = false;
    if ((uint32_t)tid < U.n_cell) split = cs.mode[tid] == 2u;
    if (__syncthreads_or(split)) eliminate_forest(U, &cs, dt, U.fgen, U.invdgen);
  }

  // ---- B: currents of HH, synapses and clamps from V(t); the passive current is
  // folded into a, b.  Items on one CV form a run; the first item of a run sums it in index order.
  for (uint32_t i = tid; i < n_hh; i += kT) {
    if (kGen && !cs.mode[multi ? U.hh_cell[i] : 0]) continue;
    const double v = U.V[__ldg(U.hh_slot + i)];
    const double m = U.m[i], h = U.h[i], n = U.n[i];
    U.xI[i] = __ldg(U.hh_gna + i) * m * m * m * h * (v - M.ena) + __ldg(U.hh_gk + i) * n * n * n * n * (v - M.ek) + __ldg(U.hh_gl + i) * (v - M.el);
  }
  for (uint32_t i = tid; i < n_syn; i += kT) {
    const uint32_t slot = __ldg(U.syn_slot + i);
    if (i > 0 && __ldg(U.syn_slot + i - 1) == slot) continue;
    if (kGen && !cs.mode[multi ? U.syn_cell[i] : 0]) continue;
    const double v = U.V[slot];
    double I = 0.0;
    uint32_t j = i;
    do {
      I += U.g[j] * (v - (M.syn_uniform ? M.syn_e_u : __ldg(U.syn_e + j)));
      ++j;
    } while (j < n_syn && __ldg(U.syn_slot + j) == slot);
    U.xI[n_hh + i] = I;
  }
  for (uint32_t i = tid; i < n_cl; i += kT) {
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
  __syncthreads();

  // ---- C: rhs_i = (C_i/delta - G_i) V_i + G_i e_i - I_i, in place of V
  if (!kGen) {
    const uint32_t n = U.n_slot;
#pragma unroll 4
    for (uint32_t s = tid; s < n; s += kT) U.V[s] = fma(__ldg(U.a + s), U.V[s], __ldg(U.b + s));
  } else {
    for (uint32_t ci = warp; ci < U.n_chunk; ci += kW) {
      const FChunk ck = load_chunk(U.chunks + ci);
      if (lane >= (int)(ck.br_n & 63u)) continue;
      const uint32_t c = U.br_cell[branch_of(ck, lane)], md = cs.mode[c];
      const uint32_t s = ck.slot0 + lane;
      if (md == 1u) U.V[s] = fma(__ldg(U.a + s), U.V[s], __ldg(U.b + s));
      else if (md == 2u) U.V[s] = fma(U.C[s] / cs.delta[c] - U.G[s], U.V[s], U.bg[s]);
    }
  }
  __syncthreads();
  // HH, synapse and clamp currents of a cell may meet on a control volume: barriers in between, unless the
  // host found that they never do in this forest
  const bool disjoint = (U.flags & UNIT_POINT_DISJOINT) != 0;
  if (n_hh) {
    for (uint32_t i = tid; i < n_hh; i += kT) {
      if (kGen && !cs.mode[multi ? U.hh_cell[i] : 0]) continue;
      U.V[__ldg(U.hh_slot + i)] -= U.xI[i];
    }
    if (!disjoint) __syncthreads();
  }
  if (n_syn) {
    for (uint32_t i = tid; i < n_syn; i += kT) {
      const uint32_t slot = __ldg(U.syn_slot + i);
      if (i > 0 && __ldg(U.syn_slot + i - 1) == slot) continue;
      if (kGen && !cs.mode[multi ? U.syn_cell[i] : 0]) continue;
      U.V[slot] -= U.xI[n_hh + i];
    }
    if (!disjoint) __syncthreads();
  }
  if (n_cl) {
    for (uint32_t i = tid; i < n_cl; i += kT) {
      const uint32_t slot = U.cl_slot[i];
      if (i > 0 && U.cl_slot[i - 1] == slot) continue;
      if (kGen && !cs.mode[multi ? U.cl_cell[i] : 0]) continue;
      U.V[slot] -= U.xI[n_hh + n_syn + i];
    }
    if (!disjoint) __syncthreads();
  }
  if (disjoint && (n_hh | n_syn | n_cl)) __syncthreads();

  // ---- D: backward sweep, deepest level first; E: forward substitution, root first; V <- V'
  for (int lvl = (int)U.n_level - 1; lvl >= 0; --lvl) {
    const FRun R = U.runs[lvl * kW + warp];
    double cf = 0.0, cr = 0.0;
    for (uint32_t ci = R.chunk_end; ci-- > R.chunk_beg;) backward_chunk<kGen>(U, cs, load_chunk(U.chunks + ci), lane, cf, cr);
    __syncthreads();
  }
  for (uint32_t lvl = 0; lvl < U.n_level; ++lvl) {
    const FRun R = U.runs[lvl * kW + warp];
    double cv = 0.0;
    for (uint32_t ci = R.chunk_beg; ci < R.chunk_end; ++ci) forward_chunk<kGen>(U, cs, load_chunk(U.chunks + ci), lane, cv);
    __syncthreads();
  }

  // ---- F: state update with V', threshold test
  for (uint32_t i = tid; i < n_hh; i += kT) {
    const uint32_t c = (kGen && multi) ? U.hh_cell[i] : 0;
    if (kGen && !cs.mode[c]) continue;
    const double delta = kGen ? cs.delta[c] : dt;
    const Rates r = hh_rates(U.V[__ldg(U.hh_slot + i)]);
    double inf = r.am / (r.am + r.bm);
    U.m[i] = inf + (U.m[i] - inf) * exp(-delta * (r.am + r.bm));
    inf = r.ah / (r.ah + r.bh);
    U.h[i] = inf + (U.h[i] - inf) * exp(-delta * (r.ah + r.bh));
    inf = r.an / (r.an + r.bn);
    U.n[i] = inf + (U.n[i] - inf) * exp(-delta * (r.an + r.bn));
  }
  for (uint32_t i = tid; i < n_syn; i += kT) {
    const uint32_t c = (kGen && multi) ? U.syn_cell[i] : 0;
    const uint32_t md = kGen ? cs.mode[c] : 1u;
    if (!md) continue;
    double decay;
    if (md == 1u) decay = M.syn_uniform ? M.syn_decay_u : __ldg(U.syn_decay + i);
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
      cs.armed[tid] = 0;
    }
    if (vd < M.theta && !cs.armed[tid]) cs.armed[tid] = 1;
    cs.tcur[tid] = cs.tnext[tid];
  }
  __syncthreads();
}

// ------------------------------------------------------------------------------------------
// A.nk grid steps of one forest.  Phase A: deliver the events due now and choose each cell's
// sub-step (reading R9), then the step itself.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void run_forest(const DevModel& M, const StepArgs& A, const FView& U, const CellS& cs,
                                           unsigned& n_sub, unsigned& n_del) {
  const int tid = threadIdx.x;
  const uint32_t n_cell = U.n_cell;
  if ((uint32_t)tid < n_cell) {
    const unsigned long long pk = (unsigned long long)__double_as_longlong(U.rt[kRtDoubles * tid + 1]);
    cs.evcur[tid] = (uint32_t)pk; cs.evend[tid] = (uint32_t)(pk >> 32);
    cs.armed[tid] = U.rt[kRtDoubles * tid + 2] != 0.0 ? 1u : 0u;
  }
  for (int64_t k = A.k_first; k < A.k_first + A.nk; ++k) {
    const double ta = (k == 0) ? A.t0 : __dadd_rn(A.t0, __dmul_rn((double)k, A.dt));
    const double tb = (k + 1 == A.nsteps) ? A.t_end : __dadd_rn(A.t0, __dmul_rn((double)(k + 1), A.dt));
    const bool nominal = (k + 1 < A.nsteps) || A.last_full;
    if ((uint32_t)tid < n_cell) cs.tcur[tid] = ta;
    __syncthreads();
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
            while (cur < end && M.ev_t[cur] <= t) { U.g[M.ev_gidx[cur] - U.g_gidx0] += M.ev_w[cur]; ++cur; ++n_del; }
            tn = cur < end ? M.ev_t[cur] : CUDART_INF;
            cs.evcur[tid] = cur; U.rt[kRtDoubles * tid] = tn;
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
      // one barrier decides both questions: bit 0 = some cell is active, bit 1 = some cell is not on a plain step
      const int any_active = __syncthreads_or(active);
      if (!any_active) break;
      const int general = __syncthreads_or(!plain);
      if (general) forest_substep<true>(M, U, cs, A.dt);
      else forest_substep<false>(M, U, cs, A.dt);
    }
  }
  if ((uint32_t)tid < n_cell) {
    const unsigned long long pk = ((unsigned long long)cs.evend[tid] << 32) | cs.evcur[tid];
    U.rt[kRtDoubles * tid + 1] = __longlong_as_double((long long)pk);
    U.rt[kRtDoubles * tid + 2] = cs.armed[tid] ? 1.0 : 0.0;
  }
}

// ------------------------------------------------------------------------------------------
// The cable step for forests: one CTA per forest of launch class `cls`.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kForestThreads, 8) cable_forest_kernel(DevModel M, StepArgs A, int cls) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ UnitHeader H;
  const ForestSmemPlan P = M.fcls[cls].plan;
  const UnitDesc d = M.units[M.fcls[cls].first + blockIdx.x];
  uint8_t* fast = M.fast + d.fast_off;
  double* Ss = (double*)smem;
  uint64_t* mbar = (uint64_t*)(smem + P.off_mbar);
  const int tid = threadIdx.x;
  if (tid == 0) {
    mbar_init(mbar, 1);
    fence_mbar_init();
    fence_proxy_async();
    mbar_expect_tx(mbar, d.state_bytes);
    bulk_g2s(Ss, M.state + d.state_base, d.state_bytes, mbar);
    bulk_prefetch_l2(fast, d.fast_bytes);            // coefficients and instance tables -> L2
  }
  if (tid < (int)(sizeof(UnitHeader) / 4)) ((uint32_t*)&H)[tid] = __ldg((const uint32_t*)fast + tid);
  __syncthreads();
  FView U;
  make_fview(U, M, H, fast, Ss);
  U.con = (double*)(smem + P.off_con);
  U.xI = (double*)(smem + P.off_xi);
  const CellS cs = carve_cells(smem + P.off_cell, U.n_cell);
  mbar_wait(mbar, 0);
  unsigned n_sub = 0, n_del = 0;
  run_forest(M, A, U, cs, n_sub, n_del);
  // ---- state record -> HBM (one bulk store)
  fence_proxy_async();
  __syncthreads();
  if (tid == 0) {
    bulk_s2g(M.state + d.state_base, Ss, d.state_bytes);
    bulk_commit();
    bulk_wait_read0();
  }
  for (int o = 16; o; o >>= 1) { n_sub += __shfl_xor_sync(kFull, n_sub, o); n_del += __shfl_xor_sync(kFull, n_del, o); }
  if ((tid & 31) == 0) {
    if (n_sub) atomicAdd(&M.counters[CNT_SUBSTEPS], (unsigned long long)n_sub);
    if (n_del) atomicAdd(&M.counters[CNT_DELIVERED], (unsigned long long)n_del);
  }
}

// ------------------------------------------------------------------------------------------
// Once per dt: f, 1/d, a, b (and per-synapse decay factors) of every forest.  One CTA per forest.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kForestThreads) forest_factor_kernel(DevModel M, double dt) {
  __shared__ UnitHeader H;
  const UnitDesc d = M.units[blockIdx.x];
  uint8_t* fast = M.fast + d.fast_off;
  if (threadIdx.x < sizeof(UnitHeader) / 4) ((uint32_t*)&H)[threadIdx.x] = ((const uint32_t*)fast)[threadIdx.x];
  __syncthreads();
  FView U;
  make_fview(U, M, H, fast, M.state + d.state_base);
  eliminate_forest(U, nullptr, dt, const_cast<double*>(U.f), const_cast<double*>(U.invd));
  double* a = const_cast<double*>(U.a);
  double* b = const_cast<double*>(U.b);
  for (uint32_t s = threadIdx.x; s < U.n_slot; s += kT) {
    a[s] = U.C[s] / dt - U.G[s];
    b[s] = U.bg[s];
  }
  if (!M.syn_uniform) {
    double* decay = const_cast<double*>(U.syn_decay);
    for (uint32_t i = threadIdx.x; i < U.n_syn; i += kT) decay[i] = exp(-dt / U.syn_tau[i]);
  }
}

// R4: gates start at their steady state for the initial voltage.
__global__ void __launch_bounds__(kForestThreads) forest_init_kernel(DevModel M) {
  __shared__ UnitHeader H;
  const UnitDesc d = M.units[blockIdx.x];
  uint8_t* fast = M.fast + d.fast_off;
  if (threadIdx.x < sizeof(UnitHeader) / 4) ((uint32_t*)&H)[threadIdx.x] = ((const uint32_t*)fast)[threadIdx.x];
  __syncthreads();
  FView U;
  make_fview(U, M, H, fast, M.state + d.state_base);
  for (uint32_t i = threadIdx.x; i < U.n_hh; i += kT) {
    const Rates r = hh_rates(U.V[U.hh_slot[i]]);
    U.m[i] = r.am / (r.am + r.bm);
    U.h[i] = r.ah / (r.ah + r.bh);
    U.n[i] = r.an / (r.an + r.bn);
  }
}

}  // namespace

cudaError_t configure_forest_kernel(int max_optin_bytes) {
  cudaFuncAttributes fa;
  cudaError_t e = cudaFuncGetAttributes(&fa, cable_forest_kernel);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(cable_forest_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_optin_bytes - (int)fa.sharedSizeBytes);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(cable_forest_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
}

cudaError_t launch_forest_factor(const DevModel& M, double dt, cudaStream_t s) {
  if (M.n_forests == 0) return cudaSuccess;
  forest_factor_kernel<<<(unsigned)M.n_forests, kForestThreads, 0, s>>>(M, dt);
  return cudaGetLastError();
}

cudaError_t launch_forest_init(const DevModel& M, cudaStream_t s) {
  if (M.n_forests == 0) return cudaSuccess;
  forest_init_kernel<<<(unsigned)M.n_forests, kForestThreads, 0, s>>>(M);
  return cudaGetLastError();
}

cudaError_t launch_forest_cable(const DevModel& M, const StepArgs& A, int cls, cudaStream_t s, int* launches) {
  const ForestClass& K = M.fcls[cls];
  if (K.count == 0) return cudaSuccess;
  cable_forest_kernel<<<(unsigned)K.count, kForestThreads, K.plan.bytes, s>>>(M, A, cls);
  if (launches) ++*launches;
  return cudaGetLastError();
}

}  // namespace arbb
