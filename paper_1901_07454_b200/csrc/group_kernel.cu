// group_kernel.cu - the cable step for cell groups (group_layout.h): cells of one topology class,
// stored cell-interleaved, lane = cell.
//
//   cable_group_kernel   persistent grid, one CTA integrates one group at a time.  The group's
//                        voltages arrive in shared memory by one bulk-async copy (TMA,
//                        cp.async.bulk + mbarrier) and leave by one bulk store; the coefficient
//                        rows (a, b, f, 1/d) stream from HBM / L2 straight into registers with
//                        coalesced loads, eight rows in flight per lane group; the next group's
//                        records are pulled into L2 by a TMA prefetch while this one is integrated.
//                        Per grid step (or fused run of steps): event delivery ->
//                        mechanism currents (eq 2a) -> rhs of the implicit Euler system
//                         -> Hines / branched Thomas sweeps: the class
//                        schedule cuts the tree into stages of independent chunks, the CTA's lane
//                        groups eliminate the chunks of a stage concurrently -> V <- V' -> gate and
//                        synapse state update with V' -> threshold test.
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
constexpr int kRows = 8;                  // rows a lane group keeps in flight in a sweep

struct GView {
  uint32_t n_cv, n_cell, n_hh, n_syn, n_cl;          // rows
  const double *f, *invd, *a, *b, *hh_gna, *hh_gk, *hh_gl, *syn_e, *syn_decay, *cl_t0, *cl_t1, *cl_amp;
  const uint16_t *hh_slot, *syn_slot, *cl_slot, *det_slot;
  double *gV, *gm, *gh, *gn, *gg, *grt;
  const double *C, *S, *sig, *G, *bg, *syn_tau;
  const SegRec* segs;
  const uint16_t *order, *sched, *child;
  uint32_t n_stage, n_seg;
  int64_t cell_base;
};

__device__ __forceinline__ void make_gview(GView& U, const DevModel& M, const GroupDesc& D) {
  U.n_cv = D.n_cv; U.n_cell = D.n_cell; U.n_hh = D.n_hh_rows; U.n_syn = D.n_syn_rows; U.n_cl = D.n_cl_rows;
  const GConstOff co = gconst_offsets(D.n_cv, D.n_hh_rows, D.n_syn_rows, D.n_cl_rows, M.syn_uniform != 0);
  const uint8_t* cb = M.fast + D.const_off;
  U.f = (const double*)(cb + co.f); U.invd = (const double*)(cb + co.invd);
  U.a = (const double*)(cb + co.a); U.b = (const double*)(cb + co.b);
  U.hh_gna = (const double*)(cb + co.hh_gna); U.hh_gk = (const double*)(cb + co.hh_gk); U.hh_gl = (const double*)(cb + co.hh_gl);
  U.syn_e = (const double*)(cb + co.syn_e); U.syn_decay = (const double*)(cb + co.syn_decay);
  U.cl_t0 = (const double*)(cb + co.cl_t0); U.cl_t1 = (const double*)(cb + co.cl_t1); U.cl_amp = (const double*)(cb + co.cl_amp);
  U.hh_slot = (const uint16_t*)(cb + co.hh_slot); U.syn_slot = (const uint16_t*)(cb + co.syn_slot);
  U.cl_slot = (const uint16_t*)(cb + co.cl_slot); U.det_slot = (const uint16_t*)(cb + co.det_slot);
  const GStateOff so = gstate_offsets(D.n_cv, D.n_hh_rows, D.n_syn_rows);
  double* gs = M.state + D.state_base;
  U.gV = gs + so.v; U.gm = gs + so.m; U.gh = gs + so.h; U.gn = gs + so.n; U.gg = gs + so.g; U.grt = gs + so.rt;
  const GGenOff go = ggen_offsets(D.n_cv, D.n_syn_rows);
  const double* gen = M.gen + D.gen_base;
  U.C = gen + go.C; U.S = gen + go.S; U.sig = gen + go.sig; U.G = gen + go.G; U.bg = gen + go.b; U.syn_tau = gen + go.syn_tau;
  const uint8_t* cp = M.topo + D.class_off;
  const ClassRecord* R = (const ClassRecord*)cp;
  U.n_stage = R->n_stage; U.n_seg = R->n_seg;
  U.segs = (const SegRec*)(cp + R->off_segs);
  U.order = (const uint16_t*)(cp + R->off_order);
  U.sched = (const uint16_t*)(cp + R->off_sched);
  U.child = (const uint16_t*)(cp + R->off_child);
  U.cell_base = D.cell_base;
}

__device__ __forceinline__ SegRec load_seg(const SegRec* p) {
  const uint4 q = __ldg((const uint4*)p);
  SegRec s;
  s.slot0 = q.x; s.pslot = q.y; s.len = (uint16_t)(q.z & 0xFFFFu); s.ccnt = (uint16_t)(q.z >> 16); s.cbeg = q.w;
  return s;
}

// ------------------------------------------------------------------------------------------
// Elimination of the diagonal of one segment for step length delta (factorisation; event-split
// sub-steps):  d_k = C_k/delta + S_k - sum_children sigma_c^2 / d_c ;  f_k = -sigma_k / d_k.
// dcon[segment] = sigma_0^2 / d_0 is what the parent control volume loses.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void eliminate_seg(const GView& U, const SegRec& sg, uint32_t seg_idx, int c, double delta,
                                              double* fout, double* invdout, double* dcon) {
  uint32_t s = (sg.slot0 + sg.len - 1) * kG + c;
  double d = U.C[s] / delta + U.S[s];
  for (uint32_t j = 0; j < sg.ccnt; ++j) d -= dcon[(uint32_t)U.child[sg.cbeg + j] * kG + c];
  double fk = 0.0, sk = 0.0;
  for (uint32_t k = sg.len; k-- > 0;) {
    const double invd = 1.0 / d;
    sk = U.sig[s];
    fk = -sk * invd;
    fout[s] = fk;
    invdout[s] = invd;
    if (k > 0) {
      s -= kG;
      d = fma(fk, sk, U.C[s] / delta + U.S[s]);      // d_p -= f*u with u = -sigma
    }
  }
  dcon[seg_idx * kG + c] = -fk * sk;
}

// ------------------------------------------------------------------------------------------
// Backward (leaves -> root) sweep of one segment on the rhs held in Vs:
//   rhs_{k-1} -= f_k rhs_k along the segment; the parent control volume loses con[segment] = f_0 rhs_0;
// every control volume is left holding rhs_k / d_k, which is what the forward sweep needs.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void backward_seg(const GView& U, const SegRec& sg, uint32_t seg_idx, int c,
                                             const double* __restrict__ F, const double* __restrict__ I,
                                             double* Vs, double* con) {
  uint32_t s = (sg.slot0 + sg.len - 1) * kG + c;
  double fp = 0.0, rp = 0.0;
  int left = sg.len;
  bool first = true;
  while (left > 0) {
    double fr[kRows], ir[kRows], vr[kRows];
#pragma unroll
    for (int j = 0; j < kRows; ++j)
      if (j < left) { fr[j] = F[s - j * kG]; ir[j] = I[s - j * kG]; vr[j] = Vs[s - j * kG]; }
    if (first) {
      for (uint32_t j = 0; j < sg.ccnt; ++j) vr[0] -= con[(uint32_t)U.child[sg.cbeg + j] * kG + c];
      first = false;
    }
#pragma unroll
    for (int j = 0; j < kRows; ++j)
      if (j < left) {
        const double r = fma(-fp, rp, vr[j]);
        Vs[s - j * kG] = r * ir[j];
        fp = fr[j]; rp = r;
      }
    s -= kRows * kG;
    left -= kRows;
  }
  con[seg_idx * kG + c] = fp * rp;
}

// Forward (root -> leaves) substitution of one segment: V'_k = rhs_k/d_k - f_k V'_{k-1}; V <- V'.
__device__ __forceinline__ void forward_seg(const SegRec& sg, int c, const double* __restrict__ F, double* Vs) {
  double vp = sg.pslot != kNoSlot ? Vs[sg.pslot * kG + c] : 0.0;
  uint32_t s = sg.slot0 * kG + c;
  int left = sg.len;
  while (left > 0) {
    double fr[kRows], vr[kRows];
#pragma unroll
    for (int j = 0; j < kRows; ++j)
      if (j < left) { fr[j] = F[s + j * kG]; vr[j] = Vs[s + j * kG]; }
#pragma unroll
    for (int j = 0; j < kRows; ++j)
      if (j < left) {
        vp = fma(-fr[j], vp, vr[j]);
        Vs[s + j * kG] = vp;
      }
    s += kRows * kG;
    left -= kRows;
  }
}

// ------------------------------------------------------------------------------------------
// One (sub-)step of every active cell of the group (phases B..F; phase A, event delivery and the
// choice of the sub-step, is in the kernel body).  md / delta are this thread's cell's.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void group_substep(const DevModel& M, const GView& U, double* Vs, double* buf, const CellS& cs,
                                              double* fgen, double* invdgen, bool any_gen, uint32_t md, double delta) {
  const int tid = threadIdx.x, c = tid % kG, h = tid / kG;
  const uint32_t nE_cv = U.n_cv * kG, nE_hh = U.n_hh * kG, nE_syn = U.n_syn * kG, nE_cl = U.n_cl * kG;
  const uint32_t n_stage = U.n_stage;

  // ---- event-split sub-steps: this cell's matrix is re-eliminated for its own delta (reading R9)
  if (any_gen) {
    for (uint32_t st = 0; st < n_stage; ++st) {
      const uint32_t beg = U.sched[st * kGroupSlots + h], end = U.sched[st * kGroupSlots + h + 1];
      if (md == 2u)
        for (uint32_t q = beg; q < end; ++q) {
          const uint32_t si = U.order[q];
          eliminate_seg(U, load_seg(U.segs + si), si, c, delta, fgen, invdgen, buf);
        }
      __syncthreads();
    }
  }

  // ---- B: currents of HH, synapses and clamps from V(t); the passive current is
  // folded into a, b.  Items of one cell on one CV form a run; its first item sums it in index order.
  double* xI = buf;
  for (uint32_t e = tid; e < nE_hh; e += kT) {
    const uint32_t slot = U.hh_slot[e];
    if (slot == kNoSlot16 || !md) continue;
    const double v = Vs[slot * kG + c];
    const double m = U.gm[e], hh = U.gh[e], n = U.gn[e];
    xI[e] = U.hh_gna[e] * m * m * m * hh * (v - M.ena) + U.hh_gk[e] * n * n * n * n * (v - M.ek) + U.hh_gl[e] * (v - M.el);
  }
  for (uint32_t e = tid; e < nE_syn; e += kT) {
    const uint32_t slot = U.syn_slot[e];
    if (slot == kNoSlot16 || !md) continue;
    if (e >= (uint32_t)kG && U.syn_slot[e - kG] == slot) continue;
    const double v = Vs[slot * kG + c];
    double I = 0.0;
    uint32_t j = e;
    do {
      I += U.gg[j] * (v - (M.syn_uniform ? M.syn_e_u : U.syn_e[j]));
      j += kG;
    } while (j < nE_syn && U.syn_slot[j] == slot);
    xI[nE_hh + e] = I;
  }
  if (nE_cl) {
    const double t = cs.tcur[c];
    for (uint32_t e = tid; e < nE_cl; e += kT) {
      const uint32_t slot = U.cl_slot[e];
      if (slot == kNoSlot16 || !md) continue;
      if (e >= (uint32_t)kG && U.cl_slot[e - kG] == slot) continue;
      double I = 0.0;
      uint32_t j = e;
      do {
        if (U.cl_t0[j] <= t && t < U.cl_t1[j]) I -= U.cl_amp[j];
        j += kG;
      } while (j < nE_cl && U.cl_slot[j] == slot);
      xI[nE_hh + nE_syn + e] = I;
    }
  }
  __syncthreads();

  // ---- C: rhs_i = (C_i/delta - G_i) V_i + G_i e_i - I_i, in place of V
  if (md == 1u) {
    uint32_t e = tid;
    for (; e + 3 * kT < nE_cv; e += 4 * kT) {
      const double a0 = U.a[e], a1 = U.a[e + kT], a2 = U.a[e + 2 * kT], a3 = U.a[e + 3 * kT];
      const double b0 = U.b[e], b1 = U.b[e + kT], b2 = U.b[e + 2 * kT], b3 = U.b[e + 3 * kT];
      Vs[e] = fma(a0, Vs[e], b0); Vs[e + kT] = fma(a1, Vs[e + kT], b1);
      Vs[e + 2 * kT] = fma(a2, Vs[e + 2 * kT], b2); Vs[e + 3 * kT] = fma(a3, Vs[e + 3 * kT], b3);
    }
    for (; e < nE_cv; e += kT) Vs[e] = fma(U.a[e], Vs[e], U.b[e]);
  } else if (md == 2u) {
    for (uint32_t e = tid; e < nE_cv; e += kT) Vs[e] = fma(U.C[e] / delta - U.G[e], Vs[e], U.bg[e]);
  }
  __syncthreads();
  if (nE_hh) {
    for (uint32_t e = tid; e < nE_hh; e += kT) {
      const uint32_t slot = U.hh_slot[e];
      if (slot == kNoSlot16 || !md) continue;
      Vs[slot * kG + c] -= xI[e];
    }
    __syncthreads();
  }
  if (nE_syn) {
    for (uint32_t e = tid; e < nE_syn; e += kT) {
      const uint32_t slot = U.syn_slot[e];
      if (slot == kNoSlot16 || !md) continue;
      if (e >= (uint32_t)kG && U.syn_slot[e - kG] == slot) continue;
      Vs[slot * kG + c] -= xI[nE_hh + e];
    }
    __syncthreads();
  }
  if (nE_cl) {
    for (uint32_t e = tid; e < nE_cl; e += kT) {
      const uint32_t slot = U.cl_slot[e];
      if (slot == kNoSlot16 || !md) continue;
      if (e >= (uint32_t)kG && U.cl_slot[e - kG] == slot) continue;
      Vs[slot * kG + c] -= xI[nE_hh + nE_syn + e];
    }
    __syncthreads();
  }

  // ---- D: backward sweep, stage by stage; E: forward substitution, stages reversed; V <- V'
  const double* F = md == 2u ? fgen : U.f;
  const double* I = md == 2u ? invdgen : U.invd;
  double* con = buf;                    // xI is dead
  for (uint32_t st = 0; st < n_stage; ++st) {
    const uint32_t beg = U.sched[st * kGroupSlots + h], end = U.sched[st * kGroupSlots + h + 1];
    if (md)
      for (uint32_t q = beg; q < end; ++q) {
        const uint32_t si = U.order[q];
        backward_seg(U, load_seg(U.segs + si), si, c, F, I, Vs, con);
      }
    __syncthreads();
  }
  for (uint32_t st = n_stage; st-- > 0;) {
    const uint32_t beg = U.sched[st * kGroupSlots + h], end = U.sched[st * kGroupSlots + h + 1];
    if (md)
      for (uint32_t q = end; q-- > beg;) forward_seg(load_seg(U.segs + U.order[q]), c, F, Vs);
    __syncthreads();
  }

  // ---- F: state update with V', threshold test
  for (uint32_t e = tid; e < nE_hh; e += kT) {
    const uint32_t slot = U.hh_slot[e];
    if (slot == kNoSlot16 || !md) continue;
    const Rates r = hh_rates(Vs[slot * kG + c]);
    double inf = r.am / (r.am + r.bm);
    U.gm[e] = inf + (U.gm[e] - inf) * exp(-delta * (r.am + r.bm));
    inf = r.ah / (r.ah + r.bh);
    U.gh[e] = inf + (U.gh[e] - inf) * exp(-delta * (r.ah + r.bh));
    inf = r.an / (r.an + r.bn);
    U.gn[e] = inf + (U.gn[e] - inf) * exp(-delta * (r.an + r.bn));
  }
  if (md) {
    for (uint32_t e = tid; e < nE_syn; e += kT) {
      if (U.syn_slot[e] == kNoSlot16) continue;
      double decay;
      if (md == 1u) decay = M.syn_uniform ? M.syn_decay_u : U.syn_decay[e];
      else decay = exp(-delta / (M.syn_uniform ? M.syn_tau_u : U.syn_tau[e]));
      U.gg[e] *= decay;
    }
  }
  if (tid < kG && md) {
    const double vd = Vs[(uint32_t)U.det_slot[tid] * kG + tid], vp = cs.vprev[tid];
    if ((uint32_t)tid < U.n_cell) {
      if (cs.armed[tid] && vp < M.theta && M.theta <= vd) {
        const double ts = cs.tcur[tid] + cs.delta[tid] * (M.theta - vp) / (vd - vp);
        const unsigned long long pos = atomicAdd(&M.counters[CNT_SPIKES], 1ull);
        if ((int64_t)pos < M.spike_cap) { M.spike_cell[pos] = M.cell_orig[U.cell_base + tid]; M.spike_t[pos] = ts; }
        else atomicOr(&M.counters[CNT_ERROR], 1ull);
        cs.armed[tid] = 0; cs.dirty[tid] = 1;
      }
      if (vd < M.theta && !cs.armed[tid]) { cs.armed[tid] = 1; cs.dirty[tid] = 1; }
    }
    cs.tcur[tid] = cs.tnext[tid];
  }
  __syncthreads();
}

// ------------------------------------------------------------------------------------------
// The cable step for cell groups.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kGroupThreads) cable_group_kernel(DevModel M, StepArgs A) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ double rt0[kG];             // time of each cell's next undelivered event
  __shared__ uint32_t flags[2];
  const GroupSmemPlan P = M.gplan;
  double* Vs = (double*)smem;
  double* buf = (double*)(smem + P.off_buf);
  const CellS cs = carve_cells(smem + P.off_cell, kG);
  uint64_t* mbar = (uint64_t*)(smem + P.off_mbar);
  const int tid = threadIdx.x, c = tid % kG;
  double* fgen = M.gscratch + (int64_t)blockIdx.x * M.gscratch_stride;
  double* invdgen = fgen + (size_t)P.slot_cap * kG;
  if (tid == 0) { mbar_init(mbar, 1); fence_mbar_init(); }
  __syncthreads();
  unsigned n_sub = 0, n_del = 0;
  uint32_t it = 0;
  for (int64_t g = blockIdx.x; g < M.n_groups; g += gridDim.x, ++it) {
    const GroupDesc D = M.groups[g];
    GView U;
    make_gview(U, M, D);
    const uint32_t vbytes = D.n_cv * kG * 8u;
    if (tid == 0) {
      fence_proxy_async();
      mbar_expect_tx(mbar, vbytes);
      bulk_g2s(Vs, U.gV, vbytes, mbar);
      const int64_t gn = g + gridDim.x;
      if (gn < M.n_groups) {             // next group's records -> L2 while this one is integrated
        const GroupDesc Dn = M.groups[gn];
        const uint32_t nb = Dn.n_cv * kG * 8u;
        const GConstOff con = gconst_offsets(Dn.n_cv, Dn.n_hh_rows, Dn.n_syn_rows, Dn.n_cl_rows, M.syn_uniform != 0);
        bulk_prefetch_l2(M.fast + Dn.const_off, con.hh_gna);
        bulk_prefetch_l2(M.state + Dn.state_base, nb);
      }
    }
    if (tid < kG) {
      const double* rt = U.grt + kRtDoubles * tid;
      const unsigned long long pk = (unsigned long long)__double_as_longlong(rt[1]);
      rt0[tid] = rt[0];
      cs.evcur[tid] = (uint32_t)pk; cs.evend[tid] = (uint32_t)(pk >> 32);
      cs.armed[tid] = rt[2] != 0.0 ? 1u : 0u;
      cs.dirty[tid] = 0;
    }
    mbar_wait(mbar, it & 1u);
    __syncthreads();

    for (int64_t k = A.k_first; k < A.k_first + A.nk; ++k) {
      const double ta = (k == 0) ? A.t0 : __dadd_rn(A.t0, __dmul_rn((double)k, A.dt));
      const double tb = (k + 1 == A.nsteps) ? A.t_end : __dadd_rn(A.t0, __dmul_rn((double)(k + 1), A.dt));
      const bool nominal = (k + 1 < A.nsteps) || A.last_full;
      if (tid < kG) cs.tcur[tid] = ta;
      for (;;) {
        // ---- A: deliver the events due now, choose each cell's (sub-)step (R9)
        if (tid < 32) {
          bool active = false, gen = false;
          if (tid < kG) {
            const double t = cs.tcur[tid];
            uint32_t md = 0;
            if (t < tb) {
              double tn = rt0[tid];
              if (tn <= t) {
                uint32_t cur = cs.evcur[tid];
                const uint32_t end = cs.evend[tid];
                while (cur < end && M.ev_t[cur] <= t) { M.state[M.ev_gidx[cur]] += M.ev_w[cur]; ++cur; ++n_del; }
                tn = cur < end ? M.ev_t[cur] : CUDART_INF;
                cs.evcur[tid] = cur; rt0[tid] = tn; cs.dirty[tid] = 1;
              }
              const double next = tn < tb ? tn : tb;
              const bool fast = nominal && t == ta && next == tb;
              cs.delta[tid] = fast ? A.dt : next - t;
              md = fast ? 1u : 2u;
              cs.tnext[tid] = next;
              cs.vprev[tid] = Vs[(uint32_t)U.det_slot[tid] * kG + tid];
              active = true;
              if ((uint32_t)tid < U.n_cell) ++n_sub;
            }
            cs.mode[tid] = md;
            gen = md == 2u;
          }
          const unsigned ba = __ballot_sync(kFull, active), bg = __ballot_sync(kFull, gen);
          if (tid == 0) { flags[0] = ba; flags[1] = bg; }
        }
        __syncthreads();                  // also orders the delivered g += w before phase B
        if (!flags[0]) break;
        const bool any_gen = flags[1] != 0;
        const uint32_t md = cs.mode[c];
        const double delta = cs.delta[c];
        group_substep(M, U, Vs, buf, cs, fgen, invdgen, any_gen, md, delta);
      }
      __syncthreads();                    // flags are rewritten by the next grid step
    }

    // ---- V' -> HBM (one bulk store), per-cell runtime
    fence_proxy_async();
    __syncthreads();
    if (tid == 0) { bulk_s2g(U.gV, Vs, vbytes); bulk_commit(); }
    if (tid < kG && cs.dirty[tid]) {
      double* rt = U.grt + kRtDoubles * tid;
      const unsigned long long pk = ((unsigned long long)cs.evend[tid] << 32) | cs.evcur[tid];
      rt[0] = rt0[tid];
      rt[1] = __longlong_as_double((long long)pk);
      rt[2] = cs.armed[tid] ? 1.0 : 0.0;
    }
    if (tid == 0) bulk_wait_read0();
    __syncthreads();                      // Vs may be overwritten by the next group's copy
  }
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
  GView U;
  make_gview(U, M, D);
  const int tid = threadIdx.x, c = tid % kG, h = tid / kG;
  double* f = const_cast<double*>(U.f);
  double* invd = const_cast<double*>(U.invd);
  for (uint32_t st = 0; st < U.n_stage; ++st) {
    const uint32_t beg = U.sched[st * kGroupSlots + h], end = U.sched[st * kGroupSlots + h + 1];
    for (uint32_t q = beg; q < end; ++q) {
      const uint32_t si = U.order[q];
      eliminate_seg(U, load_seg(U.segs + si), si, c, dt, f, invd, dcon);
    }
    __syncthreads();
  }
  double* a = const_cast<double*>(U.a);
  double* b = const_cast<double*>(U.b);
  for (uint32_t e = tid; e < U.n_cv * kG; e += kT) {
    a[e] = U.C[e] / dt - U.G[e];
    b[e] = U.bg[e];
  }
  if (!M.syn_uniform) {
    double* decay = const_cast<double*>(U.syn_decay);
    for (uint32_t e = tid; e < U.n_syn * kG; e += kT) decay[e] = exp(-dt / U.syn_tau[e]);
  }
}

// R4: gates start at their steady state for the initial voltage.
__global__ void __launch_bounds__(kGroupThreads) group_init_kernel(DevModel M) {
  const GroupDesc D = M.groups[blockIdx.x];
  GView U;
  make_gview(U, M, D);
  const int c = threadIdx.x % kG;
  for (uint32_t e = threadIdx.x; e < U.n_hh * kG; e += kT) {
    const uint32_t slot = U.hh_slot[e];
    if (slot == kNoSlot16) continue;
    const Rates r = hh_rates(U.gV[slot * kG + c]);
    U.gm[e] = r.am / (r.am + r.bm);
    U.gh[e] = r.ah / (r.ah + r.bh);
    U.gn[e] = r.an / (r.an + r.bn);
  }
}

}  // namespace

int group_ctas_per_sm(uint32_t smem_bytes) {
  const int by_smem = (int)((228u * 1024u) / (smem_bytes + 1024u + 64u));
  const int by_threads = 2048 / kGroupThreads;
  return by_smem < 1 ? 0 : (by_smem < by_threads ? by_smem : by_threads);
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
  const int smem = (int)M.gplan.bytes;
  static int configured = -1;
  if (smem > 48 * 1024 && configured < smem) {
    cudaError_t e = cudaFuncSetAttribute(cable_group_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  cable_group_kernel<<<(unsigned)grid, kGroupThreads, smem, s>>>(M, A);
  if (launches) ++*launches;
  return cudaGetLastError();
}

}  // namespace arbb
