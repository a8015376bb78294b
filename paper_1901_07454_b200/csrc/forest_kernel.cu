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

constexpr int kT = kForestThreads;         // threads of the factor / init kernels (the cable kernel has 32 kW, a template parameter)

// Pointers of one forest.  V, gates, g, runtime, con, xI address shared memory in the cable kernel
// (global memory in the factor / init kernels); everything else is global.
struct FView {
  uint32_t n_slot, n_branch, n_chunk, n_level, n_cell, n_hh, n_syn, n_clamp, flags;
  int n_warp;                       // warps the forest's runs are dealt to (forest_layout.h): kForestWarps or kForestWarpsBig
  const double *f, *invd, *a, *b, *hh_gna, *hh_gk, *hh_gl, *syn_e, *syn_decay, *cl_t0, *cl_t1, *cl_amp;
  const uint32_t *hh_slot, *syn_slot, *cl_slot;
  const uint16_t *hh_cell, *syn_cell, *cl_cell;
  double *V, *m, *h, *n, *g, *rt;
  uint32_t g_gidx0;                 // state-pool index of g[0]
  // tree record: shared memory in the cable kernel
  const FRun* runs; const FChunk* chunks; const unsigned long long* chunk_cells; const FBranch* br; const uint16_t* br_cell;
  const uint32_t *child, *cell_det, *level_br;
  const unsigned long long* masks;  // [0] cells that take part in the (sub-)step in progress, [1] cells on a step of their own length
  const double *C, *S, *sig, *G, *bg, *syn_tau;
  double *con, *xI;                 // per branch: what its parent loses; per point-mechanism instance: its current
  double *fgen, *invdgen, *dcon;    // global scratch of the forest (event-split sub-steps, factorisation)
  int64_t cell_base;
};

// tp: the forest's tree record (shared memory in the cable kernel); it starts with the host's offset table
__device__ __forceinline__ void make_fview(FView& U, const DevModel& M, const UnitHeader& H, uint8_t* fast, double* statew, const uint8_t* tp) {
  U.n_slot = H.n_slot; U.n_branch = H.n_lane; U.n_chunk = H.n_task; U.n_level = H.n_level;
  U.n_cell = H.n_cell; U.n_hh = H.n_hh; U.n_syn = H.n_syn; U.n_clamp = H.n_clamp; U.flags = H.flags;
  U.n_warp = (int)H.pad[2];
  const FOffs& o = *(const FOffs*)tp;
  U.f = (const double*)(fast + o.fast[0]); U.invd = (const double*)(fast + o.fast[1]);
  U.a = (const double*)(fast + o.fast[2]); U.b = (const double*)(fast + o.fast[3]);
  U.hh_gna = (const double*)(fast + o.fast[4]); U.hh_gk = (const double*)(fast + o.fast[5]); U.hh_gl = (const double*)(fast + o.fast[6]);
  U.syn_e = (const double*)(fast + o.fast[7]); U.syn_decay = (const double*)(fast + o.fast[8]);
  U.cl_t0 = (const double*)(fast + o.fast[9]); U.cl_t1 = (const double*)(fast + o.fast[10]); U.cl_amp = (const double*)(fast + o.fast[11]);
  U.hh_slot = (const uint32_t*)(fast + o.fast[12]); U.syn_slot = (const uint32_t*)(fast + o.fast[13]); U.cl_slot = (const uint32_t*)(fast + o.fast[14]);
  U.hh_cell = (const uint16_t*)(fast + o.fast[15]); U.syn_cell = (const uint16_t*)(fast + o.fast[16]); U.cl_cell = (const uint16_t*)(fast + o.fast[17]);
  U.V = statew + o.state[0]; U.m = statew + o.state[1]; U.h = statew + o.state[2]; U.n = statew + o.state[3];
  U.g = statew + o.state[4]; U.rt = statew + o.state[5];
  U.g_gidx0 = (uint32_t)(H.state_base + o.state[4]);
  U.runs = (const FRun*)(tp + o.topo[0]); U.chunks = (const FChunk*)(tp + o.topo[1]);
  U.chunk_cells = (const unsigned long long*)(tp + o.topo[2]); U.br = (const FBranch*)(tp + o.topo[3]);
  U.br_cell = (const uint16_t*)(tp + o.topo[4]); U.child = (const uint32_t*)(tp + o.topo[5]);
  U.cell_det = (const uint32_t*)(tp + o.topo[6]); U.level_br = (const uint32_t*)(tp + o.topo[7]);
  U.masks = nullptr;
  const double* gen = M.gen + H.gen_base;
  U.C = gen + o.gen[0]; U.S = gen + o.gen[1]; U.sig = gen + o.gen[2]; U.G = gen + o.gen[3]; U.bg = gen + o.gen[4]; U.syn_tau = gen + o.gen[5];
  double* scr = M.scratch + H.scratch_base;
  U.fgen = scr + o.scratch[0]; U.invdgen = scr + o.scratch[1]; U.dcon = scr + o.scratch[2];
  U.cell_base = H.cell_base;
}

__device__ __forceinline__ FChunk load_chunk(const FChunk* p) {
  const uint4 q = *(const uint4*)p;
  FChunk c;
  c.slot0 = q.x; c.heads = q.y; c.tails = q.z; c.br_n = q.w;
  return c;
}
__device__ __forceinline__ FBranch load_branch(const FBranch* p) {
  const uint4 q = *(const uint4*)p;
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
// Elimination of the diagonal for one step length as a segmented scan.
// With x_k = d_k - sigma_k (the conductance the subtree below the link k -> parent(k) presents to it),
//   d_k = C_k/delta + sigma_k + sum_children (sigma_c - sigma_c^2 / d_c)   becomes
//   x_k = c_k + sum_children sigma_c x_c / (x_c + sigma_c),   c_k = C_k/delta:
// capacitive conductance in parallel with (link conductance in series with the child's subtree).  Along a
// branch x_k = T_k(x_{k+1}) with the Moebius map T_k(x) = ((c_k + s) x + c_k s) / (x + s), s = sigma_{k+1};
// Moebius maps compose as 2 x 2 matrices, here with POSITIVE entries only, so the scan adds and multiplies
// positive numbers and loses no digits to cancellation (the elimination written with d_k subtracts nearly
// equal numbers when sigma >> C/delta).  f_k = -sigma_k / d_k, and a branch's parent receives
// dcon = sigma_0 x_0 / d_0.  Used once per dt for every cell (kSel false) and, on event-split sub-steps
// (reading R9), for the cells that take a step of their own length (kSel true: mode 2 only).
// ------------------------------------------------------------------------------------------
struct Mob { double a, b, c, d; };   // x -> (a x + b) / (c x + d)

// Between tree levels: when every cell of the forest is swept by one warp (UNIT_WARP_CELLS) a level only depends
// on what the same warp wrote, else on the whole CTA.
__device__ __forceinline__ void level_sync(bool warp_cells) {
  if (warp_cells) __syncwarp(); else __syncthreads();
}

// keeps the entries of a product in range: scale by the power of two that brings the largest near 1 (exact)
__device__ __forceinline__ void mob_normalise(Mob& m) {
  const double big = fmax(fmax(m.a, m.b), fmax(m.c, m.d));
  const int e = ((__double2hiint(big) >> 20) & 0x7FF);          // biased exponent; 0 only for 0 / denormals
  const double sc = __hiloint2double((2046 - (e ? e : 1023)) << 20, 0);
  m.a *= sc; m.b *= sc; m.c *= sc; m.d *= sc;
}

// kSel: 0 = once per dt, every cell, c_k = C_k/dt; 1 = event-split sub-steps: the cells in mode 2, c_k = C_k/delta;
// 2 = conductance-linearised step (ARB_OPT_LINEARISED): every active cell, c_k read from invdout[], where
// forest_substep has assembled C_k/delta + G_k + sum of the point mechanisms' conductances.
template <int kSel>
__device__ __forceinline__ void eliminate_chunk(const FView& U, const CellS* cs, double dt, const FChunk& ck, int lane,
                                                double* fout, double* invdout, double& cb, double& cd, double& csig) {
  // cb / cd: x of the first control volume of the chunk swept before this one (where a branch may continue), csig its sigma
  const int n = (int)(ck.br_n & 63u);
  const bool valid = lane < n;
  const uint32_t s = ck.slot0 + lane;
  const bool head = (ck.heads >> lane) & 1u, tail = (ck.tails >> lane) & 1u;
  const uint32_t br = branch_of(ck, lane);
  bool on = valid;
  double delta = dt;
  if (kSel) {
    if (valid) {
      const uint32_t c = U.br_cell[br];
      on = kSel == 1 ? cs->mode[c] == 2u : cs->mode[c] != 0u;
      delta = cs->delta[c];
    }
  }
  double c = 1.0, sg = 0.0;
  if (valid) { c = kSel == 2 ? invdout[s] : U.C[s] / delta; sg = U.sig[s]; }
  const double snext = __shfl_down_sync(kFull, sg, 1);
  Mob m;
  if (!valid || tail) {
    double x = c;
    if (valid && on) {                     // (a cell that sits this pass out has no fresh contributions: what the array holds
      const FBranch B = load_branch(U.br + br);      //  for it may be anything, and 0 x NaN would reach its neighbours in the scan)
      const uint32_t nc = B.ccnt & 0x7FFFu;
      if (B.ccnt & kFBranchInlineFlag) { if (nc >= 1) x += U.dcon[B.cbeg & 0xFFFFu]; if (nc == 2) x += U.dcon[B.cbeg >> 16]; }
      else for (uint32_t j = 0; j < nc; ++j) x += U.dcon[U.child[B.cbeg + j]];
    }
    m.a = 0.0; m.b = x; m.c = 0.0; m.d = 1.0;                     // constant map: the chain ends here
  } else if (lane == n - 1) {
    // the branch continues in the chunk swept before: T(cb / cd) with T(x) = ((c + s) x + c s) / (x + s), s = csig - no division
    m.a = 0.0; m.b = fma(c + csig, cb, c * csig * cd); m.c = 0.0; m.d = fma(csig, cd, cb);
  } else {
    m.a = c + snext; m.b = c * snext; m.c = 1.0; m.d = snext;
  }
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    Mob r;
    r.a = __shfl_down_sync(kFull, m.a, d); r.b = __shfl_down_sync(kFull, m.b, d);
    r.c = __shfl_down_sync(kFull, m.c, d); r.d = __shfl_down_sync(kFull, m.d, d);
    if (lane + d < 32) {
      Mob p;
      p.a = fma(m.a, r.a, m.b * r.c); p.b = fma(m.a, r.b, m.b * r.d);
      p.c = fma(m.c, r.a, m.d * r.c); p.d = fma(m.c, r.b, m.d * r.d);
      m = p;
      if (d == 2 || d == 8) mob_normalise(m);     // (two doublings from entries <= 1 stay far from overflow)
    }
  }
  // x = b / d, d_k = x + sigma: one reciprocal gives 1/d_k = d / (b + sigma d) and what the parent loses, sigma x / d_k
  const double r = 1.0 / fma(sg, m.d, m.b);
  const double invd = m.d * r;
  if (on) {
    fout[s] = -sg * invd;
    invdout[s] = invd;
    if (head) U.dcon[br] = sg * m.b * r;
  }
  cb = __shfl_sync(kFull, m.b, 0);
  cd = __shfl_sync(kFull, m.d, 0);
  csig = __shfl_sync(kFull, sg, 0);
}

template <int kSel>
__device__ __forceinline__ void eliminate_forest(const FView& U, const CellS* cs, double dt, double* fout, double* invdout) {
  // the forest's runs of a level over the warps of the block: one each in the cable kernel, one or two in the factor kernel
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warps = (int)(blockDim.x >> 5);
  for (int lvl = (int)U.n_level - 1; lvl >= 0; --lvl) {
    for (int w = warp; w < U.n_warp; w += n_warps) {
      const FRun R = U.runs[lvl * U.n_warp + w];
      double cb = 1.0, cd = 1.0, csig = 0.0;
      const unsigned long long want = kSel == 1 ? U.masks[1] : (kSel == 2 ? U.masks[0] : ~0ull);
      for (uint32_t ci = R.chunk_end; ci-- > R.chunk_beg;) {
        if (kSel && !(U.chunk_cells[ci] & want)) continue;     // no cell of this chunk takes a step of its own length
        eliminate_chunk<kSel>(U, cs, dt, load_chunk(U.chunks + ci), lane, fout, invdout, cb, cd, csig);
      }
    }
    level_sync((U.flags & UNIT_WARP_CELLS) != 0);
  }
  __syncthreads();
}

// ------------------------------------------------------------------------------------------
// Backward (leaves -> root) sweep of one chunk on the rhs held in V:
//   r_k = rhs_k - f_{k+1} r_{k+1} along a branch (suffix scan of affine maps), the last control volume
//   of a branch first loses con[child] = f_0 r_0 of every child branch; every control volume is left
//   holding r_k / d_k, which is what the forward sweep needs.
// cf, cr: f and r of the slot that follows the chunk (the previous chunk of the run), for a branch that
// continues there.
// ------------------------------------------------------------------------------------------
// lookup (warp-uniform): some cell of the chunk is not on a plain step: each lane asks for its cell's mode
// (0 inactive: left alone; 2: a step of its own length, factors from the forest's scratch record).
__device__ __forceinline__ void backward_chunk(const FView& U, const CellS& cs, const FChunk& ck, double f, double invd, int lane,
                                               bool lookup, bool lin, double& cf, double& cr) {
  const int n = (int)(ck.br_n & 63u);
  const bool valid = lane < n;
  const uint32_t s = ck.slot0 + lane;
  const bool head = (ck.heads >> lane) & 1u, tail = (ck.tails >> lane) & 1u;
  const uint32_t br = branch_of(ck, lane);
  uint32_t md = 1u;
  double r = 0.0;
  if (valid) {
    if (lookup) {
      md = cs.mode[U.br_cell[br]];
      if (md == 2u && !lin) { f = U.fgen[s]; invd = U.invdgen[s]; }
    }
    r = U.V[s];
    if (tail) {
      const FBranch B = load_branch(U.br + br);
      const uint32_t nc = B.ccnt & 0x7FFFu;
      if (B.ccnt & kFBranchInlineFlag) { if (nc >= 1) r -= U.con[B.cbeg & 0xFFFFu]; if (nc == 2) r -= U.con[B.cbeg >> 16]; }
      else for (uint32_t j = 0; j < nc; ++j) r -= U.con[U.child[B.cbeg + j]];
    }
  }
  const double fnext = __shfl_down_sync(kFull, f, 1);
  double a = 0.0;                              // multiplier of r_{k+1} in r_k; 0 cuts the chain
  if (valid && !tail) {
    if (lane == n - 1) r = fma(-cf, cr, r);    // the branch continues in the chunk swept before this one
    else a = -fnext;
  }
  // (a lane whose partner lies beyond the warp receives its own values; its multiplier is already 0 there,
  // because the window it has folded holds the chunk's last lane, whose multiplier is 0)
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const double a2 = __shfl_down_sync(kFull, a, d);
    const double r2 = __shfl_down_sync(kFull, r, d);
    r = fma(a, r2, r);
    a *= a2;
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
__device__ __forceinline__ void forward_chunk(const FView& U, const CellS& cs, const FChunk& ck, double f, int lane, bool lookup, bool lin, double& cv) {
  const int n = (int)(ck.br_n & 63u);
  const bool valid = lane < n;
  const uint32_t s = ck.slot0 + lane;
  const bool head = (ck.heads >> lane) & 1u;
  const uint32_t br = branch_of(ck, lane);
  uint32_t md = 1u;
  double a = 0.0, b = 0.0;
  if (valid) {
    if (lookup) {
      md = cs.mode[U.br_cell[br]];
      if (md == 2u && !lin) f = U.fgen[s];
    }
    const double q = U.V[s];
    if (head) {
      const uint32_t ps = U.br[br].pslot;
      b = ps != kNoSlot ? fma(-f, U.V[ps], q) : q;
    } else if (lane == 0) {
      b = fma(-f, cv, q);
    } else {
      a = -f; b = q;
    }
  }
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {            // (lanes below d receive their own values; their multiplier is 0 by then)
    const double a2 = __shfl_up_sync(kFull, a, d);
    const double b2 = __shfl_up_sync(kFull, b, d);
    b = fma(a, b2, b);
    a *= a2;
  }
  if (valid && md) U.V[s] = b;
  cv = __shfl_sync(kFull, b, n - 1);
}

// HH gate update x <- x_inf(V') + (x - x_inf) exp(-delta (alpha + beta)) (reading R5).  Not inlined:
// the exp / expm1 chains are several hundred instructions and the kernel has two call sites.  The six quotients of
// the rates and steady states (two x / expm1(x), 1 / (1 + exp), three alpha / (alpha + beta)) share ONE division: the
// reciprocal of their denominators' product, multiplied back (the kernel is bound by instruction issue, and a double
// division is ~40 instructions); results differ from the quotient-by-quotient form in the last bits only.
// one copy each of exp and expm1: the kernel's speed depends on its code staying in the instruction cache (a variant
// 20 KB larger ran 19 % slower), and inlined they are ~45 instructions per call site
__device__ __noinline__ double exp_once(double x) { return exp(x); }
__device__ __noinline__ double expm1_once(double x) { return expm1(x); }
struct Gates { double m, h, n; };
__device__ __noinline__ Gates hh_gates(double v, double delta, double m, double h, double n) {
  const double xm = -(v + 40.0) / 10.0, xn = -(v + 55.0) / 10.0;
  const double em = xm == 0.0 ? 1.0 : expm1_once(xm), en = xn == 0.0 ? 1.0 : expm1_once(xn);       // (x = 0: x / expm1(x) -> 1)
  const double eh = 1.0 + exp_once(-(v + 35.0) / 10.0);
  const double bm = 4.0 * exp_once(-(v + 65.0) / 18.0), ah = 0.07 * exp_once(-(v + 65.0) / 20.0), bn = 0.125 * exp_once(-(v + 65.0) / 80.0);
  // 1 / em, 1 / en, 1 / eh from one reciprocal
  const double p2 = em * en, inv3 = 1.0 / (p2 * eh);
  const double ieh = p2 * inv3, i2 = eh * inv3, iem = en * i2, ien = em * i2;
  const double am = xm == 0.0 ? 1.0 : xm * iem, an = 0.1 * (xn == 0.0 ? 1.0 : xn * ien), bh = ieh;
  // 1 / (am + bm), 1 / (ah + bh), 1 / (an + bn) from one reciprocal
  const double sm = am + bm, sh = ah + bh, sn = an + bn;
  const double q2 = sm * sh, jnv3 = 1.0 / (q2 * sn);
  const double isn = q2 * jnv3, j2 = sn * jnv3, ism = sh * j2, ish = sm * j2;
  Gates g;
  double inf = am * ism;
  g.m = inf + (m - inf) * exp_once(-delta * sm);
  inf = ah * ish;
  g.h = inf + (h - inf) * exp_once(-delta * sh);
  inf = an * isn;
  g.n = inf + (n - inf) * exp_once(-delta * sn);
  return g;
}

// ------------------------------------------------------------------------------------------
// One (sub-)step of every active cell of the forest, phases B..F (phase A, event delivery and the choice
// of the sub-step, is in run_forest).  kGen (a run-time flag: one copy of the code keeps the kernel inside
// the instruction cache): cells may be inactive (mode 0) or on an event-split sub-step of their own length
// (mode 2).
// ------------------------------------------------------------------------------------------
template <bool kLin, int kW>
__device__ __forceinline__ void forest_substep(const DevModel& M, const FView& U, const CellS& cs, double dt, const bool kGen) {
  constexpr int kT = 32 * kW;              // threads of the CTA (shadows the factor kernels' constant)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool multi = U.n_cell > 1;
  const uint32_t n_hh = U.n_hh, n_syn = U.n_syn, n_cl = U.n_clamp;

  // event-split sub-steps: those cells' matrices are eliminated for their own step length (reading R9)
  constexpr bool lin = kLin;               // the linearised step is a kernel instantiation of its own (code size)
  double* xG = U.xI + (n_hh + n_syn + n_cl);                 // lin: conductances beside the sources
  if (!lin && kGen && U.masks[1] != 0ull) eliminate_forest<1>(U, &cs, dt, U.fgen, U.invdgen);

  // ---- B: currents of HH, synapses and clamps from V(t); the passive current is
  // folded into a, b.  Items on one CV form a run; the first item of a run sums it in index order.
  for (uint32_t i = tid; i < n_hh; i += kT) {
    if (kGen && !cs.mode[multi ? U.hh_cell[i] : 0]) continue;
    const double v = U.V[__ldg(U.hh_slot + i)];
    const double m = U.m[i], h = U.h[i], n = U.n[i];
    if (!lin) {
      U.xI[i] = __ldg(U.hh_gna + i) * m * m * m * h * (v - M.ena) + __ldg(U.hh_gk + i) * n * n * n * n * (v - M.ek) + __ldg(U.hh_gl + i) * (v - M.el);
    } else {
      const double gna = __ldg(U.hh_gna + i) * m * m * m * h, gk = __ldg(U.hh_gk + i) * n * n * n * n, gl = __ldg(U.hh_gl + i);
      xG[i] = gna + gk + gl;
      U.xI[i] = gna * M.ena + gk * M.ek + gl * M.el;
    }
  }
  for (uint32_t i = tid; i < n_syn; i += kT) {
    const uint32_t slot = __ldg(U.syn_slot + i);
    if (i > 0 && __ldg(U.syn_slot + i - 1) == slot) continue;
    if (kGen && !cs.mode[multi ? U.syn_cell[i] : 0]) continue;
    const double v = U.V[slot];
    double I = 0.0, G = 0.0;
    uint32_t j = i;
    do {
      const double es = M.syn_uniform ? M.syn_e_u : __ldg(U.syn_e + j);
      if (!lin) I += U.g[j] * (v - es);
      else { G += U.g[j]; I += U.g[j] * es; }
      ++j;
    } while (j < n_syn && __ldg(U.syn_slot + j) == slot);
    U.xI[n_hh + i] = I;
    if (lin) xG[n_hh + i] = G;
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
    U.xI[n_hh + n_syn + i] = lin ? -I : I;                   // lin: sources are ADDED to the rhs
  }
  __syncthreads();

  // ---- C: rhs_i = (C_i/delta - G_i) V_i + G_i e_i - I_i, in place of V
  if (!kGen) {
    const uint32_t n = U.n_slot;
#pragma unroll 4
    for (uint32_t s = tid; s < n; s += kT) U.V[s] = fma(__ldg(U.a + s), U.V[s], __ldg(U.b + s));
  } else {
    const unsigned long long actc = U.masks[0];
    for (uint32_t ci = warp; ci < U.n_chunk; ci += kW) {
      if (!(U.chunk_cells[ci] & actc)) continue;
      const FChunk ck = load_chunk(U.chunks + ci);
      if (lane >= (int)(ck.br_n & 63u)) continue;
      const uint32_t c = U.br_cell[branch_of(ck, lane)], md = cs.mode[c];
      const uint32_t s = ck.slot0 + lane;
      if (md == 1u) U.V[s] = fma(__ldg(U.a + s), U.V[s], __ldg(U.b + s));
      else if (md == 2u) U.V[s] = fma(lin ? U.C[s] / cs.delta[c] : U.C[s] / cs.delta[c] - U.G[s], U.V[s], U.bg[s]);
      // lin: the diagonal without the point mechanisms, C/delta + G (the nominal one sits in the f slot)
      if (lin && md) U.invdgen[s] = md == 1u ? __ldg(U.f + s) : U.C[s] / cs.delta[c] + U.G[s];
    }
  }
  if (lin && !kGen) {
    const uint32_t n = U.n_slot;
    for (uint32_t s = tid; s < n; s += kT) U.invdgen[s] = __ldg(U.f + s);
  }
  __syncthreads();
  // HH, synapse and clamp currents of a cell may meet on a control volume: barriers in between, unless the
  // host found that they never do in this forest
  const bool disjoint = (U.flags & UNIT_POINT_DISJOINT) != 0;
  if (n_hh) {
    for (uint32_t i = tid; i < n_hh; i += kT) {
      if (kGen && !cs.mode[multi ? U.hh_cell[i] : 0]) continue;
      const uint32_t slot = __ldg(U.hh_slot + i);
      if (!lin) U.V[slot] -= U.xI[i];
      else { U.V[slot] += U.xI[i]; U.invdgen[slot] += xG[i]; }
    }
    if (!disjoint) __syncthreads();
  }
  if (n_syn) {
    for (uint32_t i = tid; i < n_syn; i += kT) {
      const uint32_t slot = __ldg(U.syn_slot + i);
      if (i > 0 && __ldg(U.syn_slot + i - 1) == slot) continue;
      if (kGen && !cs.mode[multi ? U.syn_cell[i] : 0]) continue;
      if (!lin) U.V[slot] -= U.xI[n_hh + i];
      else { U.V[slot] += U.xI[n_hh + i]; U.invdgen[slot] += xG[n_hh + i]; }
    }
    if (!disjoint) __syncthreads();
  }
  if (n_cl) {
    for (uint32_t i = tid; i < n_cl; i += kT) {
      const uint32_t slot = U.cl_slot[i];
      if (i > 0 && U.cl_slot[i - 1] == slot) continue;
      if (kGen && !cs.mode[multi ? U.cl_cell[i] : 0]) continue;
      if (!lin) U.V[slot] -= U.xI[n_hh + n_syn + i]; else U.V[slot] += U.xI[n_hh + n_syn + i];
    }
    if (!disjoint) __syncthreads();
  }
  if (disjoint && (n_hh | n_syn | n_cl)) __syncthreads();
  // lin: every active cell's matrix is eliminated afresh (its factors go to the forest's scratch record)
  if (lin) eliminate_forest<2>(U, &cs, dt, U.fgen, U.invdgen);

  // ---- D: backward sweep, deepest level first; E: forward substitution, root first; V <- V'
  // The chunk after the one being swept is fetched first (its record from shared memory, its factors from
  // L2), so that only the scan itself is exposed.  On general passes chunks none of whose cells take part
  // are skipped (a branch that spans two chunks belongs to one cell: both are swept or neither).
  const unsigned long long act = kGen ? U.masks[0] : ~0ull;
  const unsigned long long odd = kGen ? ~(U.masks[0] & ~U.masks[1]) : 0ull;     // cells that are not on a plain step
  const bool warp_cells = (U.flags & UNIT_WARP_CELLS) != 0;
  constexpr uint32_t kNone = 0xFFFFFFFFu;
  for (int lvl = (int)U.n_level - 1; lvl >= 0; --lvl) {
    const FRun R = U.runs[lvl * kW + warp];
    auto next = [&](uint32_t ci) -> uint32_t {
      while (ci > R.chunk_beg) { --ci; if (!kGen || (U.chunk_cells[ci] & act)) return ci; }
      return kNone;
    };
    auto fetch = [&](uint32_t ci, FChunk& k, double& f, double& invd) {
      k = load_chunk(U.chunks + ci);
      f = 0.0; invd = 0.0;
      if (lane < (int)(k.br_n & 63u)) {
        if (!lin) { f = __ldg(U.f + k.slot0 + lane); invd = __ldg(U.invd + k.slot0 + lane); }
        else { f = U.fgen[k.slot0 + lane]; invd = U.invdgen[k.slot0 + lane]; }
      }
    };
    double cf = 0.0, cr = 0.0, f = 0.0, invd = 0.0;
    FChunk ck;
    uint32_t cur = next(R.chunk_end);
    if (cur != kNone) fetch(cur, ck, f, invd);
    // the barrier that ends the level below comes AFTER this level's first loads have been issued (they do not
    // depend on what other warps wrote): their L2 latency overlaps the wait
    if (lvl != (int)U.n_level - 1) level_sync(warp_cells);
    while (cur != kNone) {
      const uint32_t nx = next(cur);
      FChunk nck = ck;
      double nf = 0.0, ni = 0.0;
      if (nx != kNone) fetch(nx, nck, nf, ni);
      backward_chunk(U, cs, ck, f, invd, lane, kGen && (U.chunk_cells[cur] & odd) != 0ull, lin, cf, cr);
      cur = nx; ck = nck; f = nf; invd = ni;
    }
  }
  for (uint32_t lvl = 0; lvl < U.n_level; ++lvl) {
    const FRun R = U.runs[lvl * kW + warp];
    auto next = [&](uint32_t ci) -> uint32_t {          // first chunk at or after ci that is swept
      for (; ci < R.chunk_end; ++ci) if (!kGen || (U.chunk_cells[ci] & act)) return ci;
      return kNone;
    };
    auto fetch = [&](uint32_t ci, FChunk& k, double& f) {
      k = load_chunk(U.chunks + ci);
      f = lane < (int)(k.br_n & 63u) ? (lin ? U.fgen[k.slot0 + lane] : __ldg(U.f + k.slot0 + lane)) : 0.0;
    };
    double cv = 0.0, f = 0.0;
    FChunk ck;
    uint32_t cur = next(R.chunk_beg);
    if (cur != kNone) fetch(cur, ck, f);
    level_sync(warp_cells);                // ends the level above (for the root level: the backward sweep)
    while (cur != kNone) {
      const uint32_t nx = next(cur + 1);
      FChunk nck = ck;
      double nf = 0.0;
      if (nx != kNone) fetch(nx, nck, nf);
      forward_chunk(U, cs, ck, f, lane, kGen && (U.chunk_cells[cur] & odd) != 0ull, lin, cv);
      cur = nx; ck = nck; f = nf;
    }
  }
  __syncthreads();

  // ---- F: state update with V', threshold test
  for (uint32_t i = tid; i < n_hh; i += kT) {
    const uint32_t c = (kGen && multi) ? U.hh_cell[i] : 0;
    if (kGen && !cs.mode[c]) continue;
    const double delta = kGen ? cs.delta[c] : dt;
    const Gates g = hh_gates(U.V[__ldg(U.hh_slot + i)], delta, U.m[i], U.h[i], U.n[i]);
    U.m[i] = g.m; U.h[i] = g.h; U.n[i] = g.n;
  }
  for (uint32_t i = tid; i < n_syn; i += kT) {
    const uint32_t c = (kGen && multi) ? U.syn_cell[i] : 0;
    const uint32_t md = kGen ? cs.mode[c] : 1u;
    if (!md) continue;
    double decay;
    if (md == 1u) decay = M.syn_uniform ? M.syn_decay_u : __ldg(U.syn_decay + i);
    else decay = exp_once(-cs.delta[c] / (M.syn_uniform ? M.syn_tau_u : U.syn_tau[i]));
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
template <bool kLin, int kW>
__device__ __forceinline__ void run_forest(const DevModel& M, const StepArgs& A, const FView& U, const CellS& cs,
                                           unsigned& n_sub, unsigned& n_del) {
  uint32_t* sMaskW = (uint32_t*)U.masks;     // the two 64-bit masks as four words (little endian)
  const int tid = threadIdx.x;
  const uint32_t n_cell = U.n_cell;
  bool gen_in_l2 = false;
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
      uint32_t md = 0;
      if ((uint32_t)tid < n_cell) {
        const double t = cs.tcur[tid];
        if (t < tb) {
          double tn = U.rt[kRtDoubles * tid];
          if (tn <= t) {
            uint32_t cur = cs.evcur[tid];
            const uint32_t end = cs.evend[tid];
            while (cur < end && M.ev_t[cur] <= t) { U.g[event_target(M, M.ev_gidx[cur], t, M.ev_w[cur]) - U.g_gidx0] += M.ev_w[cur]; ++cur; ++n_del; }
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
      if (tid < (int)kForestMaxCells) {       // warps 0 and 1: which cells take part, which take a step of their own length
        const unsigned on = __ballot_sync(kFull, md != 0u), own = __ballot_sync(kFull, md == 2u);
        if ((tid & 31) == 0) { sMaskW[tid >> 5] = on; sMaskW[2 + (tid >> 5)] = own; }
      }
      const int any_active = __syncthreads_or(active);
      if (!any_active) break;
      const int general = __syncthreads_or(!plain);
      if (general && !gen_in_l2) {             // the dt-independent arrays (C, S, sigma, G, G e) of the re-elimination: cold in HBM until now
        if (tid == 0) bulk_prefetch_l2(U.C, 8u * 5u * U.n_slot);
        gen_in_l2 = true;
      }
      forest_substep<kLin, kW>(M, U, cs, A.dt, general != 0);
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
template <bool kLin, int kW>
__global__ void __launch_bounds__(32 * kW, 32 / kW) cable_forest_kernel(DevModel M, StepArgs A, int cls) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ UnitHeader H;
  __shared__ __align__(8) uint64_t mbar_mem;
  __shared__ unsigned long long sMask[2];
  const UnitDesc d = M.units[M.fcls[cls].first + blockIdx.x];
  uint8_t* fast = M.fast + d.fast_off;
  double* Ss = (double*)smem;
  uint64_t* mbar = &mbar_mem;
  const int tid = threadIdx.x;
  if (tid == 0) {
    mbar_init(mbar, 1);
    fence_mbar_init();
    fence_proxy_async();
    mbar_expect_tx(mbar, d.state_bytes + d.topo_bytes);
    bulk_g2s(Ss, M.state + d.state_base, d.state_bytes, mbar);
    bulk_g2s(smem + align_up(d.state_bytes, 128), M.topo + 16ull * d.topo_off16, d.topo_bytes, mbar);   // the tree record
    bulk_prefetch_l2(fast, d.fast_bytes);            // coefficients and instance tables -> L2
  }
  if (tid < (int)(sizeof(UnitHeader) / 4)) ((uint32_t*)&H)[tid] = __ldg((const uint32_t*)fast + tid);
  __syncthreads();
  // every forest lays its own shared memory out; the launch reserves what the largest of its class needs
  ForestCaps fc;
  fc.state_bytes = d.state_bytes; fc.topo_bytes = d.topo_bytes; fc.n_branch = H.n_lane; fc.n_spec = H.n_hh + H.n_syn + H.n_clamp; fc.n_cell = H.n_cell;
  const ForestSmemPlan P = forest_smem_plan(fc);
  mbar_wait(mbar, 0);                        // state and tree records are in shared memory
  FView U;
  make_fview(U, M, H, fast, Ss, smem + P.off_topo);
  U.masks = sMask;
  U.con = (double*)(smem + P.off_con);
  U.dcon = U.con;                            // re-eliminations hand a branch's share to its parent through shared memory too (the
                                             // sweeps, which use the same array, come after them)
  U.xI = (double*)(smem + P.off_xi);
  const CellS cs = carve_cells(smem + P.off_cell, U.n_cell);
  unsigned n_sub = 0, n_del = 0;
  run_forest<kLin, kW>(M, A, U, cs, n_sub, n_del);
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
  make_fview(U, M, H, fast, M.state + d.state_base, M.topo + H.topo_off);
  double* a = const_cast<double*>(U.a);
  double* b = const_cast<double*>(U.b);
  if (!M.linearised) {
    eliminate_forest<0>(U, nullptr, dt, const_cast<double*>(U.f), const_cast<double*>(U.invd));
    for (uint32_t s = threadIdx.x; s < U.n_slot; s += kT) {
      a[s] = U.C[s] / dt - U.G[s];
      b[s] = U.bg[s];
    }
  } else {
    // conductance-linearised step: rhs = (C/dt) V + G e + ..., and the part of the diagonal that does not change
    // from step to step, C/dt + G, in the f slot (the elimination works with x_k = d_k - sigma_k and needs sigma)
    double* f = const_cast<double*>(U.f);
    double* invd = const_cast<double*>(U.invd);
    for (uint32_t s = threadIdx.x; s < U.n_slot; s += kT) {
      const double cdt = U.C[s] / dt;
      a[s] = cdt;
      b[s] = U.bg[s];
      f[s] = cdt + U.G[s];
      invd[s] = U.sig[s];
    }
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
  make_fview(U, M, H, fast, M.state + d.state_base, M.topo + H.topo_off);
  for (uint32_t i = threadIdx.x; i < U.n_hh; i += kT) {
    const Rates r = hh_rates(U.V[U.hh_slot[i]]);
    U.m[i] = r.am / (r.am + r.bm);
    U.h[i] = r.ah / (r.ah + r.bh);
    U.n[i] = r.an / (r.an + r.bn);
  }
}

}  // namespace

cudaError_t configure_forest_kernel(int max_optin_bytes) {
  for (const void* k : {(const void*)cable_forest_kernel<false, kForestWarps>, (const void*)cable_forest_kernel<true, kForestWarps>,
                        (const void*)cable_forest_kernel<false, kForestWarpsBig>, (const void*)cable_forest_kernel<true, kForestWarpsBig>}) {
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
  const unsigned n = (unsigned)K.count, b = K.plan.bytes;
  if (K.n_warp == kForestWarps) {
    if (!M.linearised) cable_forest_kernel<false, kForestWarps><<<n, 32 * kForestWarps, b, s>>>(M, A, cls);
    else cable_forest_kernel<true, kForestWarps><<<n, 32 * kForestWarps, b, s>>>(M, A, cls);
  } else {
    if (!M.linearised) cable_forest_kernel<false, kForestWarpsBig><<<n, 32 * kForestWarpsBig, b, s>>>(M, A, cls);
    else cable_forest_kernel<true, kForestWarpsBig><<<n, 32 * kForestWarpsBig, b, s>>>(M, A, cls);
  }
  if (launches) ++*launches;
  return cudaGetLastError();
}

}  // namespace arbb
