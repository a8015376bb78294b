// kernels.cu - hand-written fp64 CUDA kernels for sm_100a: the whole hot path of arbb200.
//
//   cable_kernel        per grid step (or per fused run of steps) and per cell block:
//                       event delivery -> mechanism currents (eq 2a)
//                       -> rhs of the implicit Euler system -> branched Thomas /
//                       Hines sweeps over levels of interleaved branches -> V <- V'
//                       -> gate / synapse state update with V' -> threshold test
//
//   factor_kernel       once per dt: eliminates the (constant, reading R1) matrix of every cell
//   build_events / spikes_to_events   once per min-delay epoch
//
// No tensor cores: nothing here is a dense contraction.  The path is bound by HBM traffic when
// state streams every step and by fp64 issue / dependent-chain latency when a block stays on chip.
#include "kernels.cuh"

namespace arbb {

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kMaxCells = 64;   // == BuildParams::max_cells

// ------------------------------------------------------------------------------------------
// HH rate functions (reading R5): textbook Hodgkin-Huxley 1952, 6.3 C, rest at -65 mV.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ double exprelr(double x) { return x == 0.0 ? 1.0 : x / expm1(x); }

struct Rates { double am, bm, ah, bh, an, bn; };
__device__ __forceinline__ Rates hh_rates(double v) {
  Rates r;
  r.am = exprelr(-(v + 40.0) / 10.0);
  r.bm = 4.0 * exp(-(v + 65.0) / 18.0);
  r.ah = 0.07 * exp(-(v + 65.0) / 20.0);
  r.bh = 1.0 / (1.0 + exp(-(v + 35.0) / 10.0));
  r.an = 0.1 * exprelr(-(v + 55.0) / 10.0);
  r.bn = 0.125 * exp(-(v + 65.0) / 80.0);
  return r;
}

// Pointers of one block, resolved once per CTA.
struct View {
  const Task* tasks; const uint32_t* level_begin;
  const uint32_t* br_pslot; const uint32_t* br_cbeg; const uint16_t* br_len; const uint16_t* br_cell;
  const uint16_t* br_ccnt; const uint32_t* child; const uint32_t* cell_det;
  const uint32_t* hh_slot; const uint16_t* hh_cell; const uint16_t* syn_cell;
  const uint32_t* sp_slot; const int32_t* sp_hh; const uint32_t* sp_syn_beg; const uint32_t* sp_cl_beg;
  const uint16_t* sp_syn_cnt; const uint16_t* sp_cl_cnt; const uint16_t* sp_cell;
  // gen
  const double *C, *S, *sig, *G, *bg;
  // fast
  double *f, *invd, *a, *b;
  const double *hh_gna, *hh_gk, *hh_gl, *syn_e, *syn_tau, *cl_t0, *cl_t1, *cl_amp;
  double* syn_decay;
  // state
  double *V, *m, *h, *n, *g;
  // scratch (global): factors of a non-nominal step, extra currents
  double *fgen, *invdgen;
};

__device__ __forceinline__ View make_view(const DevModel& M, const BlockInfo& bi) {
  View v;
  const uint8_t* meta = M.meta + bi.meta_base;
  MetaOff mo = meta_offsets(bi);
  v.tasks = (const Task*)(meta + mo.tasks);
  v.level_begin = (const uint32_t*)(meta + mo.level_begin);
  v.br_pslot = (const uint32_t*)(meta + mo.br_pslot);
  v.br_cbeg = (const uint32_t*)(meta + mo.br_cbeg);
  v.br_len = (const uint16_t*)(meta + mo.br_len);
  v.br_cell = (const uint16_t*)(meta + mo.br_cell);
  v.br_ccnt = (const uint16_t*)(meta + mo.br_ccnt);
  v.child = (const uint32_t*)(meta + mo.child);
  v.cell_det = (const uint32_t*)(meta + mo.cell_det);
  v.hh_slot = (const uint32_t*)(meta + mo.hh_slot);
  v.hh_cell = (const uint16_t*)(meta + mo.hh_cell);
  v.syn_cell = (const uint16_t*)(meta + mo.syn_cell);
  v.sp_slot = (const uint32_t*)(meta + mo.sp_slot);
  v.sp_hh = (const int32_t*)(meta + mo.sp_hh);
  v.sp_syn_beg = (const uint32_t*)(meta + mo.sp_syn_beg);
  v.sp_cl_beg = (const uint32_t*)(meta + mo.sp_cl_beg);
  v.sp_syn_cnt = (const uint16_t*)(meta + mo.sp_syn_cnt);
  v.sp_cl_cnt = (const uint16_t*)(meta + mo.sp_cl_cnt);
  v.sp_cell = (const uint16_t*)(meta + mo.sp_cell);
  GenOff go = gen_offsets(bi);
  const double* gen = M.gen + bi.gen_base;
  v.C = gen + go.C; v.S = gen + go.S; v.sig = gen + go.sig; v.G = gen + go.G; v.bg = gen + go.b;
  FastOff fo = fast_offsets(bi);
  double* fast = M.fast + bi.fast_base;
  v.f = fast + fo.f; v.invd = fast + fo.invd; v.a = fast + fo.a; v.b = fast + fo.b;
  v.hh_gna = fast + fo.hh_gna; v.hh_gk = fast + fo.hh_gk; v.hh_gl = fast + fo.hh_gl;
  v.syn_e = fast + fo.syn_e; v.syn_decay = fast + fo.syn_decay; v.syn_tau = fast + fo.syn_tau;
  v.cl_t0 = fast + fo.cl_t0; v.cl_t1 = fast + fo.cl_t1; v.cl_amp = fast + fo.cl_amp;
  StateOff so = state_offsets(bi);
  double* st = M.state + bi.state_base;
  v.V = st + so.v; v.m = st + so.m; v.h = st + so.h; v.n = st + so.n; v.g = st + so.g;
  double* sc = M.scratch + bi.scratch_base;
  v.fgen = sc; v.invdgen = sc + bi.n_slot;
  return v;
}

// ------------------------------------------------------------------------------------------
// Backward (leaves -> root) elimination of the diagonal for one step length, used by the
// factorisation and by non-nominal (split) steps.  For a branch (lane) with CVs k = 0..len-1:
//   d_k = C_k/delta + S_k - sum_children sigma_c^2 / d_c ;  f_k = -sigma_k / d_k = u_k / d_k
// Returns through fout/invdout; dcontrib[tl] = f_0 * u_0 is what the parent's terminal CV loses.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void eliminate_branch(const View& W, const Task& T, uint32_t lane, uint32_t tl,
                                                 double delta, double* fout, double* invdout,
                                                 double* dcontrib) {
  const uint32_t len = W.br_len[tl];
  const uint32_t base = T.slot_off + lane;
  uint32_t s = base + (len - 1) * T.width;
  double d = W.C[s] / delta + W.S[s];
  const uint32_t cb = W.br_cbeg[tl], cc = W.br_ccnt[tl];
  for (uint32_t j = 0; j < cc; ++j) d -= dcontrib[W.child[cb + j]];
  for (uint32_t k = len - 1;; --k) {
    double invd = 1.0 / d;
    double sg = W.sig[s];
    double f = -sg * invd;
    fout[s] = f;
    invdout[s] = invd;
    if (k == 0) { dcontrib[tl] = -f * sg; break; }     // f*u with u = -sigma
    s -= T.width;
    d = W.C[s] / delta + W.S[s] + f * sg;                // d_p -= f*u
  }
}

__global__ void __launch_bounds__(kThreads) factor_kernel(DevModel M, double dt) {
  __shared__ BlockInfo bi;
  if (threadIdx.x == 0) bi = M.blocks[blockIdx.x];
  __syncthreads();
  View W = make_view(M, bi);
  double* dcontrib = M.scratch + bi.scratch_base + 2 * (int64_t)bi.n_slot;   // global scratch
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int lvl = (int)bi.n_level - 1; lvl >= 0; --lvl) {
    for (uint32_t ti = W.level_begin[lvl] + warp; ti < W.level_begin[lvl + 1]; ti += kWarps) {
      Task T = W.tasks[ti];
      if ((uint32_t)lane < T.nlanes) eliminate_branch(W, T, lane, T.lane_off + lane, dt, W.f, W.invd, dcontrib);
    }
    __syncthreads();
  }
  for (uint32_t ti = warp; ti < bi.n_task; ti += kWarps) {
    Task T = W.tasks[ti];
    if ((uint32_t)lane < T.nlanes) {
      uint32_t len = W.br_len[T.lane_off + lane];
      for (uint32_t k = 0; k < len; ++k) {
        uint32_t s = T.slot_off + lane + k * T.width;
        W.a[s] = W.C[s] / dt - W.G[s];
        W.b[s] = W.bg[s];
      }
    }
  }
  for (uint32_t i = threadIdx.x; i < bi.n_syn; i += kThreads) W.syn_decay[i] = exp(-dt / W.syn_tau[i]);
}

// R4: gates start at their steady state for the initial voltage; detectors armed.
__global__ void __launch_bounds__(kThreads) init_kernel(DevModel M) {
  __shared__ BlockInfo bi;
  if (threadIdx.x == 0) bi = M.blocks[blockIdx.x];
  __syncthreads();
  View W = make_view(M, bi);
  for (uint32_t i = threadIdx.x; i < bi.n_hh; i += kThreads) {
    Rates r = hh_rates(W.V[W.hh_slot[i]]);
    W.m[i] = r.am / (r.am + r.bm);
    W.h[i] = r.ah / (r.ah + r.bh);
    W.n[i] = r.an / (r.an + r.bn);
  }
  for (uint32_t i = threadIdx.x; i < bi.n_cell; i += kThreads) {
    CellRt rt; rt.ev_cur = 0; rt.ev_end = 0; rt.armed = 1; rt.pad = 0;
    M.cell_rt[bi.cell_base + i] = rt;
  }
}

__global__ void reset_detectors_kernel(DevModel M) {
  int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c < M.n_cells) M.cell_rt[c].armed = 1;
}

// ------------------------------------------------------------------------------------------
// The cable step.  One CTA per cell block; A.nk consecutive grid steps per launch.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) cable_kernel(DevModel M, StepArgs A) {
  extern __shared__ double dyn_smem[];
  __shared__ BlockInfo bi;
  __shared__ double s_tcur[kMaxCells], s_tnext[kMaxCells], s_delta[kMaxCells], s_vprev[kMaxCells];
  __shared__ uint32_t s_evcur[kMaxCells], s_evend[kMaxCells], s_armed[kMaxCells];
  __shared__ uint8_t s_mode[kMaxCells];
  __shared__ unsigned int s_substeps, s_delivered;
  if (threadIdx.x == 0) { bi = M.blocks[blockIdx.x]; s_substeps = 0; s_delivered = 0; }
  __syncthreads();
  const View W = make_view(M, bi);
  const uint32_t lanes_pad = align_up(bi.n_lane, 16);
  double* contrib;
  double* dcontrib;
  if (bi.flags & 1u) {   // too many branches for shared memory: use the block's global scratch
    contrib = M.scratch + bi.scratch_base + 2 * (int64_t)bi.n_slot;
    dcontrib = contrib + lanes_pad;
  } else {
    contrib = dyn_smem;
    dcontrib = dyn_smem + lanes_pad;
  }
  double* const extra = W.fgen;   // extra currents live here between phases B and B2
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t n_cell = bi.n_cell;
  if ((uint32_t)tid < n_cell) {
    CellRt rt = M.cell_rt[bi.cell_base + tid];
    s_evcur[tid] = rt.ev_cur; s_evend[tid] = rt.ev_end; s_armed[tid] = rt.armed;
  }

  for (int64_t k = A.k_first; k < A.k_first + A.nk; ++k) {
    const double ta = (k == 0) ? A.t0 : __dadd_rn(A.t0, __dmul_rn((double)k, A.dt));
    const double tb = (k + 1 == A.nsteps) ? A.t_end : __dadd_rn(A.t0, __dmul_rn((double)(k + 1), A.dt));
    const bool nominal = (k + 1 < A.nsteps) || A.last_full;
    if ((uint32_t)tid < n_cell) s_tcur[tid] = ta;
    __syncthreads();
    for (;;) {
      // ---- phase A: deliver events due now, choose the sub-step (reading R9)
      int active = 0;
      if ((uint32_t)tid < n_cell) {
        const double t = s_tcur[tid];
        if (t < tb) {
          uint32_t cur = s_evcur[tid];
          const uint32_t end = s_evend[tid];
          uint32_t ndel = 0;
          while (cur < end && M.ev_t[cur] <= t) { M.state[M.ev_gidx[cur]] += M.ev_w[cur]; ++cur; ++ndel; }
          s_evcur[tid] = cur;
          double next = tb;
          if (cur < end) { double te = M.ev_t[cur]; if (te < tb) next = te; }
          const bool fast = nominal && t == ta && next == tb;
          s_delta[tid] = fast ? A.dt : next - t;
          s_mode[tid] = fast ? 1 : 2;
          s_tnext[tid] = next;
          s_vprev[tid] = W.V[W.cell_det[tid]];
          active = 1;
          atomicAdd(&s_substeps, 1u);
          if (ndel) atomicAdd(&s_delivered, ndel);
        } else {
          s_mode[tid] = 0;
        }
      }
      if (!__syncthreads_or(active)) break;

      // ---- phase B: currents of HH, synapses and clamps from V(t)
      for (uint32_t sp = tid; sp < bi.n_sp; sp += kThreads) {
        const uint32_t c = W.sp_cell[sp];
        if (!s_mode[c]) continue;
        const double v = W.V[W.sp_slot[sp]];
        double I = 0.0;
        const int32_t hi = W.sp_hh[sp];
        if (hi >= 0) {
          const double m = W.m[hi], h = W.h[hi], n = W.n[hi];
          I += W.hh_gna[hi] * m * m * m * h * (v - M.ena) + W.hh_gk[hi] * n * n * n * n * (v - M.ek) +
               W.hh_gl[hi] * (v - M.el);
        }
        const uint32_t sb = W.sp_syn_beg[sp], sc = W.sp_syn_cnt[sp];
        for (uint32_t j = 0; j < sc; ++j) I += W.g[sb + j] * (v - W.syn_e[sb + j]);
        const uint32_t cb = W.sp_cl_beg[sp], cc = W.sp_cl_cnt[sp];
        const double t = s_tcur[c];
        for (uint32_t j = 0; j < cc; ++j)
          if (W.cl_t0[cb + j] <= t && t < W.cl_t1[cb + j]) I -= W.cl_amp[cb + j];
        extra[sp] = I;
      }
      __syncthreads();
      // ---- phase C: rhs_i = (C_i/delta - G_i) V_i + G_i e_i, in place of V
      for (uint32_t ti = warp; ti < bi.n_task; ti += kWarps) {
        const Task T = W.tasks[ti];
        if ((uint32_t)lane >= T.nlanes) continue;
        const uint32_t tl = T.lane_off + lane;
        const uint32_t c = W.br_cell[tl];
        const uint32_t md = s_mode[c];
        if (!md) continue;
        const uint32_t len = W.br_len[tl];
        uint32_t s = T.slot_off + lane;
        if (md == 1) {
          for (uint32_t q = 0; q < len; ++q, s += T.width) W.V[s] = fma(W.a[s], W.V[s], W.b[s]);
        } else {
          const double delta = s_delta[c];
          for (uint32_t q = 0; q < len; ++q, s += T.width) W.V[s] = fma(W.C[s] / delta - W.G[s], W.V[s], W.bg[s]);
        }
      }
      __syncthreads();
      for (uint32_t sp = tid; sp < bi.n_sp; sp += kThreads)
        if (s_mode[W.sp_cell[sp]]) W.V[W.sp_slot[sp]] -= extra[sp];
      __syncthreads();
      // ---- phase D: backward sweep, deepest level first
      for (int lvl = (int)bi.n_level - 1; lvl >= 0; --lvl) {
        for (uint32_t ti = W.level_begin[lvl] + warp; ti < W.level_begin[lvl + 1]; ti += kWarps) {
          const Task T = W.tasks[ti];
          if ((uint32_t)lane >= T.nlanes) continue;
          const uint32_t tl = T.lane_off + lane;
          const uint32_t c = W.br_cell[tl];
          const uint32_t md = s_mode[c];
          if (!md) continue;
          const uint32_t len = W.br_len[tl];
          const double* fp = W.f;
          if (md == 2) { eliminate_branch(W, T, lane, tl, s_delta[c], W.fgen, W.invdgen, dcontrib); fp = W.fgen; }
          uint32_t s = T.slot_off + lane + (len - 1) * T.width;
          double r = W.V[s];
          const uint32_t cb = W.br_cbeg[tl], cc = W.br_ccnt[tl];
          for (uint32_t j = 0; j < cc; ++j) r -= contrib[W.child[cb + j]];
          W.V[s] = r;
          for (uint32_t q = len - 1; q > 0; --q) {
            const double fq = fp[s];
            s -= T.width;
            r = fma(-fq, r, W.V[s]);
            W.V[s] = r;
          }
          contrib[tl] = fp[s] * r;
        }
        __syncthreads();
      }
      // ---- phase E: forward substitution, root level first; V <- V'
      for (uint32_t lvl = 0; lvl < bi.n_level; ++lvl) {
        for (uint32_t ti = W.level_begin[lvl] + warp; ti < W.level_begin[lvl + 1]; ti += kWarps) {
          const Task T = W.tasks[ti];
          if ((uint32_t)lane >= T.nlanes) continue;
          const uint32_t tl = T.lane_off + lane;
          const uint32_t md = s_mode[W.br_cell[tl]];
          if (!md) continue;
          const uint32_t len = W.br_len[tl];
          const double* fp = md == 1 ? W.f : W.fgen;
          const double* ip = md == 1 ? W.invd : W.invdgen;
          const uint32_t ps = W.br_pslot[tl];
          double vp = ps == kNoSlot ? 0.0 : W.V[ps];
          uint32_t s = T.slot_off + lane;
          for (uint32_t q = 0; q < len; ++q, s += T.width) {
            vp = fma(-fp[s], vp, W.V[s] * ip[s]);
            W.V[s] = vp;
          }
        }
        __syncthreads();
      }
      // ---- phase F: state update with V', threshold test
      for (uint32_t i = tid; i < bi.n_hh; i += kThreads) {
        const uint32_t c = W.hh_cell[i];
        if (!s_mode[c]) continue;
        const double delta = s_delta[c];
        const Rates r = hh_rates(W.V[W.hh_slot[i]]);
        double inf = r.am / (r.am + r.bm);
        W.m[i] = inf + (W.m[i] - inf) * exp(-delta * (r.am + r.bm));
        inf = r.ah / (r.ah + r.bh);
        W.h[i] = inf + (W.h[i] - inf) * exp(-delta * (r.ah + r.bh));
        inf = r.an / (r.an + r.bn);
        W.n[i] = inf + (W.n[i] - inf) * exp(-delta * (r.an + r.bn));
      }
      for (uint32_t i = tid; i < bi.n_syn; i += kThreads) {
        const uint32_t c = W.syn_cell[i];
        const uint32_t md = s_mode[c];
        if (!md) continue;
        W.g[i] = W.g[i] * (md == 1 ? W.syn_decay[i] : exp(-s_delta[c] / W.syn_tau[i]));
      }
      if ((uint32_t)tid < n_cell && s_mode[tid]) {
        const double vd = W.V[W.cell_det[tid]], vp = s_vprev[tid];
        if (s_armed[tid] && vp < M.theta && M.theta <= vd) {
          const double ts = s_tcur[tid] + s_delta[tid] * (M.theta - vp) / (vd - vp);
          const unsigned long long pos = atomicAdd(&M.counters[CNT_SPIKES], 1ull);
          if ((int64_t)pos < M.spike_cap) { M.spike_cell[pos] = M.cell_orig[bi.cell_base + tid]; M.spike_t[pos] = ts; }
          else atomicOr(&M.counters[CNT_ERROR], 1ull);
          s_armed[tid] = 0;
        }
        if (vd < M.theta) s_armed[tid] = 1;
        s_tcur[tid] = s_tnext[tid];
      }
      __syncthreads();
    }
  }
  if ((uint32_t)tid < n_cell) {
    CellRt rt; rt.ev_cur = s_evcur[tid]; rt.ev_end = s_evend[tid]; rt.armed = s_armed[tid]; rt.pad = 0;
    M.cell_rt[bi.cell_base + tid] = rt;
  }
  if (tid == 0) {
    atomicAdd(&M.counters[CNT_SUBSTEPS], (unsigned long long)s_substeps);
    if (s_delivered) atomicAdd(&M.counters[CNT_DELIVERED], (unsigned long long)s_delivered);
  }
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
    const uint32_t src = M.spike_cell[s];
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

__global__ void spikes_done_kernel(DevModel M) {
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
  CellRt rt = M.cell_rt[c];
  rt.ev_cur = off; rt.ev_end = ok ? off + total : off;
  M.cell_rt[c] = rt;
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

// per cell: order by (time, synapse, weight) - lists are a handful of events long
__global__ void ev_sort_kernel(DevModel M) {
  int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= M.n_cells) return;
  const uint32_t b = M.cell_rt[c].ev_cur, e = M.cell_rt[c].ev_end;
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
}

__global__ void pool_swap_kernel(DevModel M) {
  M.counters[CNT_POOL] = M.counters[CNT_POOL_NEXT];
  M.counters[CNT_POOL_NEXT] = 0;
}

// ------------------------------------------------------------------------------------------
// read-back / state injection helpers
// ------------------------------------------------------------------------------------------
__global__ void gather_kernel(const double* state, const uint32_t* idx, int64_t n, double* out) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < n) out[i] = state[idx[i]];
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

int cable_smem_bytes(uint32_t max_block_lanes) { return (int)(2 * align_up(max_block_lanes, 16) * sizeof(double)); }
int cable_smem_limit() { return 160 * 1024; }

cudaError_t launch_factor(const DevModel& M, double dt, cudaStream_t s) {
  factor_kernel<<<(unsigned)M.n_blocks, kThreads, 0, s>>>(M, dt);
  return cudaGetLastError();
}

cudaError_t launch_init(const DevModel& M, cudaStream_t s) {
  init_kernel<<<(unsigned)M.n_blocks, kThreads, 0, s>>>(M);
  return cudaGetLastError();
}

cudaError_t launch_reset_detectors(const DevModel& M, cudaStream_t s) {
  reset_detectors_kernel<<<grid_for(M.n_cells, 256), 256, 0, s>>>(M);
  return cudaGetLastError();
}

cudaError_t launch_cable(const DevModel& M, const StepArgs& A, int dyn_smem, cudaStream_t s) {
  static int configured = -1;
  if (dyn_smem > 48 * 1024 && configured < dyn_smem) {
    cudaError_t e = cudaFuncSetAttribute(cable_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_smem);
    if (e != cudaSuccess) return e;
    configured = dyn_smem;
  }
  cable_kernel<<<(unsigned)M.n_blocks, kThreads, dyn_smem, s>>>(M, A);
  return cudaGetLastError();
}

cudaError_t launch_build_events(const DevModel& M, int cur, double t_win, cudaStream_t s, int* launches) {
  const unsigned gc = grid_for(M.n_cells, 256);
  const int64_t nb = (M.n_cells + kScanBlock - 1) / kScanBlock;
  ev_count_ext_kernel<<<gc, 256, 0, s>>>(M, t_win);
  ev_count_pool_kernel<<<592, 256, 0, s>>>(M, cur, t_win);
  scan_local_kernel<<<(unsigned)nb, kScanBlock, 0, s>>>(M.ev_fill, M.ev_off, M.scan_tmp, M.n_cells);
  scan_sums_kernel<<<1, 32, 0, s>>>(M.scan_tmp, nb, M, M.n_cells);
  ev_place_kernel<<<gc, 256, 0, s>>>(M, t_win);
  ev_scatter_pool_kernel<<<592, 256, 0, s>>>(M, cur, t_win);
  ev_sort_kernel<<<gc, 256, 0, s>>>(M);
  pool_swap_kernel<<<1, 1, 0, s>>>(M);
  if (launches) *launches += 8;
  return cudaGetLastError();
}

cudaError_t launch_spikes_to_events(const DevModel& M, int cur, cudaStream_t s, int* launches) {
  spikes_to_events_kernel<<<296, 256, 0, s>>>(M, cur);
  spikes_done_kernel<<<1, 1, 0, s>>>(M);
  if (launches) *launches += 2;
  return cudaGetLastError();
}

cudaError_t launch_gather(const double* state, const uint32_t* idx, int64_t n, double* out, cudaStream_t s) {
  if (n > 0) gather_kernel<<<grid_for(n, 256), 256, 0, s>>>(state, idx, n, out);
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
