// api.cpp - the C ABI of include/arbb200.h: workspace carving, upload, the epoch loop, read-back.
// Host logic only; every arithmetic step of the method runs in kernels.cu.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/arbb200.h"
#include "kernels.cuh"
#include "layout.hpp"

using namespace arbb;

namespace {

thread_local std::string g_create_error;

struct Region { size_t off = 0, bytes = 0; };

// Carves the caller's workspace.  The same walk gives arb_plan its size.
struct Carver {
  size_t pos = 0;
  Region take(size_t bytes) {
    Region r;
    r.off = pos; r.bytes = bytes;
    pos += (bytes + 255) / 256 * 256;
    return r;
  }
};

struct Regions {
  Region units, gdescs, ghot, ghotflag, gen, fast, state, topo, scratch, factor_dcontrib, cell_rt_idx, cell_orig, ev_off, ev_t, ev_gidx, ev_w, ev_fill,
      ext_off, ext_t, ext_gidx, ext_w, ext_cur, conn_off, conn_dst, conn_gidx, conn_delay, conn_w,
      pool_t[2], pool_dst[2], pool_gidx[2], pool_w[2], spike_cell, spike_t, counters, scan_tmp,
      cv_idx, syn_idx, hh_m_idx, hh_stride, hh_cv, io, pc_kind, pc_par, pc_src_off, pc_src_time, pc_cv, lazy_run, run_off, run_gidx;
  size_t total = 0;
};

struct Caps { int64_t pool = 0, ev = 0, spikes = 0; };

// Capacities (include/arbb200.h, "Capacities").  The pool holds events in flight: a connection whose
// delay spans k epochs carries up to k events per spike train period; the default allows one spike every
// 2 ms per connection over the longest delay, and at least four events per connection.
Caps capacities(const HostModel& H, const arb_desc& d) {
  Caps c;
  const int64_t per_conn = std::max<int64_t>(4, (int64_t)std::ceil(H.max_delay / 2.0) + 1);
  c.pool = d.cap_events > 0 ? d.cap_events : per_conn * H.n_conn + 1024;
  c.ev = c.pool + H.n_ext + 16;
  c.spikes = d.cap_spikes > 0 ? d.cap_spikes : std::max<int64_t>(1 << 20, 64 * H.n_cells);
  return c;
}
constexpr int64_t kDrainSteps = 2000;   // the device spike buffer is drained at least this often

// upper bound of the CTAs of a cell-group launch
int64_t group_cta_cap(const HostModel& H) { return std::min<int64_t>(H.n_groups, kMaxGroupCtas); }

Regions carve(const HostModel& H, const Caps& cap) {
  Regions R;
  Carver C;
  const size_t nc = (size_t)H.n_cells;
  R.units = C.take(sizeof(UnitDesc) * (size_t)H.n_units);
  R.gdescs = C.take(sizeof(GroupDesc) * (size_t)H.n_groups);
  R.ghot = C.take(4 * 3 * (size_t)H.n_groups);
  R.ghotflag = C.take(4 * 2 * (size_t)H.n_groups);
  R.gen = C.take(8 * (size_t)H.gen_doubles);
  R.fast = C.take((size_t)H.fast_bytes);
  R.state = C.take(8 * (size_t)H.state_doubles);
  R.topo = C.take((size_t)H.topo_bytes);
  R.scratch = C.take(8 * (size_t)H.scratch_doubles);
  R.factor_dcontrib = C.take(8 * (size_t)H.n_lanes);
  R.cell_rt_idx = C.take(4 * nc);
  R.cell_orig = C.take(4 * nc);
  R.ev_off = C.take(4 * (nc + 1));
  R.ev_t = C.take(8 * (size_t)cap.ev);
  R.ev_gidx = C.take(4 * (size_t)cap.ev);
  R.ev_w = C.take(8 * (size_t)cap.ev);
  R.ev_fill = C.take(4 * nc);
  R.ext_off = C.take(4 * (nc + 1));
  R.ext_t = C.take(8 * (size_t)H.n_ext);
  R.ext_gidx = C.take(4 * (size_t)H.n_ext);
  R.ext_w = C.take(8 * (size_t)H.n_ext);
  R.ext_cur = C.take(4 * nc);
  R.conn_off = C.take(4 * ((size_t)H.n_src + 1));
  R.conn_dst = C.take(4 * (size_t)H.n_conn);
  R.conn_gidx = C.take(4 * (size_t)H.n_conn);
  R.conn_delay = C.take(8 * (size_t)H.n_conn);
  R.conn_w = C.take(8 * (size_t)H.n_conn);
  for (int i = 0; i < 2; ++i) {
    R.pool_t[i] = C.take(8 * (size_t)cap.pool);
    R.pool_dst[i] = C.take(4 * (size_t)cap.pool);
    R.pool_gidx[i] = C.take(4 * (size_t)cap.pool);
    R.pool_w[i] = C.take(8 * (size_t)cap.pool);
  }
  R.spike_cell = C.take(4 * (size_t)cap.spikes);
  R.spike_t = C.take(8 * (size_t)cap.spikes);
  R.counters = C.take(8 * CNT_COUNT);
  R.scan_tmp = C.take(4 * ((nc + 1023) / 1024 + 1));
  R.cv_idx = C.take(4 * (size_t)H.n_cv);
  R.syn_idx = C.take(4 * (size_t)H.n_syn);
  R.hh_m_idx = C.take(4 * (size_t)H.n_hh);
  R.hh_stride = C.take(4 * (size_t)H.n_hh);
  R.hh_cv = C.take(4 * (size_t)H.n_hh);
  R.io = C.take(8 * (size_t)std::max<int64_t>(std::max(H.n_cv, H.n_syn), 16));
  R.pc_kind = C.take(4 * (size_t)H.n_pcells);
  R.pc_par = C.take(48 * (size_t)H.n_pcells);
  R.pc_src_off = C.take(4 * ((size_t)H.n_pcells + 1));
  R.pc_src_time = C.take(8 * (size_t)H.n_sched);
  R.pc_cv = C.take(4 * (size_t)H.n_pcells);
  R.lazy_run = C.take(4 * (size_t)H.n_lazy);
  R.run_off = C.take(4 * ((size_t)H.n_runs + 1));
  R.run_gidx = C.take(4 * (size_t)H.n_runs);
  R.total = C.pos;
  return R;
}

}  // namespace

struct arb_model {
  HostModel H;          // pools are released after upload; counts and maps stay
  Regions R;
  Caps cap;
  DevModel D;
  char* ws = nullptr;
  cudaStream_t stream = nullptr;
  double t = 0.0, factored_dt = 0.0;
  int64_t grid_steps = 0, launches = 0;
  int64_t opt_fused = 0, opt_epoch = 0, opt_timing = 0, last_epoch_steps = 0;
  std::vector<cudaEvent_t> tev;          // timing events, reused (ARB_OPT_TIMING)
  double cable_ms = 0, event_ms = 0;
  int64_t cable_timed = 0, event_timed = 0;
  int cur_pool = 0;
  int sm_count = 148;
  int group_grid = 0, last_ggrid = 0;
  // the cable kernels of one grid step (cell groups, the forest launch classes, block units) do not depend on
  // each other: they run on side streams forked from / joined to the model's stream with events
  static constexpr int kSide = 1 + kForestClasses;
  cudaStream_t side[kSide] = {};
  cudaEvent_t fork_ev = nullptr, join_ev[kSide] = {};
  int64_t opt_overlap = 1;
  int64_t group_launches = 0, opt_group_ctas = 0, opt_hot = 1;
  bool prev_marked_hot = false;
  int64_t group_slots = 0, group_streamed = 0;   // statistics: CV slots incl. padding, bytes one grid step streams
  bool broken = false;
  int broken_code = ARB_E_OVERFLOW;
  std::string err;
  // spike history in host memory: arb_advance drains the device buffer into it
  std::vector<uint32_t> sp_cell;
  std::vector<double> sp_time;
  bool sp_sorted = true;
  // shards: spikes not yet handed to arb_spike_block (global ids)
  std::vector<int64_t> pend_gid;
  std::vector<double> pend_t;
};

namespace {

template <class T>
T* at(arb_model* m, const Region& r) { return reinterpret_cast<T*>(m->ws + r.off); }

int fail(arb_model* m, int code, const std::string& s) {
  if (m) m->err = s; else g_create_error = s;
  return code;
}

int cuda_fail(arb_model* m, cudaError_t e, const char* where) {
  return fail(m, ARB_E_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}

#define CU(m, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(m, e_, #call); } while (0)

template <class T>
cudaError_t upload(arb_model* m, const Region& r, const std::vector<T>& v) {
  if (v.empty()) return cudaSuccess;
  return cudaMemcpyAsync(m->ws + r.off, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, m->stream);
}

// layout options travel in the description (no process-wide state)
int params_of(const arb_desc& d, BuildParams& P, std::string& err) {
  if (d.layout_group_min_cells < 0 || d.layout_forest_cv < 0 || d.cap_spikes < 0 || d.cap_events < 0) { err = "negative layout / capacity option"; return ARB_E_INVALID; }
  if (d.layout_forest_cv > 0) { P.forest_cv = (uint32_t)std::min<int64_t>(d.layout_forest_cv, 1 << 20); P.forest_cv_auto = false; }
  if (d.layout_group_min_cells > 0) P.group_min_cells = d.layout_group_min_cells >= 0x7FFFFFFF ? 0u : (uint32_t)d.layout_group_min_cells;
  return ARB_OK;
}

}  // namespace

extern "C" {

int arb_plan(const arb_desc* desc, size_t* workspace_bytes) {
  if (!desc || !workspace_bytes) return fail(nullptr, ARB_E_NULL, "arb_plan: NULL argument");
  try {
    HostModel H;
    std::string err;
    BuildParams P;
    int rc = params_of(*desc, P, err);
    if (!rc) rc = build(*desc, P, false, H, err);
    if (rc) return fail(nullptr, rc, err);
    *workspace_bytes = carve(H, capacities(H, *desc)).total;
    return ARB_OK;
  } catch (const std::bad_alloc&) {
    return fail(nullptr, ARB_E_NOMEM, "arb_plan: out of host memory");
  }
}

int arb_create(const arb_desc* desc, void* dev_workspace, size_t bytes, void* cuda_stream, arb_model** out) {
  if (!desc || !dev_workspace || !out) return fail(nullptr, ARB_E_NULL, "arb_create: NULL argument");
  *out = nullptr;
  arb_model* m = nullptr;
  try {
    m = new arb_model();
    std::string err;
    BuildParams BP;
    int rc = params_of(*desc, BP, err);
    if (!rc) rc = build(*desc, BP, true, m->H, err);
    if (rc) { delete m; return fail(nullptr, rc, err); }
    HostModel& H = m->H;
    m->cap = capacities(H, *desc);
    m->R = carve(H, m->cap);
    if (bytes < m->R.total) { delete m; return fail(nullptr, ARB_E_WORKSPACE, "arb_create: workspace smaller than arb_plan reported"); }
    if (reinterpret_cast<uintptr_t>(dev_workspace) % 256) { delete m; return fail(nullptr, ARB_E_WORKSPACE, "arb_create: workspace must be 256-byte aligned"); }
    m->ws = static_cast<char*>(dev_workspace);
    m->stream = static_cast<cudaStream_t>(cuda_stream);
    {
      int dev = 0, sms = 0;
      if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) {
        delete m;
        return fail(nullptr, ARB_E_CUDA, "arb_create: no CUDA device (there is no CPU fallback)");
      }
      m->sm_count = sms;
    }
    // the kernels' shared-memory opt-in is per device: (re)done for every model, never cached
    if (configure_kernels() != cudaSuccess) { delete m; return fail(nullptr, ARB_E_CUDA, "arb_create: cannot opt the cable kernels into large shared memory"); }
    int group_ctas = 0;
    if (H.n_groups > 0 && (group_ctas = group_ctas_per_sm(group_smem_plan(H.gcaps).bytes)) == 0) { delete m; return fail(nullptr, ARB_E_INVALID, "arb_create: a cell group does not fit in shared memory"); }
    auto bail = [&](cudaError_t e, const char* w) { std::string s = std::string(w) + ": " + cudaGetErrorString(e); delete m; return fail(nullptr, ARB_E_CUDA, s); };
    cudaError_t e;
    const Regions& R = m->R;
    if ((e = cudaMemsetAsync(m->ws, 0, m->R.total, m->stream)) != cudaSuccess) return bail(e, "cudaMemsetAsync");
    if ((e = upload(m, R.units, H.descs)) != cudaSuccess) return bail(e, "upload units");
    if ((e = upload(m, R.gdescs, H.gdescs)) != cudaSuccess) return bail(e, "upload groups");
    if ((e = upload(m, R.gen, H.gen)) != cudaSuccess) return bail(e, "upload gen");
    if ((e = upload(m, R.fast, H.fast)) != cudaSuccess) return bail(e, "upload fast");
    if ((e = upload(m, R.state, H.state)) != cudaSuccess) return bail(e, "upload state");
    if ((e = upload(m, R.topo, H.topo)) != cudaSuccess) return bail(e, "upload topo");
    if ((e = upload(m, R.cell_orig, H.cell_order)) != cudaSuccess) return bail(e, "upload cell order");
    if ((e = upload(m, R.cell_rt_idx, H.cell_rt_idx)) != cudaSuccess) return bail(e, "upload cell runtime map");
    if ((e = upload(m, R.ext_off, H.ext_off)) != cudaSuccess) return bail(e, "upload ext_off");
    if ((e = upload(m, R.ext_t, H.ext_t)) != cudaSuccess) return bail(e, "upload ext_t");
    if ((e = upload(m, R.ext_gidx, H.ext_gidx)) != cudaSuccess) return bail(e, "upload ext_gidx");
    if ((e = upload(m, R.ext_w, H.ext_w)) != cudaSuccess) return bail(e, "upload ext_w");
    {
      std::vector<uint32_t> cur(H.ext_off.begin(), H.ext_off.end() - 1);
      if ((e = upload(m, R.ext_cur, cur)) != cudaSuccess) return bail(e, "upload ext_cur");
      if ((e = cudaStreamSynchronize(m->stream)) != cudaSuccess) return bail(e, "sync");
    }
    if ((e = upload(m, R.conn_off, H.conn_off)) != cudaSuccess) return bail(e, "upload conn_off");
    if ((e = upload(m, R.conn_dst, H.conn_dst)) != cudaSuccess) return bail(e, "upload conn_dst");
    if ((e = upload(m, R.conn_gidx, H.conn_gidx)) != cudaSuccess) return bail(e, "upload conn_gidx");
    if ((e = upload(m, R.conn_delay, H.conn_delay)) != cudaSuccess) return bail(e, "upload conn_delay");
    if ((e = upload(m, R.conn_w, H.conn_w)) != cudaSuccess) return bail(e, "upload conn_w");
    if ((e = upload(m, R.cv_idx, H.cv_state_idx)) != cudaSuccess) return bail(e, "upload cv map");
    if ((e = upload(m, R.syn_idx, H.syn_state_idx)) != cudaSuccess) return bail(e, "upload syn map");
    if ((e = upload(m, R.hh_m_idx, H.hh_m_idx)) != cudaSuccess) return bail(e, "upload hh map");
    if ((e = upload(m, R.hh_stride, H.hh_stride)) != cudaSuccess) return bail(e, "upload hh map");
    if ((e = upload(m, R.hh_cv, H.hh_cv)) != cudaSuccess) return bail(e, "upload hh map");
    if ((e = upload(m, R.pc_kind, H.pc_kind)) != cudaSuccess || (e = upload(m, R.pc_par, H.pc_par)) != cudaSuccess ||
        (e = upload(m, R.pc_src_off, H.pc_src_off)) != cudaSuccess || (e = upload(m, R.pc_src_time, H.pc_src_time)) != cudaSuccess ||
        (e = upload(m, R.pc_cv, H.pc_cv)) != cudaSuccess) return bail(e, "upload point cells");
    if ((e = upload(m, R.lazy_run, H.lazy_run)) != cudaSuccess || (e = upload(m, R.run_off, H.run_off)) != cudaSuccess ||
        (e = upload(m, R.run_gidx, H.run_gidx)) != cudaSuccess) return bail(e, "upload synapse runs");
    DevModel& D = m->D;
    std::memset(&D, 0, sizeof D);
    D.units = at<UnitDesc>(m, R.units);
    D.n_units = H.n_units; D.n_forests = H.n_forests; D.n_cells = H.n_cells;
    for (int k = 0; k < kForestClasses; ++k) D.fcls[k] = H.fcls[k];
    D.gen = at<double>(m, R.gen); D.fast = at<uint8_t>(m, R.fast); D.state = at<double>(m, R.state);
    D.topo = at<uint8_t>(m, R.topo); D.scratch = at<double>(m, R.scratch);
    D.factor_dcontrib = at<double>(m, R.factor_dcontrib);
    D.cell_orig = at<uint32_t>(m, R.cell_orig); D.cell_rt_idx = at<uint32_t>(m, R.cell_rt_idx);
    D.ev_off = at<uint32_t>(m, R.ev_off); D.ev_t = at<double>(m, R.ev_t); D.ev_gidx = at<uint32_t>(m, R.ev_gidx);
    D.ev_w = at<double>(m, R.ev_w); D.ev_fill = at<uint32_t>(m, R.ev_fill); D.ev_cap = m->cap.ev;
    D.ext_off = at<uint32_t>(m, R.ext_off); D.ext_t = at<double>(m, R.ext_t); D.ext_gidx = at<uint32_t>(m, R.ext_gidx);
    D.ext_w = at<double>(m, R.ext_w); D.ext_cur = at<uint32_t>(m, R.ext_cur);
    D.conn_off = at<uint32_t>(m, R.conn_off); D.conn_dst = at<uint32_t>(m, R.conn_dst); D.conn_gidx = at<uint32_t>(m, R.conn_gidx);
    D.conn_delay = at<double>(m, R.conn_delay); D.conn_w = at<double>(m, R.conn_w);
    D.gid_base = H.gid_base;
    D.lazy_base = (uint32_t)H.lazy_base; D.lazy_n = (uint32_t)H.n_lazy; D.n_runs = H.n_runs;
    D.lazy_run = at<uint32_t>(m, R.lazy_run); D.run_off = at<uint32_t>(m, R.run_off); D.run_gidx = at<uint32_t>(m, R.run_gidx);
    D.n_pcells = H.n_pcells; D.pc_first = H.pc_first; D.pc_state_base = H.pc_state_base;
    D.pc_kind = at<int32_t>(m, R.pc_kind); D.pc_par = at<double>(m, R.pc_par); D.pc_src_off = at<uint32_t>(m, R.pc_src_off);
    D.pc_src_time = at<double>(m, R.pc_src_time); D.pc_cv = at<uint32_t>(m, R.pc_cv);
    for (int i = 0; i < 2; ++i) {
      D.pool[i].t = at<double>(m, R.pool_t[i]); D.pool[i].dst = at<uint32_t>(m, R.pool_dst[i]);
      D.pool[i].gidx = at<uint32_t>(m, R.pool_gidx[i]); D.pool[i].w = at<double>(m, R.pool_w[i]);
    }
    D.syn_uniform = H.syn_uniform ? 1 : 0; D.syn_e_u = H.syn_e_u; D.syn_tau_u = H.syn_tau_u; D.syn_decay_u = 1.0;
    D.groups = at<GroupDesc>(m, R.gdescs); D.n_groups = H.n_groups;
    for (const GroupDesc& g : H.gdescs) {
      const GConstOff co = gconst_offsets(g.n_cv, g.n_hh_rows, g.n_syn_rows, g.n_cl_rows, H.syn_uniform);
      m->group_slots += (int64_t)g.n_cv * kG;
      m->group_streamed += co.total + 8 * (int64_t)gstate_offsets(g.n_cv, g.n_hh_rows, g.n_syn_rows).total + 8 * (int64_t)gcv_elems(g.n_cv);
    }
    D.gplan = group_smem_plan(H.gcaps);
    D.l2_prefetch = 1;
    D.ghot = at<uint32_t>(m, R.ghot); D.ghotflag = at<uint32_t>(m, R.ghotflag);   // zeroed with the workspace
    if (H.n_groups > 0)
      m->group_grid = (int)std::min<int64_t>(group_cta_cap(H), (int64_t)m->sm_count * group_ctas);
    D.pool_cap = m->cap.pool;
    D.spike_cell = at<uint32_t>(m, R.spike_cell); D.spike_t = at<double>(m, R.spike_t); D.spike_cap = m->cap.spikes;
    D.counters = at<unsigned long long>(m, R.counters);
    D.scan_tmp = at<uint32_t>(m, R.scan_tmp);
    D.ena = H.ena; D.ek = H.ek; D.el = H.el; D.theta = H.threshold;
    D.sm_count = m->sm_count;
    {
      const unsigned long long g0[2] = {(unsigned long long)m->group_grid, (unsigned long long)m->group_grid};
      if ((e = cudaMemcpyAsync(D.counters + CNT_GROUP0, g0, sizeof g0, cudaMemcpyHostToDevice, m->stream)) != cudaSuccess) return bail(e, "upload counters");
      if ((e = cudaStreamSynchronize(m->stream)) != cudaSuccess) return bail(e, "cudaStreamSynchronize");
      m->last_ggrid = m->group_grid;
    }
    if ((e = launch_init(D, m->stream)) != cudaSuccess) return bail(e, "init kernel");
    if ((e = launch_forest_init(D, m->stream)) != cudaSuccess) return bail(e, "forest init kernel");
    {
      int n_kinds = (H.n_groups > 0) + (H.n_units > H.n_forests);
      for (int k = 0; k < kForestClasses; ++k) n_kinds += H.fcls[k].count > 0;
      if (n_kinds > 1) {                   // side streams only where there is something to overlap
        if ((e = cudaEventCreateWithFlags(&m->fork_ev, cudaEventDisableTiming)) != cudaSuccess) return bail(e, "cudaEventCreate");
        for (int i = 0; i < arb_model::kSide; ++i) {
          if ((e = cudaStreamCreateWithFlags(&m->side[i], cudaStreamNonBlocking)) != cudaSuccess) return bail(e, "cudaStreamCreate");
          if ((e = cudaEventCreateWithFlags(&m->join_ev[i], cudaEventDisableTiming)) != cudaSuccess) return bail(e, "cudaEventCreate");
        }
      }
    }
    if ((e = launch_group_init(D, m->stream)) != cudaSuccess) return bail(e, "group init kernel");
    if ((e = cudaStreamSynchronize(m->stream)) != cudaSuccess) return bail(e, "cudaStreamSynchronize");
    // host pools are no longer needed
    std::vector<double>().swap(H.gen); std::vector<uint8_t>().swap(H.fast); std::vector<double>().swap(H.state);
    std::vector<uint8_t>().swap(H.topo); std::vector<UnitDesc>().swap(H.descs); std::vector<GroupDesc>().swap(H.gdescs); std::vector<uint32_t>().swap(H.cell_rt_idx);
    std::vector<uint32_t>().swap(H.cv_state_idx); std::vector<uint32_t>().swap(H.syn_state_idx);
    std::vector<uint32_t>().swap(H.hh_m_idx); std::vector<uint32_t>().swap(H.hh_stride); std::vector<uint32_t>().swap(H.hh_cv);
    std::vector<uint32_t>().swap(H.conn_off); std::vector<uint32_t>().swap(H.conn_dst); std::vector<uint32_t>().swap(H.conn_gidx);
    std::vector<double>().swap(H.conn_delay); std::vector<double>().swap(H.conn_w);
    std::vector<uint32_t>().swap(H.ext_off); std::vector<uint32_t>().swap(H.ext_gidx);
    std::vector<double>().swap(H.ext_t); std::vector<double>().swap(H.ext_w);
    *out = m;
    return ARB_OK;
  } catch (const std::bad_alloc&) {
    delete m;
    return fail(nullptr, ARB_E_NOMEM, "arb_create: out of host memory");
  }
}

}  // extern "C"

namespace {

// Moves the spikes of the device buffer into the host history and empties the buffer.  Only valid at an
// epoch boundary, after spikes_to_events has walked every spike (CNT_SPIKES_DONE == CNT_SPIKES).  Returns
// the error bits seen so far in *err_bits.
int drain(arb_model* m, unsigned long long* cnt) {
  DevModel& D = m->D;
  CU(m, cudaMemcpyAsync(cnt, D.counters, sizeof(unsigned long long) * CNT_COUNT, cudaMemcpyDeviceToHost, m->stream));
  CU(m, cudaStreamSynchronize(m->stream));
  const size_t n = (size_t)std::min<unsigned long long>(cnt[CNT_SPIKES], (unsigned long long)m->cap.spikes);
  if (n > 0) {
    const size_t old = m->sp_cell.size();
    m->sp_cell.resize(old + n);
    m->sp_time.resize(old + n);
    CU(m, cudaMemcpyAsync(m->sp_cell.data() + old, D.spike_cell, 4 * n, cudaMemcpyDeviceToHost, m->stream));
    CU(m, cudaMemcpyAsync(m->sp_time.data() + old, D.spike_t, 8 * n, cudaMemcpyDeviceToHost, m->stream));
    CU(m, cudaMemsetAsync(D.counters + CNT_SPIKES, 0, 2 * sizeof(unsigned long long), m->stream));   // CNT_SPIKES, CNT_SPIKES_DONE
    CU(m, cudaStreamSynchronize(m->stream));
    m->sp_sorted = false;
    if (m->H.n_src != m->H.n_cells || m->H.gid_base != 0)
      for (size_t i = old; i < old + n; ++i) { m->pend_gid.push_back(m->H.gid_base + (int64_t)m->sp_cell[i]); m->pend_t.push_back(m->sp_time[i]); }
  }
  return ARB_OK;
}

int check_error_bits(arb_model* m, const unsigned long long* cnt) {
  const unsigned long long e = cnt[CNT_ERROR];
  if (!e) return ARB_OK;
  m->broken = true;
  char buf[320];
  if (e & 8ull) {
    m->broken_code = ARB_E_DIVERGED;
    snprintf(buf, sizeof buf, "a detector voltage became NaN / Inf: the time step is too long for the explicit membrane currents (reading R1)");
  } else {
    m->broken_code = ARB_E_OVERFLOW;
    snprintf(buf, sizeof buf, "capacity exceeded:%s%s%s; create the model again with a larger arb_desc.%s (spikes seen %llu of cap_spikes %lld, events in flight %llu of cap_events %lld)",
             (e & 1) ? " spike buffer" : "", (e & 2) ? " event pool" : "", (e & 4) ? " epoch event list" : "",
             (e & 1) ? "cap_spikes" : "cap_events", cnt[CNT_SPIKES], (long long)m->cap.spikes,
             std::max(cnt[CNT_POOL], cnt[CNT_POOL_PEAK]), (long long)m->cap.pool);
  }
  return fail(m, m->broken_code, buf);
}

}  // namespace

extern "C" {

int arb_advance(arb_model* m, double t_end, double dt) {
  if (!m) return fail(nullptr, ARB_E_NULL, "arb_advance: NULL model");
  if (m->broken) return fail(m, m->broken_code, "model unusable after an earlier error: " + m->err);
  if (!(dt > 0) || !std::isfinite(dt) || !std::isfinite(t_end)) return fail(m, ARB_E_INVALID, "arb_advance: dt must be > 0 and finite");
  if (t_end < m->t) return fail(m, ARB_E_INVALID, "arb_advance: t_end earlier than the current time");
  if (m->H.n_conn > 0 && m->H.min_delay < dt) return fail(m, ARB_E_INVALID, "arb_advance: dt longer than the shortest connection delay");
  if (t_end == m->t) return ARB_OK;
  DevModel& D = m->D;
  // from the first launch on, a failure leaves the device state half-advanced: the model is unusable
  auto cu_broken = [&](cudaError_t e, const char* where) {
    m->broken = true; m->broken_code = ARB_E_CUDA;
    return cuda_fail(m, e, where);
  };
#define CUB(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cu_broken(e_, #call); } while (0)
  if (dt != m->factored_dt) {
    D.syn_decay_u = D.syn_uniform ? std::exp(-dt / D.syn_tau_u) : 1.0;
    CUB(launch_factor(D, dt, m->stream));
    CUB(launch_forest_factor(D, dt, m->stream));
    CUB(launch_group_factor(D, dt, m->H.g_seg_cap, m->stream));
    m->factored_dt = dt;
    m->launches++;
  }
  // time grid (reading R9): t_k = t0 + k*dt by multiplication, last point = t_end
  const double t0 = m->t;
  int64_t nsteps = (int64_t)std::ceil((t_end - t0) / dt - 1e-9);
  if (nsteps < 1) nsteps = 1;
  const int last_full = std::fabs((t0 + (double)nsteps * dt) - t_end) <= 1e-9 * dt;
  // epoch: cells are independent for one minimum delay (reading R12); the 1e-6 guard is
  // described in include/arbb200.h (arb_advance)
  int64_t epoch = 1024;
  if (m->H.n_conn > 0) epoch = std::min<int64_t>(epoch, std::max<int64_t>(1, (int64_t)std::floor(m->H.min_delay / dt - 1e-6)));
  if (m->opt_epoch > 0) epoch = std::min(epoch, m->opt_epoch);
  const int64_t fused = m->opt_fused > 0 ? std::min(m->opt_fused, epoch) : epoch;
  m->last_epoch_steps = epoch;
  // a changed CTA count invalidates the work counters (they are reset to gridDim.x by the previous launch)
  const int ggrid = m->opt_group_ctas > 0 ? (int)std::min<int64_t>(m->opt_group_ctas, m->group_grid) : m->group_grid;
  if (ggrid != m->last_ggrid && m->H.n_groups > 0) {
    const unsigned long long g0[2] = {(unsigned long long)ggrid, (unsigned long long)ggrid};
    CUB(cudaMemcpyAsync(D.counters + CNT_GROUP0, g0, sizeof g0, cudaMemcpyHostToDevice, m->stream));
    CUB(cudaStreamSynchronize(m->stream));
    m->last_ggrid = ggrid;
  }
  int launches = 0;
  // optional device timing (ARB_OPT_TIMING): four events per epoch on the model's stream
  size_t n_tev = 0;
  std::vector<int> tev_cable, tev_event;   // launches between events (1,2) and (0,1)+(2,3)
  auto stamp = [&]() -> cudaError_t {
    if (!m->opt_timing) return cudaSuccess;
    if (n_tev == m->tev.size()) {
      cudaEvent_t ev;
      cudaError_t ce = cudaEventCreate(&ev);
      if (ce != cudaSuccess) return ce;
      m->tev.push_back(ev);
    }
    return cudaEventRecord(m->tev[n_tev++], m->stream);
  };
  auto collect_timing = [&]() {
    for (size_t i = 0; i + 3 < n_tev; i += 4) {
      float a = 0, b = 0, c = 0;
      cudaEventElapsedTime(&a, m->tev[i], m->tev[i + 1]);
      cudaEventElapsedTime(&b, m->tev[i + 1], m->tev[i + 2]);
      cudaEventElapsedTime(&c, m->tev[i + 2], m->tev[i + 3]);
      m->cable_ms += b; m->event_ms += a + c;
      m->cable_timed += tev_cable[i / 4]; m->event_timed += tev_event[i / 4];
    }
    n_tev = 0; tev_cable.clear(); tev_event.clear();
  };
  unsigned long long cnt[CNT_COUNT];
  int64_t since_drain = 0;
  for (int64_t k = 0; k < nsteps;) {
    const int64_t n_ep = std::min(epoch, nsteps - k);
    const double t_win = (k + n_ep == nsteps) ? t_end : t0 + (double)(k + n_ep) * dt;
    int l0 = launches;
    CUB(stamp());
    CUB(launch_build_events(D, m->cur_pool, t_win, m->stream, &launches));
    CUB(launch_point_cells(D, t_win, m->stream, &launches));
    m->cur_pool ^= 1;
    CUB(stamp());
    int l1 = launches;
    for (int64_t j = 0; j < n_ep; j += fused) {
      StepArgs A;
      A.t0 = t0; A.dt = dt; A.t_end = t_end; A.k_first = k + j; A.nk = std::min(fused, n_ep - j); A.nsteps = nsteps; A.last_full = last_full;
      A.parity = (int)(m->group_launches & 1);
      A.launch_id = (uint32_t)m->group_launches++;
      A.mark_hot = (A.nk == 1 && m->opt_hot) ? 1 : 0;
      A.hot_valid = m->prev_marked_hot ? 1 : 0;
      m->prev_marked_hot = A.mark_hot != 0;
      // cell groups on the model's stream; forests (largest launch class first) and block units beside them
      const bool overlap = m->fork_ev != nullptr && m->opt_overlap;
      if (overlap) CUB(cudaEventRecord(m->fork_ev, m->stream));
      int side = 0;
      auto on_side = [&](auto&& launch) -> cudaError_t {
        if (!overlap) return launch(m->stream);
        cudaStream_t st = m->side[side];
        cudaError_t ce = cudaStreamWaitEvent(st, m->fork_ev, 0);
        if (ce == cudaSuccess) ce = launch(st);
        if (ce == cudaSuccess) ce = cudaEventRecord(m->join_ev[side], st);
        if (ce == cudaSuccess) ce = cudaStreamWaitEvent(m->stream, m->join_ev[side], 0);
        ++side;
        return ce;
      };
      for (int c = kForestClasses - 1; c >= 0; --c)
        if (D.fcls[c].count > 0) CUB(on_side([&](cudaStream_t st) { return launch_forest_cable(D, A, c, st, &launches); }));
      if (D.n_units > D.n_forests) CUB(on_side([&](cudaStream_t st) { return launch_cable(D, A, st, &launches); }));
      CUB(launch_group_cable(D, A, ggrid, m->stream, &launches));
    }
    CUB(stamp());
    int l2 = launches;
    if (m->H.n_conn > 0) CUB(launch_spikes_to_events(D, m->cur_pool, m->stream, &launches));
    CUB(stamp());
    tev_cable.push_back(l2 - l1);
    tev_event.push_back((l1 - l0) + (launches - l2));
    k += n_ep;
    since_drain += n_ep;
    // the spike buffer is emptied into host memory at the end of the call and at least every kDrainSteps steps
    if (k == nsteps || since_drain >= kDrainSteps) {
      int rc = drain(m, cnt);
      if (rc) { m->broken = true; m->broken_code = rc; return rc; }
      collect_timing();
      since_drain = 0;
      if (cnt[CNT_ERROR]) break;
    }
  }
  m->launches += launches;
  m->t = t_end;
  m->grid_steps += nsteps;
  return check_error_bits(m, cnt);
#undef CUB
}

int64_t arb_spikes(arb_model* m, int64_t* cell, double* time, int64_t cap) {
  if (!m) return fail(nullptr, ARB_E_NULL, "arb_spikes: NULL model");
  if (cap > 0 && (!cell || !time)) return fail(m, ARB_E_NULL, "arb_spikes: NULL output");
  const int64_t count = (int64_t)m->sp_cell.size();
  if (cap <= 0 || count == 0) return count;
  try {
    if (!m->sp_sorted) {
      std::vector<int64_t> idx(count);
      for (int64_t i = 0; i < count; ++i) idx[i] = i;
      const std::vector<uint32_t>& c = m->sp_cell;
      const std::vector<double>& t = m->sp_time;
      std::sort(idx.begin(), idx.end(), [&](int64_t a, int64_t b) { return t[a] != t[b] ? t[a] < t[b] : c[a] < c[b]; });
      std::vector<uint32_t> c2(count);
      std::vector<double> t2(count);
      for (int64_t i = 0; i < count; ++i) { c2[i] = c[idx[i]]; t2[i] = t[idx[i]]; }
      m->sp_cell.swap(c2); m->sp_time.swap(t2);
      m->sp_sorted = true;
    }
    for (int64_t i = 0; i < std::min(cap, count); ++i) { cell[i] = m->sp_cell[i]; time[i] = m->sp_time[i]; }
  } catch (const std::bad_alloc&) {
    return fail(m, ARB_E_NOMEM, "arb_spikes: out of host memory");
  }
  return count;
}

int64_t arb_spike_block(arb_model* m, void* dev_block, int64_t cap) {
  if (!m || !dev_block) return fail(m, ARB_E_NULL, "arb_spike_block: NULL argument");
  if (cap < 0) return fail(m, ARB_E_INVALID, "arb_spike_block: negative capacity");
  const int64_t n = (int64_t)m->pend_gid.size();
  if (n > cap) return fail(m, ARB_E_OVERFLOW, "arb_spike_block: " + std::to_string(n) + " spikes do not fit a block of " + std::to_string(cap));
  try {
    std::vector<unsigned long long> blk(1 + 2 * (size_t)cap, 0ull);
    blk[0] = (unsigned long long)n;
    for (int64_t i = 0; i < n; ++i) {
      blk[1 + i] = (unsigned long long)m->pend_gid[i];
      std::memcpy(&blk[1 + cap + i], &m->pend_t[i], 8);
    }
    CU(m, cudaMemcpyAsync(dev_block, blk.data(), 8 * blk.size(), cudaMemcpyHostToDevice, m->stream));
    CU(m, cudaStreamSynchronize(m->stream));
  } catch (const std::bad_alloc&) {
    return fail(m, ARB_E_NOMEM, "arb_spike_block: out of host memory");
  }
  m->pend_gid.clear(); m->pend_t.clear();
  return n;
}

int arb_apply_spike_blocks(arb_model* m, const void* dev_blocks, int64_t n_blocks, int64_t cap, int64_t own_block) {
  if (!m || !dev_blocks) return fail(m, ARB_E_NULL, "arb_apply_spike_blocks: NULL argument");
  if (m->broken) return fail(m, m->broken_code, "model unusable after an earlier error: " + m->err);
  if (n_blocks < 0 || cap < 0) return fail(m, ARB_E_INVALID, "arb_apply_spike_blocks: negative count");
  if (m->H.n_conn == 0 || n_blocks == 0) return ARB_OK;
  // the events join the pool the next arb_advance builds its epoch lists from
  CU(m, launch_remote_spikes_to_events(m->D, m->cur_pool, static_cast<const unsigned long long*>(dev_blocks), n_blocks, cap, own_block, m->stream));
  unsigned long long cnt[CNT_COUNT];
  CU(m, cudaMemcpyAsync(cnt, m->D.counters, sizeof cnt, cudaMemcpyDeviceToHost, m->stream));
  CU(m, cudaStreamSynchronize(m->stream));
  m->launches += 2;
  return check_error_bits(m, cnt);
}

int arb_clear_spikes(arb_model* m) {
  if (!m) return fail(nullptr, ARB_E_NULL, "arb_clear_spikes: NULL model");
  m->sp_cell.clear(); m->sp_time.clear(); m->sp_sorted = true;
  return ARB_OK;
}

int arb_voltage(arb_model* m, double* out, int64_t n_cv) {
  if (!m || !out) return fail(m, ARB_E_NULL, "arb_voltage: NULL argument");
  if (n_cv != m->H.n_cv) return fail(m, ARB_E_INVALID, "arb_voltage: n_cv mismatch");
  double* io = at<double>(m, m->R.io);
  CU(m, launch_gather(m->D.state, at<uint32_t>(m, m->R.cv_idx), n_cv, io, m->stream));
  CU(m, launch_lif_relax(m->D, m->t, io, m->stream));
  CU(m, cudaMemcpyAsync(out, io, 8 * (size_t)n_cv, cudaMemcpyDeviceToHost, m->stream));
  CU(m, cudaStreamSynchronize(m->stream));
  return ARB_OK;
}

int arb_gates_noalloc(arb_model* m, int what, double* out, int64_t n_cv) {
  if (!m || !out) return fail(m, ARB_E_NULL, "arb_gates_noalloc: NULL argument");
  if (what != ARB_PROBE_M && what != ARB_PROBE_H && what != ARB_PROBE_N) return fail(m, ARB_E_INVALID, "arb_gates_noalloc: selector is not a gate (ARB_PROBE_M / H / N)");
  if (n_cv != m->H.n_cv) return fail(m, ARB_E_INVALID, "arb_gates_noalloc: n_cv mismatch");
  if (n_cv > noalloc_max_cv())
    return fail(m, ARB_E_INVALID, "arb_gates_noalloc: " + std::to_string(n_cv) + " control volumes exceed the static staging array of " +
                                  std::to_string(noalloc_max_cv()) + " doubles; use arb_probe (staging in the caller's workspace)");
  CU(m, launch_noalloc_gates(m->D.state, at<uint32_t>(m, m->R.hh_m_idx), at<uint32_t>(m, m->R.hh_stride), at<uint32_t>(m, m->R.hh_cv),
                             what - ARB_PROBE_M, m->H.n_hh, n_cv, out, m->stream));
  CU(m, cudaStreamSynchronize(m->stream));
  return ARB_OK;
}

int64_t arb_noalloc_max_cv(void) { return noalloc_max_cv(); }

int arb_probe(arb_model* m, int what, double* out, int64_t n) {
  if (!m || !out) return fail(m, ARB_E_NULL, "arb_probe: NULL argument");
  double* io = at<double>(m, m->R.io);
  switch (what) {
    case ARB_PROBE_M: case ARB_PROBE_H: case ARB_PROBE_N: {
      if (n != m->H.n_cv) return fail(m, ARB_E_INVALID, "arb_probe: size mismatch");
      CU(m, cudaMemsetAsync(io, 0, 8 * (size_t)n, m->stream));
      CU(m, launch_gather_hh(m->D.state, at<uint32_t>(m, m->R.hh_m_idx), at<uint32_t>(m, m->R.hh_stride),
                             at<uint32_t>(m, m->R.hh_cv), what - ARB_PROBE_M, m->H.n_hh, io, m->stream));
      CU(m, cudaMemcpyAsync(out, io, 8 * (size_t)n, cudaMemcpyDeviceToHost, m->stream));
      CU(m, cudaStreamSynchronize(m->stream));
      return ARB_OK;
    }
    case ARB_PROBE_SYN_G: {
      if (n != m->H.n_syn) return fail(m, ARB_E_INVALID, "arb_probe: size mismatch");
      if (n == 0) return ARB_OK;
      CU(m, launch_gather_syn(m->D, at<uint32_t>(m, m->R.syn_idx), n, m->t, io, m->stream));
      CU(m, cudaMemcpyAsync(out, io, 8 * (size_t)n, cudaMemcpyDeviceToHost, m->stream));
      CU(m, cudaStreamSynchronize(m->stream));
      return ARB_OK;
    }
    case ARB_PROBE_TIME:
      if (n < 1) return fail(m, ARB_E_INVALID, "arb_probe: size mismatch");
      out[0] = m->t;
      return ARB_OK;
    case ARB_PROBE_TIMING:
      if (n < 4) return fail(m, ARB_E_INVALID, "arb_probe: size mismatch");
      out[0] = m->cable_ms; out[1] = (double)m->cable_timed; out[2] = m->event_ms; out[3] = (double)m->event_timed;
      return ARB_OK;
    case ARB_PROBE_NSTEPS: case ARB_PROBE_STATS: {
      if (n < (what == ARB_PROBE_NSTEPS ? 2 : 8)) return fail(m, ARB_E_INVALID, "arb_probe: size mismatch");
      unsigned long long cnt[CNT_COUNT];
      CU(m, cudaMemcpyAsync(cnt, m->D.counters, sizeof cnt, cudaMemcpyDeviceToHost, m->stream));
      CU(m, cudaStreamSynchronize(m->stream));
      if (what == ARB_PROBE_NSTEPS) { out[0] = (double)m->grid_steps; out[1] = (double)cnt[CNT_SUBSTEPS]; return ARB_OK; }
      int64_t slots = 0, streamed = 0;
      for (const auto& u : m->H.units) { slots += u.n_slot; streamed += u.fast_bytes + u.state_bytes; }
      slots += m->group_slots; streamed += m->group_streamed;
      out[0] = (double)m->H.n_units; out[1] = (double)slots; out[2] = (double)m->H.n_lanes;
      out[3] = (double)m->R.total; out[4] = (double)cnt[CNT_DELIVERED]; out[5] = (double)m->launches;
      out[6] = (double)m->last_epoch_steps; out[7] = (double)streamed;
      if (n >= 12) {
        out[8] = 0.0; out[9] = 0.0; out[10] = 0.0;      // (warp units of round 1: replaced by forests)
        out[11] = (double)m->H.topo_records;
      }
      if (n >= 16) {
        out[12] = (double)m->H.n_groups; out[13] = (double)m->H.n_classes; out[14] = (double)m->group_grid;
        out[15] = (double)m->D.gplan.bytes;
      }
      if (n >= 20) {
        int64_t fctas = 0; uint32_t fsmem = 0;
        for (int k = 0; k < kForestClasses; ++k) { fctas = std::max(fctas, m->H.fcls[k].count); if (m->H.fcls[k].count) fsmem = std::max(fsmem, m->H.fcls[k].plan.bytes); }
        out[16] = (double)m->H.n_forests; out[17] = (double)(m->H.n_units - m->H.n_forests); out[18] = (double)fctas; out[19] = (double)fsmem;
      }
      return ARB_OK;
    }
  }
  return fail(m, ARB_E_INVALID, "arb_probe: unknown selector");
}

int arb_set_state(arb_model* m, const double* v, const double* hh_m, const double* hh_h, const double* hh_n, const double* syn_g) {
  if (!m) return fail(nullptr, ARB_E_NULL, "arb_set_state: NULL model");
  double* io = at<double>(m, m->R.io);
  if (v) {
    CU(m, cudaMemcpyAsync(io, v, 8 * (size_t)m->H.n_cv, cudaMemcpyHostToDevice, m->stream));
    CU(m, launch_scatter(m->D.state, at<uint32_t>(m, m->R.cv_idx), m->H.n_cv, io, m->stream));
    CU(m, cudaStreamSynchronize(m->stream));
  }
  const double* gates[3] = {hh_m, hh_h, hh_n};
  for (int w = 0; w < 3; ++w)
    if (gates[w]) {
      CU(m, cudaMemcpyAsync(io, gates[w], 8 * (size_t)m->H.n_cv, cudaMemcpyHostToDevice, m->stream));
      CU(m, launch_scatter_hh(m->D.state, at<uint32_t>(m, m->R.hh_m_idx), at<uint32_t>(m, m->R.hh_stride),
                              at<uint32_t>(m, m->R.hh_cv), w, m->H.n_hh, io, m->stream));
      CU(m, cudaStreamSynchronize(m->stream));
    }
  if (syn_g && m->H.n_syn > 0) {
    CU(m, cudaMemcpyAsync(io, syn_g, 8 * (size_t)m->H.n_syn, cudaMemcpyHostToDevice, m->stream));
    CU(m, launch_scatter(m->D.state, at<uint32_t>(m, m->R.syn_idx), m->H.n_syn, io, m->stream));
    CU(m, launch_lazy_rebuild(m->D, m->t, m->stream));      // cells that keep one conductance per run (R22)
    CU(m, cudaStreamSynchronize(m->stream));
  }
  CU(m, launch_reset_detectors(m->D, m->stream));
  if (v) CU(m, launch_point_reset(m->D, m->t, m->stream));
  CU(m, cudaStreamSynchronize(m->stream));
  return ARB_OK;
}

int arb_set_option(arb_model* m, int key, int64_t value) {
  if (!m) return fail(nullptr, ARB_E_NULL, "arb_set_option: NULL model");
  if (value < 0) return fail(m, ARB_E_INVALID, "arb_set_option: negative value");
  switch (key) {
    case ARB_OPT_FUSED_STEPS: m->opt_fused = value; return ARB_OK;
    case ARB_OPT_EPOCH_STEPS: m->opt_epoch = value; return ARB_OK;
    case ARB_OPT_OVERLAP: m->opt_overlap = value != 0; return ARB_OK;
    case ARB_OPT_LINEARISED:
      if (value != 0 && m->H.n_units > m->H.n_forests)
        return fail(m, ARB_E_INVALID, "arb_set_option: the conductance-linearised step is not available for block units (cells with "
                                      ">= 1,024 synapses or too large for shared memory)");
      if ((value != 0) != (m->D.linearised != 0)) { m->D.linearised = value != 0; m->factored_dt = 0.0; }   // coefficients are rebuilt
      return ARB_OK;
    case ARB_OPT_L2_PREFETCH: m->D.l2_prefetch = value != 0; return ARB_OK;
    case ARB_OPT_GROUP_CTAS: m->opt_group_ctas = value; return ARB_OK;
    case ARB_OPT_HOT_FIRST: m->opt_hot = value != 0; m->prev_marked_hot = false; return ARB_OK;
    case ARB_OPT_TIMING:
      m->opt_timing = value;
      m->cable_ms = m->event_ms = 0; m->cable_timed = m->event_timed = 0;
      return ARB_OK;
  }
  return fail(m, ARB_E_INVALID, "arb_set_option: unknown key");
}

// ---- the mechanism catalogue: a table that names the hand-written mechanisms and cell kinds ----
namespace {
struct CatParam { const char* field; const char* unit; double def; };
struct CatEntry { const char* name; int kind; int n; CatParam par[6]; };
const CatEntry kCatalogue[] = {
    {"hh", 0, 6, {{"hh_gnabar", "S/cm2", 0.12}, {"hh_gkbar", "S/cm2", 0.036}, {"hh_gl", "S/cm2", 3e-4}, {"hh_ena", "mV", 50.0},
                  {"hh_ek", "mV", -77.0}, {"hh_el", "mV", -54.3}}},
    {"pas", 0, 2, {{"pas_g", "S/cm2", 1e-5}, {"pas_e", "mV", -65.0}}},
    {"expsyn", 1, 2, {{"syn_tau", "ms", 2.0}, {"syn_e", "mV", 0.0}}},
    {"iclamp", 1, 3, {{"clamp_t0", "ms", 0.0}, {"clamp_t1", "ms", 0.0}, {"clamp_amp", "nA", 0.0}}},
    {"lif", 2, 6, {{"lif_tau_m", "ms", 10.0}, {"lif_v_th", "mV", -50.0}, {"lif_c_m", "nF", 0.25}, {"lif_e_l", "mV", -65.0},
                   {"lif_e_r", "mV", -70.0}, {"lif_t_ref", "ms", 2.0}}},
    {"spike_source", 2, 1, {{"src_time", "ms", 0.0}}},
};
constexpr int kCatalogueSize = (int)(sizeof kCatalogue / sizeof kCatalogue[0]);
}  // namespace

int arb_catalogue_size(void) { return kCatalogueSize; }

int arb_catalogue_entry(int index, const char** name, int* kind, int* n_params) {
  if (index < 0 || index >= kCatalogueSize) return ARB_E_INVALID;
  if (name) *name = kCatalogue[index].name;
  if (kind) *kind = kCatalogue[index].kind;
  if (n_params) *n_params = kCatalogue[index].n;
  return ARB_OK;
}

int arb_catalogue_param(int index, int param, const char** field, const char** unit, double* default_value) {
  if (index < 0 || index >= kCatalogueSize || param < 0 || param >= kCatalogue[index].n) return ARB_E_INVALID;
  if (field) *field = kCatalogue[index].par[param].field;
  if (unit) *unit = kCatalogue[index].par[param].unit;
  if (default_value) *default_value = kCatalogue[index].par[param].def;
  return ARB_OK;
}

int arb_catalogue_find(const char* name) {
  if (!name) return -1;
  for (int i = 0; i < kCatalogueSize; ++i) if (std::strcmp(name, kCatalogue[i].name) == 0) return i;
  return -1;
}

void arb_destroy(arb_model* m) {
  if (!m) return;
  if (m->ws) cudaStreamSynchronize(m->stream);
  for (cudaEvent_t ev : m->tev) cudaEventDestroy(ev);
  for (int i = 0; i < arb_model::kSide; ++i) {
    if (m->side[i]) { cudaStreamSynchronize(m->side[i]); cudaStreamDestroy(m->side[i]); }
    if (m->join_ev[i]) cudaEventDestroy(m->join_ev[i]);
  }
  if (m->fork_ev) cudaEventDestroy(m->fork_ev);
  delete m;
}

const char* arb_last_error(const arb_model* m) { return m ? m->err.c_str() : g_create_error.c_str(); }

}  // extern "C"
