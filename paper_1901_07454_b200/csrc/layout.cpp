// layout.cpp - see layout.hpp.  Host preprocessing only; nothing here runs per time step.
#include "layout.hpp"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstring>
#include <limits>
#include <thread>

namespace arbb {

namespace {

bool finite(double x) { return std::isfinite(x); }

template <class F>
void parallel_for(int64_t n, F&& f) {
  unsigned hw = std::thread::hardware_concurrency();
  int nt = (int)std::min<int64_t>(std::max(1u, std::min(hw, 32u)), std::max<int64_t>(1, n / 8));
  if (nt <= 1) {
    for (int64_t i = 0; i < n; ++i) f(i);
    return;
  }
  std::atomic<int64_t> next(0);
  std::vector<std::thread> th;
  for (int t = 0; t < nt; ++t)
    th.emplace_back([&] {
      for (;;) {
        int64_t i0 = next.fetch_add(16);
        if (i0 >= n) break;
        for (int64_t i = i0; i < std::min(n, i0 + 16); ++i) f(i);
      }
    });
  for (auto& t : th) t.join();
}

struct Lane {          // one branch of one cell of the block
  uint32_t level, len, lc, br;
  uint32_t cv_begin;   // into BlockScratch::cvs
  int32_t parent_br;   // branch id inside the cell or -1
  uint32_t first_cv;
};

struct CellScratch {
  uint32_t lane_begin = 0, n_br = 0;  // lanes of this cell are [lane_begin, lane_begin + n_br) before sorting
};

}  // namespace

int validate(const arb_desc& d, std::string& err) {
  auto fail = [&](int code, const std::string& s) { err = s; return code; };
  if (d.n_cells < 0 || d.n_clamp < 0 || d.n_conn < 0 || d.n_ext < 0) return fail(ARB_E_INVALID, "negative count");
  if (d.n_cells == 0) return fail(ARB_E_INVALID, "model has no cells");
  if (!d.cv_off || !d.cv_parent || !d.cv_area || !d.cv_cm || !d.cv_raxial) return fail(ARB_E_NULL, "compartment arrays must not be NULL");
  bool hh_any = d.hh_gnabar || d.hh_gkbar || d.hh_gl;
  if (hh_any && !(d.hh_gnabar && d.hh_gkbar && d.hh_gl)) return fail(ARB_E_INVALID, "hh arrays must be all given or all NULL");
  if ((d.pas_g != nullptr) != (d.pas_e != nullptr)) return fail(ARB_E_INVALID, "pas_g and pas_e must both be given or both be NULL");
  if (d.cv_off[0] != 0) return fail(ARB_E_INVALID, "cv_off[0] must be 0");
  if (d.syn_off && d.syn_off[0] != 0) return fail(ARB_E_INVALID, "syn_off[0] must be 0");
  int64_t n_syn = d.syn_off ? d.syn_off[d.n_cells] : 0;
  if (n_syn > 0 && (!d.syn_cv || !d.syn_tau || !d.syn_e)) return fail(ARB_E_NULL, "synapse arrays must not be NULL");
  if (d.n_clamp > 0 && (!d.clamp_cell || !d.clamp_cv || !d.clamp_t0 || !d.clamp_t1 || !d.clamp_amp)) return fail(ARB_E_NULL, "clamp arrays must not be NULL");
  if (d.n_conn > 0 && (!d.conn_src || !d.conn_dst || !d.conn_syn || !d.conn_delay || !d.conn_weight)) return fail(ARB_E_NULL, "connection arrays must not be NULL");
  if (d.n_ext > 0 && (!d.ext_cell || !d.ext_syn || !d.ext_time || !d.ext_weight)) return fail(ARB_E_NULL, "external event arrays must not be NULL");
  if ((d.n_conn > 0 || d.n_ext > 0) && !d.syn_off) return fail(ARB_E_INVALID, "connections / events need synapses");
  if (!finite(d.threshold) || (hh_any && (!finite(d.hh_ena) || !finite(d.hh_ek) || !finite(d.hh_el)))) return fail(ARB_E_INVALID, "non-finite scalar parameter");
  for (int64_t c = 0; c < d.n_cells; ++c) {
    if (d.cv_off[c + 1] <= d.cv_off[c]) return fail(ARB_E_INVALID, "cell " + std::to_string(c) + " has no compartments");
    if (d.syn_off && d.syn_off[c + 1] < d.syn_off[c]) return fail(ARB_E_INVALID, "syn_off is not monotone");
  }
  if (d.cv_off[d.n_cells] >= (int64_t)0xFFFF0000u) return fail(ARB_E_INVALID, "more than 2^32 compartments are not supported");
  std::atomic<int> bad(0);
  std::atomic<int64_t> bad_cell(-1);
  parallel_for(d.n_cells, [&](int64_t c) {
    if (bad.load(std::memory_order_relaxed)) return;
    int64_t a = d.cv_off[c], n = d.cv_off[c + 1] - a;
    int why = 0;
    for (int64_t i = 0; i < n && !why; ++i) {
      int32_t p = d.cv_parent[a + i];
      if ((i == 0 && p != -1) || (i > 0 && (p < 0 || p >= i))) why = 1;
      else if (!(d.cv_area[a + i] > 0) || !finite(d.cv_area[a + i]) || !(d.cv_cm[a + i] > 0) || !finite(d.cv_cm[a + i])) why = 2;
      else if (i > 0 && (!(d.cv_raxial[a + i] > 0) || !finite(d.cv_raxial[a + i]))) why = 3;
      else if (d.cv_vinit && !finite(d.cv_vinit[a + i])) why = 4;
      else if (hh_any && (!finite(d.hh_gnabar[a + i]) || !finite(d.hh_gkbar[a + i]) || !finite(d.hh_gl[a + i]))) why = 5;
      else if (d.pas_g && (!finite(d.pas_g[a + i]) || !finite(d.pas_e[a + i]))) why = 5;
    }
    if (!why && d.syn_off)
      for (int64_t s = d.syn_off[c]; s < d.syn_off[c + 1] && !why; ++s) {
        if (d.syn_cv[s] < 0 || d.syn_cv[s] >= n) why = 6;
        else if (!(d.syn_tau[s] > 0) || !finite(d.syn_tau[s]) || !finite(d.syn_e[s])) why = 7;
      }
    if (!why && d.det_cv && (d.det_cv[c] < 0 || d.det_cv[c] >= n)) why = 8;
    if (why) { bad.store(why); bad_cell.store(c); }
  });
  if (bad.load()) {
    static const char* msg[] = {"", "bad parent index (need -1 for CV 0, else 0 <= parent < index)", "area and cm must be finite and > 0",
                                "axial resistance must be finite and > 0", "non-finite vinit", "non-finite mechanism parameter",
                                "synapse CV out of range", "synapse tau must be > 0 and finite", "detector CV out of range"};
    return fail(ARB_E_INVALID, std::string(msg[bad.load()]) + " (cell " + std::to_string(bad_cell.load()) + ")");
  }
  for (int64_t k = 0; k < d.n_clamp; ++k) {
    int64_t c = d.clamp_cell[k];
    if (c < 0 || c >= d.n_cells || d.clamp_cv[k] < 0 || d.clamp_cv[k] >= d.cv_off[c + 1] - d.cv_off[c]) return fail(ARB_E_INVALID, "clamp cell / CV out of range");
    if (std::isnan(d.clamp_t0[k]) || std::isnan(d.clamp_t1[k]) || !finite(d.clamp_amp[k])) return fail(ARB_E_INVALID, "non-finite clamp parameter");
  }
  for (int64_t k = 0; k < d.n_conn; ++k) {
    int64_t s = d.conn_src[k], t = d.conn_dst[k];
    if (s < 0 || s >= d.n_cells || t < 0 || t >= d.n_cells) return fail(ARB_E_INVALID, "connection cell out of range");
    if (d.conn_syn[k] < 0 || d.conn_syn[k] >= d.syn_off[t + 1] - d.syn_off[t]) return fail(ARB_E_INVALID, "connection synapse out of range");
    if (!(d.conn_delay[k] > 0) || !finite(d.conn_delay[k])) return fail(ARB_E_INVALID, "connection delay must be > 0 and finite (PAPER.md:96)");
    if (!finite(d.conn_weight[k])) return fail(ARB_E_INVALID, "non-finite connection weight");
  }
  for (int64_t k = 0; k < d.n_ext; ++k) {
    int64_t c = d.ext_cell[k];
    if (c < 0 || c >= d.n_cells) return fail(ARB_E_INVALID, "external event cell out of range");
    if (d.ext_syn[k] < 0 || d.ext_syn[k] >= d.syn_off[c + 1] - d.syn_off[c]) return fail(ARB_E_INVALID, "external event synapse out of range");
    if (!(d.ext_time[k] >= 0) || !finite(d.ext_time[k]) || !finite(d.ext_weight[k])) return fail(ARB_E_INVALID, "external event earlier than t = 0 or non-finite");
  }
  return ARB_OK;
}

namespace {

// Everything about one block.  Called twice: counts only (plan), then with the pools to fill.
struct BlockBuilder {
  const arb_desc& d;
  const BuildParams& P;
  const HostModel& H;
  const std::vector<int64_t>& clamp_off;   // clamps grouped by caller's cell
  const std::vector<int64_t>& clamp_idx;

  std::vector<Lane> lanes;
  std::vector<uint32_t> cvs;               // CV lists of all lanes
  std::vector<uint32_t> nchild, br_of;
  std::vector<CellScratch> cells;

  void decompose(int64_t cell_begin, uint32_t n_cell) {
    lanes.clear(); cvs.clear(); cells.assign(n_cell, CellScratch());
    for (uint32_t lc = 0; lc < n_cell; ++lc) {
      int64_t orig = H.cell_order[cell_begin + lc];
      int64_t a = d.cv_off[orig];
      uint32_t n = (uint32_t)(d.cv_off[orig + 1] - a);
      const int32_t* par = d.cv_parent + a;
      nchild.assign(n, 0);
      br_of.assign(n, 0);
      for (uint32_t i = 1; i < n; ++i) nchild[par[i]]++;
      cells[lc].lane_begin = (uint32_t)lanes.size();
      // pass 1: branch id of every CV (parent < index, so one forward sweep suffices)
      const std::vector<uint32_t>& nch = nchild;
      uint32_t nb = 0;
      std::vector<uint32_t> blen;
      for (uint32_t i = 0; i < n; ++i) {
        bool fresh = (i == 0) || nch[par[i]] != 1 || blen[br_of[par[i]]] >= P.max_branch_len;
        if (fresh) {
          Lane L;
          L.lc = lc; L.br = nb; L.len = 0; L.first_cv = i;
          L.parent_br = (i == 0) ? -1 : (int32_t)br_of[par[i]];
          L.level = (i == 0) ? 0 : lanes[cells[lc].lane_begin + L.parent_br].level + 1;
          L.cv_begin = 0;
          lanes.push_back(L);
          blen.push_back(0);
          br_of[i] = nb++;
        } else {
          br_of[i] = br_of[par[i]];
        }
        blen[br_of[i]]++;
      }
      cells[lc].n_br = nb;
      // pass 2: CV lists, proximal -> distal (ascending index inside a branch)
      uint32_t base = (uint32_t)cvs.size();
      uint32_t acc = 0;
      for (uint32_t b = 0; b < nb; ++b) {
        Lane& L = lanes[cells[lc].lane_begin + b];
        L.len = blen[b];
        L.cv_begin = base + acc;
        acc += blen[b];
        blen[b] = 0;  // becomes the fill cursor
      }
      cvs.resize(base + n);
      for (uint32_t i = 0; i < n; ++i) {
        Lane& L = lanes[cells[lc].lane_begin + br_of[i]];
        cvs[L.cv_begin + blen[br_of[i]]++] = i;
      }
    }
  }

  // Builds block `b`.  When pools are given (fill), writes them; always returns the counts.
  BlockInfo run(int64_t cell_begin, uint32_t n_cell, const BlockInfo* placed, HostModel* out, int64_t hh_global) {
    decompose(cell_begin, n_cell);
    BlockInfo bi;
    std::memset(&bi, 0, sizeof bi);
    if (placed) bi = *placed;
    bi.cell_base = cell_begin;
    bi.n_cell = n_cell;
    const uint32_t n_lane = (uint32_t)lanes.size();
    // order of lanes inside the block: level, then longest first (sliced-ELL style padding)
    std::vector<uint32_t> order(n_lane);
    for (uint32_t i = 0; i < n_lane; ++i) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](uint32_t x, uint32_t y) {
      const Lane &A = lanes[x], &B = lanes[y];
      if (A.level != B.level) return A.level < B.level;
      if (A.len != B.len) return A.len > B.len;
      return x < y;
    });
    std::vector<uint32_t> tl_of(n_lane);   // unsorted lane -> block-local lane index
    for (uint32_t t = 0; t < n_lane; ++t) tl_of[order[t]] = t;
    std::vector<Task> tasks;
    std::vector<uint32_t> level_begin;
    uint32_t slot = 0, n_level = 0;
    for (uint32_t t = 0; t < n_lane;) {
      uint32_t lvl = lanes[order[t]].level;
      while (level_begin.size() <= lvl) level_begin.push_back((uint32_t)tasks.size());
      uint32_t e = t;
      while (e < n_lane && e - t < 32 && lanes[order[e]].level == lvl) ++e;
      Task T;
      T.slot_off = slot; T.lane_off = t; T.nlanes = (uint16_t)(e - t);
      T.width = (uint16_t)align_up(e - t, 4);
      T.maxlen = (uint16_t)lanes[order[t]].len; T.level = (uint16_t)lvl;
      slot += (uint32_t)T.maxlen * T.width;
      tasks.push_back(T);
      n_level = lvl + 1;
      t = e;
    }
    level_begin.push_back((uint32_t)tasks.size());
    bi.n_slot = align_up(slot, 16);
    bi.n_lane = n_lane;
    bi.n_task = (uint32_t)tasks.size();
    bi.n_level = n_level;
    // counts of mechanisms
    uint32_t n_hh = 0, n_syn = 0, n_clamp = 0, n_sp = 0, n_child = 0;
    for (uint32_t i = 0; i < n_lane; ++i) n_child += lanes[i].parent_br >= 0 ? 1 : 0;
    for (uint32_t lc = 0; lc < n_cell; ++lc) {
      int64_t orig = H.cell_order[cell_begin + lc];
      int64_t a = d.cv_off[orig];
      uint32_t n = (uint32_t)(d.cv_off[orig + 1] - a);
      std::vector<uint8_t> flag(n, 0);
      if (d.hh_gnabar)
        for (uint32_t i = 0; i < n; ++i)
          if (d.hh_gnabar[a + i] != 0.0 || d.hh_gkbar[a + i] != 0.0 || d.hh_gl[a + i] != 0.0) { flag[i] = 1; ++n_hh; }
      if (d.syn_off) {
        for (int64_t s = d.syn_off[orig]; s < d.syn_off[orig + 1]; ++s) flag[d.syn_cv[s]] = 1;
        n_syn += (uint32_t)(d.syn_off[orig + 1] - d.syn_off[orig]);
      }
      for (int64_t q = clamp_off[orig]; q < clamp_off[orig + 1]; ++q) flag[d.clamp_cv[clamp_idx[q]]] = 1;
      n_clamp += (uint32_t)(clamp_off[orig + 1] - clamp_off[orig]);
      for (uint32_t i = 0; i < n; ++i) n_sp += flag[i];
    }
    bi.n_hh = n_hh; bi.n_syn = n_syn; bi.n_clamp = n_clamp; bi.n_sp = n_sp; bi.n_child = n_child;
    MetaOff mo = meta_offsets(bi);
    bi.meta_bytes = mo.total;
    if (!out) return bi;

    // ------------------------------------------------------------------ fill
    FastOff fo = fast_offsets(bi);
    StateOff so = state_offsets(bi);
    GenOff go = gen_offsets(bi);
    double* gen = out->gen.data() + bi.gen_base;
    double* fast = out->fast.data() + bi.fast_base;
    double* st = out->state.data() + bi.state_base;
    uint8_t* meta = out->meta.data() + bi.meta_base;
    std::memcpy(meta + mo.tasks, tasks.data(), tasks.size() * sizeof(Task));
    std::memcpy(meta + mo.level_begin, level_begin.data(), level_begin.size() * 4);
    uint32_t* br_pslot = (uint32_t*)(meta + mo.br_pslot);
    uint32_t* br_cbeg = (uint32_t*)(meta + mo.br_cbeg);
    uint16_t* br_len = (uint16_t*)(meta + mo.br_len);
    uint16_t* br_cell = (uint16_t*)(meta + mo.br_cell);
    uint16_t* br_ccnt = (uint16_t*)(meta + mo.br_ccnt);
    uint32_t* child = (uint32_t*)(meta + mo.child);
    uint32_t* cell_det = (uint32_t*)(meta + mo.cell_det);
    uint32_t* hh_slot = (uint32_t*)(meta + mo.hh_slot);
    uint16_t* hh_cell = (uint16_t*)(meta + mo.hh_cell);
    uint16_t* syn_cell = (uint16_t*)(meta + mo.syn_cell);
    uint32_t* sp_slot = (uint32_t*)(meta + mo.sp_slot);
    int32_t* sp_hh = (int32_t*)(meta + mo.sp_hh);
    uint32_t* sp_syn_beg = (uint32_t*)(meta + mo.sp_syn_beg);
    uint32_t* sp_cl_beg = (uint32_t*)(meta + mo.sp_cl_beg);
    uint16_t* sp_syn_cnt = (uint16_t*)(meta + mo.sp_syn_cnt);
    uint16_t* sp_cl_cnt = (uint16_t*)(meta + mo.sp_cl_cnt);
    uint16_t* sp_cell = (uint16_t*)(meta + mo.sp_cell);

    // slot of lane t, position k
    std::vector<uint32_t> task_of(n_lane);
    for (uint32_t ti = 0; ti < tasks.size(); ++ti)
      for (uint32_t l = 0; l < tasks[ti].nlanes; ++l) task_of[tasks[ti].lane_off + l] = ti;
    auto slot_of = [&](uint32_t tl, uint32_t k) {
      const Task& T = tasks[task_of[tl]];
      return T.slot_off + k * (uint32_t)T.width + (tl - T.lane_off);
    };
    // children lists: for each parent lane, its child lanes in DESCENDING first-CV order (the
    // order in which a leaves->root elimination meets them)
    std::vector<std::vector<uint32_t>> kids(n_lane);
    for (uint32_t i = 0; i < n_lane; ++i)
      if (lanes[i].parent_br >= 0) kids[cells[lanes[i].lc].lane_begin + lanes[i].parent_br].push_back(i);
    uint32_t cpos = 0;
    for (uint32_t i = 0; i < n_lane; ++i) {
      uint32_t tl = tl_of[i];
      const Lane& L = lanes[i];
      br_len[tl] = (uint16_t)L.len;
      br_cell[tl] = (uint16_t)L.lc;
      if (L.parent_br >= 0) {
        uint32_t pi = cells[L.lc].lane_begin + L.parent_br;
        br_pslot[tl] = slot_of(tl_of[pi], lanes[pi].len - 1);
      } else {
        br_pslot[tl] = kNoSlot;
      }
      std::sort(kids[i].begin(), kids[i].end(), [&](uint32_t x, uint32_t y) { return lanes[x].first_cv > lanes[y].first_cv; });
      br_cbeg[tl] = cpos;
      br_ccnt[tl] = (uint16_t)kids[i].size();
      for (uint32_t k : kids[i]) child[cpos++] = tl_of[k];
    }
    // per CV: slot, constants, initial state
    uint32_t hh_pos = 0, syn_pos = 0, cl_pos = 0, sp_pos = 0;
    for (uint32_t lc = 0; lc < n_cell; ++lc) {
      int64_t orig = H.cell_order[cell_begin + lc];
      int64_t a = d.cv_off[orig];
      uint32_t n = (uint32_t)(d.cv_off[orig + 1] - a);
      const int32_t* par = d.cv_parent + a;
      std::vector<uint32_t> cv_slot(n);
      for (uint32_t b2 = 0; b2 < cells[lc].n_br; ++b2) {
        const Lane& L = lanes[cells[lc].lane_begin + b2];
        uint32_t tl = tl_of[cells[lc].lane_begin + b2];
        for (uint32_t k = 0; k < L.len; ++k) cv_slot[cvs[L.cv_begin + k]] = slot_of(tl, k);
      }
      std::vector<double> S(n, 0.0);
      for (uint32_t i = 1; i < n; ++i) S[i] = 1.0 / d.cv_raxial[a + i];
      for (uint32_t i = 1; i < n; ++i) S[par[i]] += 1.0 / d.cv_raxial[a + i];   // ascending child order
      for (uint32_t i = 0; i < n; ++i) {
        uint32_t s = cv_slot[i];
        double area = d.cv_area[a + i];
        gen[go.C + s] = d.cv_cm[a + i] * area * 1e-5;                 // nF
        gen[go.S + s] = S[i];                                         // uS
        gen[go.sig + s] = i ? 1.0 / d.cv_raxial[a + i] : 0.0;         // uS
        double G = d.pas_g ? d.pas_g[a + i] * area * 1e-2 : 0.0;      // uS
        gen[go.G + s] = G;
        gen[go.b + s] = d.pas_g ? G * d.pas_e[a + i] : 0.0;           // nA
        st[so.v + s] = d.cv_vinit ? d.cv_vinit[a + i] : -65.0;
        out->cv_state_idx[a + i] = (uint32_t)(bi.state_base + so.v + s);
      }
      cell_det[lc] = cv_slot[d.det_cv ? d.det_cv[orig] : 0];
      // mechanisms, grouped per CV in ascending CV order; synapses and clamps ascending inside a CV
      std::vector<std::vector<int64_t>> syn_on(n), cl_on(n);
      if (d.syn_off)
        for (int64_t s = d.syn_off[orig]; s < d.syn_off[orig + 1]; ++s) syn_on[d.syn_cv[s]].push_back(s);
      for (int64_t q = clamp_off[orig]; q < clamp_off[orig + 1]; ++q) cl_on[d.clamp_cv[clamp_idx[q]]].push_back(clamp_idx[q]);
      for (uint32_t i = 0; i < n; ++i) {
        bool hh = d.hh_gnabar && (d.hh_gnabar[a + i] != 0.0 || d.hh_gkbar[a + i] != 0.0 || d.hh_gl[a + i] != 0.0);
        if (!hh && syn_on[i].empty() && cl_on[i].empty()) continue;
        sp_slot[sp_pos] = cv_slot[i];
        sp_cell[sp_pos] = (uint16_t)lc;
        sp_hh[sp_pos] = hh ? (int32_t)hh_pos : -1;
        if (hh) {
          double sc = d.cv_area[a + i] * 1e-2;
          fast[fo.hh_gna + hh_pos] = d.hh_gnabar[a + i] * sc;
          fast[fo.hh_gk + hh_pos] = d.hh_gkbar[a + i] * sc;
          fast[fo.hh_gl + hh_pos] = d.hh_gl[a + i] * sc;
          hh_slot[hh_pos] = cv_slot[i];
          hh_cell[hh_pos] = (uint16_t)lc;
          out->hh_m_idx[hh_global + hh_pos] = (uint32_t)(bi.state_base + so.m + hh_pos);
          out->hh_stride[hh_global + hh_pos] = so.h - so.m;
          out->hh_cv[hh_global + hh_pos] = (uint32_t)(a + i);
          ++hh_pos;
        }
        sp_syn_beg[sp_pos] = syn_pos;
        sp_syn_cnt[sp_pos] = (uint16_t)std::min<size_t>(syn_on[i].size(), 65535);
        for (int64_t s : syn_on[i]) {
          fast[fo.syn_e + syn_pos] = d.syn_e[s];
          fast[fo.syn_tau + syn_pos] = d.syn_tau[s];
          syn_cell[syn_pos] = (uint16_t)lc;
          out->syn_state_idx[s] = (uint32_t)(bi.state_base + so.g + syn_pos);
          ++syn_pos;
        }
        sp_cl_beg[sp_pos] = cl_pos;
        sp_cl_cnt[sp_pos] = (uint16_t)std::min<size_t>(cl_on[i].size(), 65535);
        for (int64_t k : cl_on[i]) {
          fast[fo.cl_t0 + cl_pos] = d.clamp_t0[k];
          fast[fo.cl_t1 + cl_pos] = d.clamp_t1[k];
          fast[fo.cl_amp + cl_pos] = d.clamp_amp[k];
          ++cl_pos;
        }
        ++sp_pos;
      }
    }
    return bi;
  }
};

}  // namespace

int build(const arb_desc& d, const BuildParams& P, bool fill, HostModel& H, std::string& err) {
  int rc = validate(d, err);
  if (rc) return rc;
  H = HostModel();
  H.n_cells = d.n_cells;
  H.n_cv = d.cv_off[d.n_cells];
  H.n_syn = d.syn_off ? d.syn_off[d.n_cells] : 0;
  H.n_clamp = d.n_clamp; H.n_conn = d.n_conn; H.n_ext = d.n_ext;
  H.ena = d.hh_ena; H.ek = d.hh_ek; H.el = d.hh_el; H.threshold = d.threshold;
  const int64_t nc = d.n_cells;
  // synapses / clamps on one CV are counted in 16 bits
  // internal cell order: identity for homogeneous networks, else big cells first (load balance)
  H.cell_order.resize(nc);
  for (int64_t c = 0; c < nc; ++c) H.cell_order[c] = (uint32_t)c;
  bool homogeneous = true;
  int64_t n0 = d.cv_off[1] - d.cv_off[0];
  for (int64_t c = 1; c < nc && homogeneous; ++c) homogeneous = (d.cv_off[c + 1] - d.cv_off[c]) == n0;
  if (!homogeneous)
    std::stable_sort(H.cell_order.begin(), H.cell_order.end(), [&](uint32_t x, uint32_t y) {
      return d.cv_off[x + 1] - d.cv_off[x] > d.cv_off[y + 1] - d.cv_off[y];
    });
  H.cell_internal.resize(nc);
  for (int64_t i = 0; i < nc; ++i) H.cell_internal[H.cell_order[i]] = (uint32_t)i;
  // partition into blocks
  std::vector<int64_t> blk_begin;
  {
    int64_t cvs = 0; uint32_t cells = 0;
    for (int64_t i = 0; i < nc; ++i) {
      int64_t n = d.cv_off[H.cell_order[i] + 1] - d.cv_off[H.cell_order[i]];
      if (cells == 0 || cvs + n > P.target_slots || cells >= P.max_cells) { blk_begin.push_back(i); cvs = 0; cells = 0; }
      cvs += n; ++cells;
    }
    blk_begin.push_back(nc);
  }
  H.n_blocks = (int64_t)blk_begin.size() - 1;
  H.blocks.resize(H.n_blocks);
  H.cell_block.resize(nc);
  // clamps grouped by cell
  std::vector<int64_t> clamp_off(nc + 1, 0), clamp_idx(d.n_clamp);
  for (int64_t k = 0; k < d.n_clamp; ++k) clamp_off[d.clamp_cell[k] + 1]++;
  for (int64_t c = 0; c < nc; ++c) clamp_off[c + 1] += clamp_off[c];
  {
    std::vector<int64_t> cur(clamp_off.begin(), clamp_off.end() - 1);
    for (int64_t k = 0; k < d.n_clamp; ++k) clamp_idx[cur[d.clamp_cell[k]]++] = k;
  }
  // pass 1: counts
  std::atomic<int> too_many(0);
  parallel_for(H.n_blocks, [&](int64_t b) {
    BlockBuilder B{d, P, H, clamp_off, clamp_idx, {}, {}, {}, {}, {}};
    H.blocks[b] = B.run(blk_begin[b], (uint32_t)(blk_begin[b + 1] - blk_begin[b]), nullptr, nullptr, 0);
    for (int64_t i = blk_begin[b]; i < blk_begin[b + 1]; ++i) H.cell_block[i] = (uint32_t)b;
    if (H.blocks[b].n_level > 60000 || H.blocks[b].n_slot > 0x7FFFFFFFu) too_many.store(1);
  });
  if (too_many.load()) { err = "a cell is too deep or too large for the block layout"; return ARB_E_INVALID; }
  // placement
  std::vector<uint32_t> hh_first(H.n_blocks);
  for (int64_t b = 0; b < H.n_blocks; ++b) {
    BlockInfo& bi = H.blocks[b];
    bi.gen_base = H.gen_doubles;     H.gen_doubles += gen_offsets(bi).total;
    bi.fast_base = H.fast_doubles;   H.fast_doubles += fast_offsets(bi).total;
    bi.state_base = H.state_doubles; H.state_doubles += state_offsets(bi).total;
    bi.meta_base = H.meta_bytes;     H.meta_bytes += align_up(bi.meta_bytes, 128);
    bi.scratch_base = H.scratch_doubles; H.scratch_doubles += 2 * (int64_t)bi.n_slot + 2 * align_up(bi.n_lane, 16);
    hh_first[b] = (uint32_t)H.n_hh;  H.n_hh += bi.n_hh;
    H.n_lanes += bi.n_lane;
    H.max_block_slots = std::max(H.max_block_slots, bi.n_slot);
    H.max_block_lanes = std::max(H.max_block_lanes, bi.n_lane);
    H.max_block_cells = std::max(H.max_block_cells, bi.n_cell);
  }
  if (H.state_doubles >= (int64_t)0xFFFFFFF0u) { err = "state pool exceeds 2^32 doubles"; return ARB_E_INVALID; }
  // delays
  H.min_delay = std::numeric_limits<double>::infinity();
  H.max_delay = 0;
  for (int64_t k = 0; k < d.n_conn; ++k) { H.min_delay = std::min(H.min_delay, d.conn_delay[k]); H.max_delay = std::max(H.max_delay, d.conn_delay[k]); }
  if (!fill) return ARB_OK;

  // pass 2: fill
  H.gen.assign(H.gen_doubles, 0.0);
  H.fast.assign(H.fast_doubles, 0.0);
  H.state.assign(H.state_doubles, 0.0);
  H.meta.assign(H.meta_bytes, 0);
  H.cv_state_idx.resize(H.n_cv);
  H.syn_state_idx.resize(H.n_syn);
  H.hh_m_idx.resize(H.n_hh); H.hh_stride.resize(H.n_hh); H.hh_cv.resize(H.n_hh);
  parallel_for(H.n_blocks, [&](int64_t b) {
    BlockBuilder B{d, P, H, clamp_off, clamp_idx, {}, {}, {}, {}, {}};
    BlockInfo placed = H.blocks[b];
    B.run(blk_begin[b], (uint32_t)(blk_begin[b + 1] - blk_begin[b]), &placed, &H, hh_first[b]);
  });
  // connections grouped by caller's source cell, ascending k inside a group
  H.conn_off.assign(nc + 1, 0);
  for (int64_t k = 0; k < d.n_conn; ++k) H.conn_off[d.conn_src[k] + 1]++;
  for (int64_t c = 0; c < nc; ++c) H.conn_off[c + 1] += H.conn_off[c];
  H.conn_dst.resize(d.n_conn); H.conn_gidx.resize(d.n_conn); H.conn_delay.resize(d.n_conn); H.conn_w.resize(d.n_conn);
  {
    std::vector<uint32_t> cur(H.conn_off.begin(), H.conn_off.end() - 1);
    for (int64_t k = 0; k < d.n_conn; ++k) {
      uint32_t p = cur[d.conn_src[k]]++;
      H.conn_dst[p] = H.cell_internal[d.conn_dst[k]];
      H.conn_gidx[p] = H.syn_state_idx[d.syn_off[d.conn_dst[k]] + d.conn_syn[k]];
      H.conn_delay[p] = d.conn_delay[k];
      H.conn_w[p] = d.conn_weight[k];
    }
  }
  // external events grouped by internal cell, sorted by (time, synapse, weight)
  H.ext_off.assign(nc + 1, 0);
  for (int64_t k = 0; k < d.n_ext; ++k) H.ext_off[H.cell_internal[d.ext_cell[k]] + 1]++;
  for (int64_t c = 0; c < nc; ++c) H.ext_off[c + 1] += H.ext_off[c];
  H.ext_t.resize(d.n_ext); H.ext_gidx.resize(d.n_ext); H.ext_w.resize(d.n_ext);
  {
    std::vector<int64_t> idx(d.n_ext);
    std::vector<uint32_t> cur(H.ext_off.begin(), H.ext_off.end() - 1);
    for (int64_t k = 0; k < d.n_ext; ++k) idx[cur[H.cell_internal[d.ext_cell[k]]]++] = k;
    parallel_for(nc, [&](int64_t c) {
      auto b = idx.begin() + H.ext_off[c], e = idx.begin() + H.ext_off[c + 1];
      std::sort(b, e, [&](int64_t x, int64_t y) {
        if (d.ext_time[x] != d.ext_time[y]) return d.ext_time[x] < d.ext_time[y];
        if (d.ext_syn[x] != d.ext_syn[y]) return d.ext_syn[x] < d.ext_syn[y];
        return x < y;
      });
    });
    for (int64_t p = 0; p < d.n_ext; ++p) {
      int64_t k = idx[p];
      H.ext_t[p] = d.ext_time[k];
      H.ext_gidx[p] = H.syn_state_idx[d.syn_off[d.ext_cell[k]] + d.ext_syn[k]];
      H.ext_w[p] = d.ext_weight[k];
    }
  }
  return ARB_OK;
}

}  // namespace arbb
