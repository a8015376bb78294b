// layout.cpp - see layout.hpp.  Host preprocessing only; nothing here runs per time step.
#include "layout.hpp"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstring>
#include <limits>
#include <thread>
#include <unordered_map>

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

uint64_t fnv1a(const uint8_t* p, size_t n) {
  uint64_t h = 1469598103934665603ull;
  for (size_t i = 0; i < n; ++i) { h ^= p[i]; h *= 1099511628211ull; }
  return h;
}

}  // namespace

int validate(const arb_desc& d, std::string& err) {
  auto fail = [&](int code, const std::string& s) { err = s; return code; };
  if (d.n_cells < 0 || d.n_clamp < 0 || d.n_conn < 0 || d.n_ext < 0) return fail(ARB_E_INVALID, "negative count");
  if (d.shard_n_global < 0 || d.shard_gid_base < 0 || (d.shard_n_global > 0 && d.shard_gid_base + d.n_cells > d.shard_n_global))
    return fail(ARB_E_INVALID, "shard_gid_base / shard_n_global do not describe a range of the network");
  if (d.shard_n_global >= (int64_t)0x7FFFFFFF) return fail(ARB_E_INVALID, "more than 2^31 cells are not supported");
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
  if (d.cell_kind) {
    if (!d.lif_tau_m || !d.lif_v_th || !d.lif_c_m || !d.lif_e_l || !d.lif_e_r || !d.lif_t_ref || !d.src_off || (d.src_off[d.n_cells] > 0 && !d.src_time))
      return fail(ARB_E_NULL, "cell_kind needs the lif_* arrays and src_off / src_time");
    if (d.src_off[0] != 0) return fail(ARB_E_INVALID, "src_off[0] must be 0");
    for (int64_t c = 0; c < d.n_cells; ++c) {
      const int32_t kd = d.cell_kind[c];
      if (kd < 0 || kd > 2) return fail(ARB_E_INVALID, "cell_kind must be 0, 1 or 2");
      if (d.src_off[c + 1] < d.src_off[c]) return fail(ARB_E_INVALID, "src_off is not monotone");
      if (kd != 0 && d.cv_off[c + 1] - d.cv_off[c] != 1) return fail(ARB_E_INVALID, "a LIF / source cell owns exactly one control volume");
      if (kd == 1 && (!(d.lif_tau_m[c] > 0) || !finite(d.lif_tau_m[c]) || !(d.lif_c_m[c] > 0) || !finite(d.lif_c_m[c]) || !(d.lif_t_ref[c] >= 0) ||
                      !finite(d.lif_t_ref[c]) || !finite(d.lif_v_th[c]) || !finite(d.lif_e_l[c]) || !finite(d.lif_e_r[c]) || !(d.lif_e_r[c] < d.lif_v_th[c])))
        return fail(ARB_E_INVALID, "bad LIF parameters (cell " + std::to_string(c) + ")");
      for (int64_t q = d.src_off[c]; q < d.src_off[c + 1]; ++q)
        if (!(d.src_time[q] >= 0) || !finite(d.src_time[q]) || (q > d.src_off[c] && d.src_time[q] < d.src_time[q - 1]))
          return fail(ARB_E_INVALID, "a spike schedule must be finite, >= 0 and ascending");
    }
    if (d.src_off[d.n_cells] >= (int64_t)0xFFFFFFF0u) return fail(ARB_E_INVALID, "more than 2^32 scheduled spikes are not supported");
  }
  for (int64_t k = 0; k < d.n_clamp; ++k) {
    int64_t c = d.clamp_cell[k];
    if (c < 0 || c >= d.n_cells || d.clamp_cv[k] < 0 || d.clamp_cv[k] >= d.cv_off[c + 1] - d.cv_off[c]) return fail(ARB_E_INVALID, "clamp cell / CV out of range");
    if (std::isnan(d.clamp_t0[k]) || std::isnan(d.clamp_t1[k]) || !finite(d.clamp_amp[k])) return fail(ARB_E_INVALID, "non-finite clamp parameter");
  }
  for (int64_t k = 0; k < d.n_conn; ++k) {
    int64_t s = d.conn_src[k], t = d.conn_dst[k];
    const int64_t n_src = d.shard_n_global > 0 ? d.shard_n_global : d.n_cells;
    if (s < 0 || s >= n_src || t < 0 || t >= d.n_cells) return fail(ARB_E_INVALID, "connection cell out of range");
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

// Everything about one unit.  Called twice: counts + topo record (plan), then with the pools to fill.
struct UnitBuilder {
  const arb_desc& d;
  const BuildParams& P;
  const HostModel& H;
  const std::vector<int64_t>& clamp_off;   // clamps grouped by caller's cell
  const std::vector<int64_t>& clamp_idx;

  std::vector<Lane> lanes;
  std::vector<uint32_t> cvs;               // CV lists of all lanes
  std::vector<uint32_t> nchild, br_of, blen;
  std::vector<CellScratch> cells;
  // layout of the unit
  std::vector<uint32_t> order, tl_of, task_of, row_begin, rowoff;
  std::vector<Task> tasks;
  std::vector<uint32_t> level_begin;
  bool bad = false;                        // a count does not fit its field
  // forests (forest_layout.h)
  bool forest = false, warp_cells = false;
  int n_warp = kForestWarps;               // warps that sweep the forest (kForestWarps or kForestWarpsBig)
  std::vector<uint32_t> fslot0, flevel_br;
  std::vector<FRun> fruns;
  std::vector<FChunk> fchunks;
  std::vector<uint64_t> fchunk_cells;

  bool has_hh(int64_t gi) const {
    return d.hh_gnabar && (d.hh_gnabar[gi] != 0.0 || d.hh_gkbar[gi] != 0.0 || d.hh_gl[gi] != 0.0);
  }

  void decompose(int64_t cell_begin, uint32_t n_cell) {
    lanes.clear(); cvs.clear(); cells.assign(n_cell, CellScratch());
    for (uint32_t lc = 0; lc < n_cell; ++lc) {
      int64_t orig = H.cell_order[cell_begin + lc];
      int64_t a = d.cv_off[orig];
      uint32_t n = (uint32_t)(d.cv_off[orig + 1] - a);
      const int32_t* par = d.cv_parent + a;
      nchild.assign(n, 0);
      br_of.assign(n, 0);
      blen.clear();
      for (uint32_t i = 1; i < n; ++i) nchild[par[i]]++;
      cells[lc].lane_begin = (uint32_t)lanes.size();
      // pass 1: branch id of every CV (parent < index, so one forward sweep suffices)
      uint32_t nb = 0;
      for (uint32_t i = 0; i < n; ++i) {
        bool fresh = (i == 0) || nchild[par[i]] != 1 || blen[br_of[par[i]]] >= (forest ? kForestMaxBranchLen : P.max_branch_len);
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

  // tasks and ragged rows (unit_layout.h)
  uint32_t make_tasks() {
    const uint32_t n_lane = (uint32_t)lanes.size();
    order.resize(n_lane);
    for (uint32_t i = 0; i < n_lane; ++i) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](uint32_t x, uint32_t y) {
      const Lane &A = lanes[x], &B = lanes[y];
      if (A.level != B.level) return A.level < B.level;
      if (A.len != B.len) return A.len > B.len;
      return x < y;
    });
    tl_of.resize(n_lane);
    for (uint32_t t = 0; t < n_lane; ++t) tl_of[order[t]] = t;
    tasks.clear(); level_begin.clear(); row_begin.clear(); rowoff.clear();
    task_of.resize(n_lane);
    uint32_t slot = 0;
    for (uint32_t t = 0; t < n_lane;) {
      uint32_t lvl = lanes[order[t]].level;
      while (level_begin.size() <= lvl) level_begin.push_back((uint32_t)tasks.size());
      uint32_t e = t;
      while (e < n_lane && e - t < 32 && lanes[order[e]].level == lvl) ++e;
      Task T;
      T.slot_off = slot; T.lane_off = t; T.nlanes = (uint16_t)(e - t);
      const uint32_t maxlen = lanes[order[t]].len;
      T.maxlen_full = (uint16_t)(maxlen | (lanes[order[e - 1]].len == maxlen ? kTaskFull : 0));
      row_begin.push_back((uint32_t)rowoff.size());
      uint32_t acc = 0;
      for (uint32_t k = 0; k < maxlen; ++k) {
        rowoff.push_back(acc);
        uint32_t cnt = 0;
        for (uint32_t l = t; l < e; ++l) cnt += lanes[order[l]].len > k;
        acc += cnt;
      }
      T.nslots = acc;
      for (uint32_t l = t; l < e; ++l) task_of[l] = (uint32_t)tasks.size();
      slot += acc;
      tasks.push_back(T);
      t = e;
    }
    level_begin.push_back((uint32_t)tasks.size());
    return slot;
  }

  // forest: slot order level -> warp -> branch -> control volume; runs, chunks (forest_layout.h)
  uint32_t make_forest() {
    const uint32_t n_lane = (uint32_t)lanes.size();
    uint32_t n_level = 0;
    for (const Lane& L : lanes) n_level = std::max(n_level, L.level + 1);
    std::vector<std::vector<uint32_t>> by_level(n_level);
    for (uint32_t i = 0; i < n_lane; ++i) by_level[lanes[i].level].push_back(i);
    order.clear(); fslot0.clear(); flevel_br.clear(); fchunks.clear(); fchunk_cells.clear();
    // many cells: whole cells are dealt to the warps (largest first to the least loaded warp)
    warp_cells = cells.size() >= kForestWarpCellsMin;
    std::vector<uint32_t> cell_warp(cells.size(), 0);
    if (warp_cells) {
      std::vector<uint64_t> ccv(cells.size(), 0);
      for (const Lane& L : lanes) ccv[L.lc] += L.len;
      std::vector<uint32_t> by_size(cells.size());
      for (uint32_t c = 0; c < cells.size(); ++c) by_size[c] = c;
      std::stable_sort(by_size.begin(), by_size.end(), [&](uint32_t x, uint32_t y) { return ccv[x] > ccv[y]; });
      uint64_t wl[kForestMaxWarps] = {0};
      for (uint32_t c : by_size) {
        int best = 0;
        for (int w = 1; w < n_warp; ++w) if (wl[w] < wl[best]) best = w;
        cell_warp[c] = (uint32_t)best;
        wl[best] += ccv[c];
      }
    }
    fruns.assign((size_t)n_level * n_warp, FRun{0, 0});
    uint32_t slot = 0;
    for (uint32_t lvl = 0; lvl < n_level; ++lvl) {
      flevel_br.push_back((uint32_t)order.size());
      auto& v = by_level[lvl];
      std::stable_sort(v.begin(), v.end(), [&](uint32_t x, uint32_t y) { return lanes[x].len > lanes[y].len; });
      std::vector<uint32_t> dealt[kForestMaxWarps];
      uint64_t load[kForestMaxWarps] = {0};
      for (uint32_t i : v) {               // longest first onto the least loaded warp - or to the warp that owns the cell
        int best = 0;
        if (warp_cells) best = (int)cell_warp[lanes[i].lc];
        else for (int w = 1; w < n_warp; ++w) if (load[w] < load[best]) best = w;
        dealt[best].push_back(i);
        load[best] += lanes[i].len;
      }
      for (int w = 0; w < n_warp; ++w) {
        // branches of one cell next to each other: a pass in which few cells are active skips whole chunks
        std::stable_sort(dealt[w].begin(), dealt[w].end(), [&](uint32_t x, uint32_t y) { return lanes[x].lc < lanes[y].lc; });
        FRun& R = fruns[(size_t)lvl * n_warp + w];
        R.chunk_beg = (uint32_t)fchunks.size();
        const uint32_t pos0 = (uint32_t)order.size(), slot_beg = slot;
        for (uint32_t i : dealt[w]) { order.push_back(i); fslot0.push_back(slot); slot += lanes[i].len; }
        uint32_t pos = pos0;               // branch that holds the current slot
        for (uint32_t c0 = slot_beg; c0 < slot; c0 += 32) {
          FChunk ck;
          const uint32_t n = std::min(32u, slot - c0);
          while (fslot0[pos] + lanes[order[pos]].len <= c0) ++pos;
          ck.slot0 = c0; ck.heads = 0; ck.tails = 0; ck.br_n = pos * 64u + n;
          uint32_t q = pos;
          uint64_t cellmask = 0;
          for (uint32_t l = 0; l < 32; ++l) {
            if (l >= n) { ck.heads |= 1u << l; ck.tails |= 1u << l; continue; }
            const uint32_t sl = c0 + l;
            while (fslot0[q] + lanes[order[q]].len <= sl) ++q;
            cellmask |= 1ull << lanes[order[q]].lc;
            if (sl == fslot0[q]) ck.heads |= 1u << l;
            if (sl == fslot0[q] + lanes[order[q]].len - 1) ck.tails |= 1u << l;
          }
          fchunks.push_back(ck);
          fchunk_cells.push_back(cellmask);
        }
        R.chunk_end = (uint32_t)fchunks.size();
      }
    }
    flevel_br.push_back((uint32_t)order.size());
    tl_of.resize(n_lane);
    for (uint32_t t = 0; t < n_lane; ++t) tl_of[order[t]] = t;
    if (n_lane >= (1u << 26)) bad = true;  // FChunk::br_n
    return slot;
  }

  uint32_t slot_of(uint32_t tl, uint32_t k) const {
    if (forest) return fslot0[tl] + k;
    const uint32_t ti = task_of[tl];
    return tasks[ti].slot_off + rowoff[row_begin[ti] + k] + (tl - tasks[ti].lane_off);
  }

  UnitCounts run(int64_t cell_begin, uint32_t n_cell, std::vector<uint8_t>* topo_out, const UnitCounts* placed, HostModel* out) {
    decompose(cell_begin, n_cell);
    UnitCounts uc;
    if (placed) uc = *placed;
    uc.cell_base = cell_begin;
    uc.n_cell = n_cell;
    const uint32_t n_lane = (uint32_t)lanes.size();
    uc.n_cv = forest ? make_forest() : make_tasks();
    uc.n_slot = align_up(uc.n_cv, 2);
    uc.n_lane = n_lane;
    uc.n_task = forest ? (uint32_t)fchunks.size() : (uint32_t)tasks.size();
    uc.n_level = forest ? (uint32_t)flevel_br.size() - 1 : (uint32_t)level_begin.size() - 1;
    uint32_t n_hh = 0, n_syn = 0, n_clamp = 0, n_child = 0;
    for (uint32_t i = 0; i < n_lane; ++i) n_child += lanes[i].parent_br >= 0 ? 1 : 0;
    for (uint32_t lc = 0; lc < n_cell; ++lc) {
      int64_t orig = H.cell_order[cell_begin + lc];
      int64_t a = d.cv_off[orig];
      uint32_t n = (uint32_t)(d.cv_off[orig + 1] - a);
      for (uint32_t i = 0; i < n; ++i) n_hh += has_hh(a + i);
      if (d.syn_off) n_syn += (uint32_t)(d.syn_off[orig + 1] - d.syn_off[orig]);
      n_clamp += (uint32_t)(clamp_off[orig + 1] - clamp_off[orig]);
    }
    uc.n_hh = n_hh; uc.n_syn = n_syn; uc.n_clamp = n_clamp; uc.n_child = n_child;
    const FastOff fo = fast_offsets(uc.n_slot, n_hh, n_syn, n_clamp, n_cell, H.syn_uniform);
    const StateOff so = state_offsets(uc.n_slot, n_hh, n_syn, n_cell);
    uc.fast_bytes = fo.total;
    uc.state_bytes = 8 * so.total;

    // children lists: for each parent lane, its child lanes in DESCENDING first-CV order (the order
    // in which a leaves->root elimination meets them)
    std::vector<std::vector<uint32_t>> kids(n_lane);
    for (uint32_t i = 0; i < n_lane; ++i)
      if (lanes[i].parent_br >= 0) kids[cells[lanes[i].lc].lane_begin + lanes[i].parent_br].push_back(i);

    if (forest && !placed) {
      // does any control volume carry two kinds of point mechanism?  (their currents are then subtracted in turn)
      bool disjoint = true;
      std::vector<uint8_t> kind;
      for (uint32_t lc = 0; lc < n_cell && disjoint; ++lc) {
        const int64_t orig = H.cell_order[cell_begin + lc];
        const int64_t a0 = d.cv_off[orig];
        kind.assign((size_t)(d.cv_off[orig + 1] - a0), 0);
        for (size_t i = 0; i < kind.size(); ++i) if (has_hh(a0 + (int64_t)i)) kind[i] |= 1;
        if (d.syn_off) for (int64_t q = d.syn_off[orig]; q < d.syn_off[orig + 1]; ++q) kind[d.syn_cv[q]] |= 2;
        for (int64_t q = clamp_off[orig]; q < clamp_off[orig + 1]; ++q) kind[d.clamp_cv[clamp_idx[q]]] |= 4;
        for (uint8_t k : kind) if (k & (k - 1)) disjoint = false;
      }
      uc.flags |= UNIT_FOREST | (disjoint ? UNIT_POINT_DISJOINT : 0u) | (warp_cells ? UNIT_WARP_CELLS : 0u);
    }
    if (topo_out && forest) {
      const FTopoOff to = ftopo_offsets(uc.n_level, uc.n_task, n_lane, n_child, n_cell, (uint32_t)n_warp);
      topo_out->assign(to.total, 0);
      uint8_t* tp = topo_out->data();
      {
        FOffs fo2;
        std::memset(&fo2, 0, sizeof fo2);
        const uint32_t fv[18] = {fo.f, fo.invd, fo.a, fo.b, fo.hh_gna, fo.hh_gk, fo.hh_gl, fo.syn_e, fo.syn_decay, fo.cl_t0, fo.cl_t1,
                                 fo.cl_amp, fo.hh_slot, fo.syn_slot, fo.cl_slot, fo.hh_cell, fo.syn_cell, fo.cl_cell};
        std::memcpy(fo2.fast, fv, sizeof fv);
        const uint32_t sv[6] = {so.v, so.m, so.h, so.n, so.g, so.rt};
        std::memcpy(fo2.state, sv, sizeof sv);
        const GenOff go2 = gen_offsets(uc.n_slot, n_syn);
        const uint32_t gv[6] = {go2.C, go2.S, go2.sig, go2.G, go2.b, go2.syn_tau};
        std::memcpy(fo2.gen, gv, sizeof gv);
        const uint32_t tv[8] = {to.runs, to.chunks, to.chunk_cells, to.branches, to.br_cell, to.child, to.cell_det, to.level_br};
        std::memcpy(fo2.topo, tv, sizeof tv);
        const FScratchOff sc2 = fscratch_offsets(uc.n_slot, n_lane);
        const uint32_t cv2[3] = {sc2.fgen, sc2.invdgen, sc2.dcon};
        std::memcpy(fo2.scratch, cv2, sizeof cv2);
        std::memcpy(tp + to.offs, &fo2, sizeof fo2);
      }
      std::memcpy(tp + to.runs, fruns.data(), fruns.size() * sizeof(FRun));
      std::memcpy(tp + to.chunks, fchunks.data(), fchunks.size() * sizeof(FChunk));
      std::memcpy(tp + to.chunk_cells, fchunk_cells.data(), fchunk_cells.size() * 8);
      std::memcpy(tp + to.level_br, flevel_br.data(), flevel_br.size() * 4);
      FBranch* brec = (FBranch*)(tp + to.branches);
      uint16_t* br_cell = (uint16_t*)(tp + to.br_cell);
      uint32_t* child = (uint32_t*)(tp + to.child);
      uint32_t* cell_det = (uint32_t*)(tp + to.cell_det);
      uint32_t cpos = 0;
      for (uint32_t tl = 0; tl < n_lane; ++tl) {       // in slot order
        const uint32_t i = order[tl];
        const Lane& L = lanes[i];
        FBranch& R = brec[tl];
        R.slot0 = fslot0[tl];
        R.len = (uint16_t)L.len;
        br_cell[tl] = (uint16_t)L.lc;
        if (L.parent_br >= 0) {
          const uint32_t pi = cells[L.lc].lane_begin + L.parent_br;
          R.pslot = slot_of(tl_of[pi], lanes[pi].len - 1);
        } else {
          R.pslot = kNoSlot;
        }
        std::sort(kids[i].begin(), kids[i].end(), [&](uint32_t x, uint32_t y) { return lanes[x].first_cv > lanes[y].first_cv; });
        R.cbeg = cpos;
        if (kids[i].size() > 32767) bad = true;          // (bit 15 of ccnt is kFBranchInlineFlag)
        R.ccnt = (uint16_t)std::min<size_t>(kids[i].size(), 32767);
        for (uint32_t k : kids[i]) child[cpos++] = tl_of[k];
        // up to two children travel in the record itself (forest_layout.h): one dependent load less per branch end
        if (kids[i].size() <= kFBranchInlineChildren && n_lane <= 0xFFFFu) {
          uint32_t packed = 0;
          for (size_t k = 0; k < kids[i].size(); ++k) packed |= tl_of[kids[i][k]] << (16 * k);
          R.cbeg = packed;
          R.ccnt |= kFBranchInlineFlag;
        }
      }
      for (uint32_t lc = 0; lc < n_cell; ++lc) {
        const int64_t orig = H.cell_order[cell_begin + lc];
        const uint32_t det = d.det_cv ? (uint32_t)d.det_cv[orig] : 0u;
        const uint32_t lb = cells[lc].lane_begin;
        uint32_t found = kNoSlot;
        for (uint32_t b2 = 0; b2 < cells[lc].n_br && found == kNoSlot; ++b2) {
          const Lane& L = lanes[lb + b2];
          if (det < L.first_cv) continue;
          for (uint32_t k = 0; k < L.len; ++k)
            if (cvs[L.cv_begin + k] == det) { found = slot_of(tl_of[lb + b2], k); break; }
        }
        cell_det[lc] = found;
      }
    }
    if (topo_out && !forest) {
      const TopoOff to = topo_offsets(uc.n_task, uc.n_level, n_lane, n_child, n_cell);
      topo_out->assign(to.total, 0);
      uint8_t* tp = topo_out->data();
      std::memcpy(tp + to.tasks, tasks.data(), tasks.size() * sizeof(Task));
      std::memcpy(tp + to.level_begin, level_begin.data(), level_begin.size() * 4);
      LaneRec* lrec = (LaneRec*)(tp + to.lanes);
      uint32_t* child = (uint32_t*)(tp + to.child);
      uint32_t* cell_det = (uint32_t*)(tp + to.cell_det);
      uint32_t cpos = 0;
      for (uint32_t tl = 0; tl < n_lane; ++tl) {       // in unit-local branch order
        const uint32_t i = order[tl];
        const Lane& L = lanes[i];
        LaneRec& R = lrec[tl];
        R.len = (uint16_t)L.len;
        R.cell = (uint16_t)L.lc;
        R.pad = 0;
        if (L.parent_br >= 0) {
          uint32_t pi = cells[L.lc].lane_begin + L.parent_br;
          R.pslot = slot_of(tl_of[pi], lanes[pi].len - 1);
        } else {
          R.pslot = kNoSlot;
        }
        std::sort(kids[i].begin(), kids[i].end(), [&](uint32_t x, uint32_t y) { return lanes[x].first_cv > lanes[y].first_cv; });
        R.cbeg = cpos;
        if (kids[i].size() > 65535) bad = true;
        R.ccnt = (uint16_t)std::min<size_t>(kids[i].size(), 65535);
        for (uint32_t k : kids[i]) child[cpos++] = tl_of[k];
      }
      for (uint32_t lc = 0; lc < n_cell; ++lc) {
        int64_t orig = H.cell_order[cell_begin + lc];
        uint32_t det = d.det_cv ? (uint32_t)d.det_cv[orig] : 0u;
        // slot of the detector CV: find its branch
        const uint32_t lb = cells[lc].lane_begin;
        uint32_t found = kNoSlot;
        for (uint32_t b2 = 0; b2 < cells[lc].n_br && found == kNoSlot; ++b2) {
          const Lane& L = lanes[lb + b2];
          if (det < L.first_cv) continue;
          for (uint32_t k = 0; k < L.len; ++k)
            if (cvs[L.cv_begin + k] == det) { found = slot_of(tl_of[lb + b2], k); break; }
        }
        cell_det[lc] = found;
      }
    }
    if (!out) return uc;

    // ------------------------------------------------------------------ fill
    const GenOff go = gen_offsets(uc.n_slot, n_syn);
    uint8_t* fast = out->fast.data() + uc.fast_off;
    double* st = out->state.data() + uc.state_base;
    double* gen = out->gen.data() + uc.gen_base;
    UnitHeader hd;
    std::memset(&hd, 0, sizeof hd);
    hd.n_slot = uc.n_slot; hd.n_lane = n_lane; hd.n_task = uc.n_task; hd.n_level = uc.n_level;
    hd.n_cell = n_cell; hd.n_hh = n_hh; hd.n_syn = n_syn; hd.n_clamp = n_clamp;
    hd.n_child = n_child; hd.flags = uc.flags; hd.fast_bytes = uc.fast_bytes; hd.state_bytes = uc.state_bytes;
    hd.topo_off = uc.topo_off; hd.gen_base = uc.gen_base; hd.state_base = uc.state_base;
    hd.cell_base = uc.cell_base; hd.scratch_base = uc.scratch_base;
    hd.pad[0] = (uint32_t)(uc.lane_base & 0xFFFFFFFFu); hd.pad[1] = (uint32_t)((uint64_t)uc.lane_base >> 32);
    hd.pad[2] = (uint32_t)n_warp;
    std::memcpy(fast, &hd, sizeof hd);
    double* hh_gna = (double*)(fast + fo.hh_gna);
    double* hh_gk = (double*)(fast + fo.hh_gk);
    double* hh_gl = (double*)(fast + fo.hh_gl);
    double* syn_e = (double*)(fast + fo.syn_e);
    double* cl_t0 = (double*)(fast + fo.cl_t0);
    double* cl_t1 = (double*)(fast + fo.cl_t1);
    double* cl_amp = (double*)(fast + fo.cl_amp);
    uint32_t* hh_slot = (uint32_t*)(fast + fo.hh_slot);
    uint32_t* syn_slot = (uint32_t*)(fast + fo.syn_slot);
    uint32_t* cl_slot = (uint32_t*)(fast + fo.cl_slot);
    uint16_t* hh_cell = (uint16_t*)(fast + fo.hh_cell);
    uint16_t* syn_cell = (uint16_t*)(fast + fo.syn_cell);
    uint16_t* cl_cell = (uint16_t*)(fast + fo.cl_cell);
    const bool multi = n_cell > 1;

    struct Item { uint32_t slot, lc; int64_t id; };
    std::vector<Item> syn_items, cl_items;
    syn_items.reserve(n_syn); cl_items.reserve(n_clamp);
    uint32_t hh_pos = 0;
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
        out->cv_state_idx[a + i] = (uint32_t)(uc.state_base + so.v + s);
        if (has_hh(a + i)) {
          double sc = area * 1e-2;
          hh_gna[hh_pos] = d.hh_gnabar[a + i] * sc;
          hh_gk[hh_pos] = d.hh_gkbar[a + i] * sc;
          hh_gl[hh_pos] = d.hh_gl[a + i] * sc;
          hh_slot[hh_pos] = s;
          if (multi) hh_cell[hh_pos] = (uint16_t)lc;
          out->hh_m_idx[uc.hh_base + hh_pos] = (uint32_t)(uc.state_base + so.m + hh_pos);
          out->hh_stride[uc.hh_base + hh_pos] = so.h - so.m;
          out->hh_cv[uc.hh_base + hh_pos] = (uint32_t)(a + i);
          ++hh_pos;
        }
      }
      if (d.syn_off)
        for (int64_t s = d.syn_off[orig]; s < d.syn_off[orig + 1]; ++s) syn_items.push_back({cv_slot[d.syn_cv[s]], lc, s});
      for (int64_t q = clamp_off[orig]; q < clamp_off[orig + 1]; ++q) cl_items.push_back({cv_slot[d.clamp_cv[clamp_idx[q]]], lc, clamp_idx[q]});
      // runtime triple: no event pending, empty segment, detector armed (reading R10)
      double* rt = st + so.rt + kRtDoubles * lc;
      rt[0] = std::numeric_limits<double>::infinity();
      rt[1] = 0.0;
      rt[2] = 1.0;
      out->cell_rt_idx[cell_begin + lc] = (uint32_t)(uc.state_base + so.rt + kRtDoubles * lc);
    }
    // point mechanisms sorted by (slot, caller's index): the items on one CV form a run that one
    // lane sums in ascending index order
    auto by_slot = [](const Item& x, const Item& y) { return x.slot != y.slot ? x.slot < y.slot : x.id < y.id; };
    std::sort(syn_items.begin(), syn_items.end(), by_slot);
    std::sort(cl_items.begin(), cl_items.end(), by_slot);
    for (uint32_t p = 0; p < syn_items.size(); ++p) {
      const Item& it = syn_items[p];
      syn_slot[p] = it.slot;
      if (multi) syn_cell[p] = (uint16_t)it.lc;
      if (!H.syn_uniform) syn_e[p] = d.syn_e[it.id];
      gen[go.syn_tau + p] = d.syn_tau[it.id];
      out->syn_state_idx[it.id] = (uint32_t)(uc.state_base + so.g + p);
    }
    for (uint32_t p = 0; p < cl_items.size(); ++p) {
      const Item& it = cl_items[p];
      cl_slot[p] = it.slot;
      if (multi) cl_cell[p] = (uint16_t)it.lc;
      cl_t0[p] = d.clamp_t0[it.id];
      cl_t1[p] = d.clamp_t1[it.id];
      cl_amp[p] = d.clamp_amp[it.id];
    }
    return uc;
  }
};

}  // namespace


namespace {

// ---------------------------------------------------------------------------------------------
// Cell groups (group_layout.h)
// ---------------------------------------------------------------------------------------------
struct ClassInfo {
  uint32_t n_cv = 0, n_seg = 0;
  std::vector<uint32_t> cv_slot;       // control volume -> slot
  std::vector<uint8_t> record;         // ClassRecord + arrays
  int64_t topo_off = 0;
  std::vector<uint32_t> cells;         // caller's cell ids, ascending
  bool grouped = false;
};

constexpr uint32_t kMinChunk = 16;     // control volumes below which a stage is not split further
constexpr uint32_t kMaxSegLen = 4096;

// Segments, stages of independent chunks, slot numbering and the serialised record of one tree.
void build_class(const int32_t* par, uint32_t n, ClassInfo& K) {
  K.n_cv = n;
  std::vector<uint32_t> nchild(n, 0), seg_of(n, 0);
  for (uint32_t i = 1; i < n; ++i) nchild[par[i]]++;
  struct Seg { uint32_t first, len; int32_t parent; std::vector<uint32_t> kids; };
  std::vector<Seg> segs;
  for (uint32_t i = 0; i < n; ++i) {
    const bool fresh = i == 0 || nchild[par[i]] != 1 || segs[seg_of[par[i]]].len >= kMaxSegLen ||
                       i != segs[seg_of[par[i]]].first + segs[seg_of[par[i]]].len;
    if (fresh) {
      Seg sg;
      sg.first = i; sg.len = 0; sg.parent = i == 0 ? -1 : (int32_t)seg_of[par[i]];
      seg_of[i] = (uint32_t)segs.size();
      segs.push_back(sg);
    } else {
      seg_of[i] = seg_of[par[i]];
    }
    segs[seg_of[i]].len++;
  }
  // a chain that is not numbered consecutively is cut, so CV k of a segment is always first + k, and
  // children hang off the last control volume of their parent segment
  const uint32_t ns = (uint32_t)segs.size();
  K.n_seg = ns;
  for (uint32_t s2 = 1; s2 < ns; ++s2) segs[segs[s2].parent].kids.push_back(s2);
  // stages: repeatedly peel the maximal subtrees that fit the per-slot share of what is left
  std::vector<uint8_t> left(ns, 1);
  std::vector<uint64_t> w(ns, 0);
  std::vector<std::vector<std::vector<uint32_t>>> stages;   // [stage][slot] -> segments in backward order
  uint32_t n_left = ns;
  while (n_left > 0) {
    for (uint32_t s2 = ns; s2-- > 0;) {
      if (!left[s2]) continue;
      w[s2] = segs[s2].len;
      for (uint32_t k : segs[s2].kids) if (left[k]) w[s2] += w[k];
    }
    const uint64_t total = w[0];
    const uint64_t cap = std::max<uint64_t>((total + kGroupSlots - 1) / kGroupSlots, kMinChunk);
    std::vector<uint32_t> roots;
    for (uint32_t s2 = 0; s2 < ns; ++s2)
      if (left[s2] && w[s2] <= cap && (segs[s2].parent < 0 || w[segs[s2].parent] > cap)) roots.push_back(s2);
    if (roots.empty())
      for (uint32_t s2 = 0; s2 < ns; ++s2) {
        if (!left[s2]) continue;
        bool leaf = true;
        for (uint32_t k : segs[s2].kids) leaf = leaf && !left[k];
        if (leaf) roots.push_back(s2);
      }
    std::stable_sort(roots.begin(), roots.end(), [&](uint32_t x, uint32_t y) { return w[x] > w[y]; });
    std::vector<std::vector<uint32_t>> slots(kGroupSlots);
    std::vector<uint64_t> load(kGroupSlots, 0);
    for (uint32_t r : roots) {
      uint32_t best = 0;
      for (uint32_t h = 1; h < (uint32_t)kGroupSlots; ++h) if (load[h] < load[best]) best = h;
      load[best] += w[r];
      // the remaining subtree of r, children before parents (descending segment id)
      std::vector<uint32_t> sub{r};
      for (size_t q = 0; q < sub.size(); ++q)
        for (uint32_t k : segs[sub[q]].kids) if (left[k]) sub.push_back(k);
      std::sort(sub.begin(), sub.end(), [](uint32_t x, uint32_t y) { return x > y; });
      slots[best].insert(slots[best].end(), sub.begin(), sub.end());
    }
    for (auto& v : slots) for (uint32_t s2 : v) { left[s2] = 0; --n_left; }
    stages.push_back(std::move(slots));
  }
  // slots: ascending addresses along the forward sweep
  std::vector<uint32_t> slot0(ns, 0);
  uint32_t next = 0;
  for (size_t st = stages.size(); st-- > 0;)
    for (uint32_t h = 0; h < (uint32_t)kGroupSlots; ++h)
      for (size_t q = stages[st][h].size(); q-- > 0;) {
        const uint32_t s2 = stages[st][h][q];
        slot0[s2] = next;
        next += segs[s2].len;
      }
  K.cv_slot.resize(n);
  for (uint32_t i = 0; i < n; ++i) K.cv_slot[i] = slot0[seg_of[i]] + (i - segs[seg_of[i]].first);
  // record
  uint32_t n_child = ns - 1;
  ClassRecord R;
  std::memset(&R, 0, sizeof R);
  R.n_cv = n; R.n_seg = ns; R.n_stage = (uint32_t)stages.size(); R.n_child = n_child;
  uint32_t p = sizeof(ClassRecord);
  auto sec = [&](uint32_t bytes) { uint32_t at = p; p = align_up(p + bytes, 16); return at; };
  R.off_segs = sec(ns * (uint32_t)sizeof(SegRec));
  R.off_order = sec(ns * 2);
  R.off_sched = sec(((uint32_t)stages.size() * kGroupSlots + 1) * 2);
  R.off_child = sec(n_child * 2);
  R.bytes = align_up(p, 128);
  R.n_block = (uint32_t)stages.size();
  while (R.n_block > 0) {
    bool narrow = true;
    for (uint32_t h = kLaneGroups; h < (uint32_t)kGroupSlots; ++h) narrow = narrow && stages[R.n_block - 1][h].empty();
    if (!narrow) break;
    --R.n_block;
  }
  K.record.assign(R.bytes, 0);
  std::memcpy(K.record.data(), &R, sizeof R);
  SegRec* sr = (SegRec*)(K.record.data() + R.off_segs);
  uint16_t* order = (uint16_t*)(K.record.data() + R.off_order);
  uint16_t* sched = (uint16_t*)(K.record.data() + R.off_sched);
  uint16_t* child = (uint16_t*)(K.record.data() + R.off_child);
  // Segments are numbered in processing order on the device (the q-th segment the backward sweep meets is segment q:
  // order[] is the identity and the kernels do not read it), and a segment with at most two children carries them in
  // its record (cbeg = child0 | child1 << 16) - two dependent shared-memory loads less per chunk of a sweep.
  std::vector<uint32_t> pos_of(ns, 0);
  uint32_t opos = 0, spos = 0;
  for (size_t st = 0; st < stages.size(); ++st)
    for (uint32_t h = 0; h < (uint32_t)kGroupSlots; ++h) {
      sched[spos++] = (uint16_t)opos;
      for (uint32_t s2 : stages[st][h]) { order[opos] = (uint16_t)opos; pos_of[s2] = opos++; }
    }
  sched[spos] = (uint16_t)opos;
  uint32_t cpos = 0;
  for (uint32_t q = 0; q < ns; ++q) {
    uint32_t s2 = 0;
    while (pos_of[s2] != q) ++s2;
    SegRec& r = sr[q];
    r.slot0 = slot0[s2];
    r.pslot = segs[s2].parent < 0 ? kNoSlot : K.cv_slot[par[segs[s2].first]];
    r.len = (uint16_t)segs[s2].len;
    r.ccnt = (uint16_t)segs[s2].kids.size();
    r.cbeg = cpos;
    // children in descending order: the order in which a leaves -> root elimination meets them
    uint32_t packed = 0, k = 0;
    for (size_t j = segs[s2].kids.size(); j-- > 0; ++k) {
      const uint32_t ch = pos_of[segs[s2].kids[j]];
      child[cpos++] = (uint16_t)ch;
      if (k < 2) packed |= ch << (16 * k);
    }
    if (r.ccnt <= kSegInlineChildren) r.cbeg = packed;
  }
}

struct GroupCounts { uint32_t cls = 0, n_cell = 0, n_hh_rows = 0, n_syn_rows = 0, n_cl_rows = 0; int64_t cell_begin = 0, hh_base = 0; bool disjoint = false; };

}  // namespace

// Synapse runs (second half; reading R22).  In a cell with many synapses, the synapses on one
// control volume with the same (tau, e) only enter a step through their TOTAL conductance: I = (sum g_j)(V - e) and
// sum g_j <- (sum g_j) exp(-delta / tau) are exact for the exponential integrator (R7).  Such cells are handed to the
// builders with one synapse per run; every original synapse keeps a lazy record (g_j, time of last touch) that an
// event brings up to date, so that read-back returns the individual g_j.
struct SynRuns {
  std::vector<int64_t> syn_off;           // derived description: per cell
  std::vector<int32_t> syn_cv;
  std::vector<double> syn_tau, syn_e;
  std::vector<int64_t> map;               // original synapse -> derived synapse (global index)
  std::vector<int64_t> lid;               // original synapse -> lazy record, or -1
  std::vector<int64_t> run_of_lazy;       // lazy record -> derived synapse (its run)
  int64_t n_lazy = 0, n_runs = 0;
};

static void build_runs(const arb_desc& d, const BuildParams& P, SynRuns& R) {
  const int64_t nc = d.n_cells, ns = d.syn_off ? d.syn_off[nc] : 0;
  R.syn_off.assign(nc + 1, 0);
  R.map.assign(ns, 0); R.lid.assign(ns, -1);
  R.syn_cv.reserve(ns); R.syn_tau.reserve(ns); R.syn_e.reserve(ns);
  std::vector<int64_t> order;
  for (int64_t c = 0; c < nc; ++c) {
    const int64_t a = d.syn_off[c], n = d.syn_off[c + 1] - a;
    bool merge = P.merge_min_syn > 0 && n >= (int64_t)P.merge_min_syn && !(d.cell_kind && d.cell_kind[c] != 0);
    auto same = [&](int64_t x, int64_t y) { return d.syn_cv[x] == d.syn_cv[y] && d.syn_tau[x] == d.syn_tau[y] && d.syn_e[x] == d.syn_e[y]; };
    if (merge) {
      order.resize(n);
      for (int64_t i = 0; i < n; ++i) order[i] = a + i;
      std::sort(order.begin(), order.end(), [&](int64_t x, int64_t y) {
        if (d.syn_cv[x] != d.syn_cv[y]) return d.syn_cv[x] < d.syn_cv[y];
        if (d.syn_tau[x] != d.syn_tau[y]) return d.syn_tau[x] < d.syn_tau[y];
        if (d.syn_e[x] != d.syn_e[y]) return d.syn_e[x] < d.syn_e[y];
        return x < y;
      });
      int64_t nr = 1;
      for (int64_t i = 1; i < n; ++i) nr += !same(order[i], order[i - 1]);
      merge = 2 * nr <= n;                          // worth it only when runs are much fewer than synapses
    }
    if (!merge) {
      for (int64_t s = a; s < a + n; ++s) {
        R.map[s] = (int64_t)R.syn_cv.size();
        R.syn_cv.push_back(d.syn_cv[s]); R.syn_tau.push_back(d.syn_tau[s]); R.syn_e.push_back(d.syn_e[s]);
      }
    } else {
      for (int64_t i = 0; i < n; ++i) {
        const int64_t s = order[i];
        if (i == 0 || !same(s, order[i - 1])) { ++R.n_runs; R.syn_cv.push_back(d.syn_cv[s]); R.syn_tau.push_back(d.syn_tau[s]); R.syn_e.push_back(d.syn_e[s]); }
        R.map[s] = (int64_t)R.syn_cv.size() - 1;
        R.lid[s] = R.n_lazy++;                      // records of a run are contiguous, in ascending original index
        R.run_of_lazy.push_back(R.map[s]);
      }
    }
    R.syn_off[c + 1] = (int64_t)R.syn_cv.size();
  }
}

int build(const arb_desc& d_in, const BuildParams& P, bool fill, HostModel& H, std::string& err) {
  int rc = validate(d_in, err);
  if (rc) return rc;
  // synapse runs: from here on `d` is the description the kernels integrate (one synapse per run in merged cells)
  SynRuns runs;
  arb_desc d_mod = d_in;
  if (d_in.syn_off && P.merge_min_syn > 0) {
    bool any = false;
    for (int64_t c = 0; c < d_in.n_cells && !any; ++c)
      any = d_in.syn_off[c + 1] - d_in.syn_off[c] >= (int64_t)P.merge_min_syn && !(d_in.cell_kind && d_in.cell_kind[c] != 0);
    if (any) {
      build_runs(d_in, P, runs);
      d_mod.syn_off = runs.syn_off.data(); d_mod.syn_cv = runs.syn_cv.data();
      d_mod.syn_tau = runs.syn_tau.data(); d_mod.syn_e = runs.syn_e.data();
    }
  }
  const arb_desc& d = d_mod;
  const int64_t n_syn_orig = d_in.syn_off ? d_in.syn_off[d_in.n_cells] : 0;
  H = HostModel();
  H.n_cells = d.n_cells;
  H.n_cv = d.cv_off[d.n_cells];
  H.n_syn = d.syn_off ? d.syn_off[d.n_cells] : 0;
  H.n_clamp = d.n_clamp; H.n_conn = d.n_conn; H.n_ext = d.n_ext;
  H.gid_base = d.shard_n_global > 0 ? d.shard_gid_base : 0;
  H.n_src = d.shard_n_global > 0 ? d.shard_n_global : d.n_cells;
  H.ena = d.hh_ena; H.ek = d.hh_ek; H.el = d.hh_el; H.threshold = d.threshold;
  const int64_t nc = d.n_cells;
  // uniform synapse parameters (true for every BASELINE config): no per-synapse e / decay arrays
  H.syn_uniform = H.n_syn > 0;
  if (H.n_syn > 0) {
    H.syn_tau_u = d.syn_tau[0]; H.syn_e_u = d.syn_e[0];
    for (int64_t s = 1; s < H.n_syn && H.syn_uniform; ++s) H.syn_uniform = d.syn_tau[s] == H.syn_tau_u && d.syn_e[s] == H.syn_e_u;
  }
  // clamps grouped by cell
  std::vector<int64_t> clamp_off(nc + 1, 0), clamp_idx(d.n_clamp);
  for (int64_t k = 0; k < d.n_clamp; ++k) clamp_off[d.clamp_cell[k] + 1]++;
  for (int64_t c = 0; c < nc; ++c) clamp_off[c + 1] += clamp_off[c];
  {
    std::vector<int64_t> cur(clamp_off.begin(), clamp_off.end() - 1);
    for (int64_t k = 0; k < d.n_clamp; ++k) clamp_idx[cur[d.clamp_cell[k]]++] = k;
  }
  // HH instances and branches (maximal unbranched chains) of every cell
  std::vector<uint32_t> cell_hh(nc, 0), cell_nbr(nc, 0), cell_lvl(nc, 0);   // ..., branch levels of the cell's tree
  parallel_for(nc, [&](int64_t c) {
    const int64_t a = d.cv_off[c], n = d.cv_off[c + 1] - a;
    uint32_t nh = 0;
    if (d.hh_gnabar)
      for (int64_t i = a; i < a + n; ++i) nh += d.hh_gnabar[i] != 0.0 || d.hh_gkbar[i] != 0.0 || d.hh_gl[i] != 0.0;
    cell_hh[c] = nh;
    std::vector<uint32_t> nchild((size_t)n, 0);
    for (int64_t i = 1; i < n; ++i) nchild[d.cv_parent[a + i]]++;
    uint32_t nb = 1;
    for (int64_t i = 1; i < n; ++i) nb += nchild[d.cv_parent[a + i]] != 1;
    cell_nbr[c] = nb + (uint32_t)(n / kForestMaxBranchLen);     // chains longer than a branch may hold are cut
    std::vector<uint32_t> lvl((size_t)n, 0);
    uint32_t deepest = 0;
    for (int64_t i = 1; i < n; ++i) {
      const int64_t p = d.cv_parent[a + i];
      lvl[i] = lvl[p] + (nchild[p] != 1 ? 1u : 0u);
      deepest = std::max(deepest, lvl[i]);
    }
    cell_lvl[c] = deepest + 1 + (uint32_t)(n / kForestMaxBranchLen);
  });
  // shared memory a forest of these counts needs (forest_layout.h)
  auto forest_need = [&](uint64_t n_cv, uint64_t n_br, uint64_t n_hh, uint64_t n_syn, uint64_t n_clamp, uint64_t n_cell, int n_warp, uint32_t n_level) -> uint64_t {
    if (n_cv > 0x0FFFFFFFull || n_syn > 0x0FFFFFFFull || n_clamp > 0x0FFFFFFFull) return ~0ull;
    ForestCaps fc;
    fc.state_bytes = 8 * state_offsets(align_up((uint32_t)n_cv, 2), (uint32_t)n_hh, (uint32_t)n_syn, (uint32_t)n_cell).total;
    fc.n_branch = (uint32_t)n_br; fc.n_spec = (uint32_t)(n_hh + n_syn + n_clamp); fc.n_cell = (uint32_t)n_cell;
    fc.topo_bytes = ftopo_bound((uint32_t)n_cv, (uint32_t)n_br, (uint32_t)n_cell, (uint32_t)n_warp, n_level);
    return forest_smem_plan(fc).bytes;
  };
  auto cell_counts = [&](int64_t c, uint64_t& n_cv, uint64_t& n_syn, uint64_t& n_cl) {
    n_cv = (uint64_t)(d.cv_off[c + 1] - d.cv_off[c]);
    n_syn = d.syn_off ? (uint64_t)(d.syn_off[c + 1] - d.syn_off[c]) : 0;
    n_cl = (uint64_t)(clamp_off[c + 1] - clamp_off[c]);
  };
  // ---- topology classes -> cell groups (group_layout.h)
  std::vector<ClassInfo> classes;
  std::vector<int32_t> cell_class(nc, -1);
  std::vector<GroupCounts> groups;
  std::vector<uint32_t> group_cells;
  if (P.group_min_cells > 0) {
    std::vector<uint64_t> hash(nc);
    parallel_for(nc, [&](int64_t c) {
      hash[c] = fnv1a((const uint8_t*)(d.cv_parent + d.cv_off[c]), 4 * (size_t)(d.cv_off[c + 1] - d.cv_off[c]));
    });
    std::unordered_map<uint64_t, std::vector<int32_t>> by_hash;
    for (int64_t c = 0; c < nc; ++c) {
      const uint32_t n = (uint32_t)(d.cv_off[c + 1] - d.cv_off[c]);
      if (n > std::min(P.group_max_cv, kGroupMaxCv) || (d.cell_kind && d.cell_kind[c] != 0)) continue;
      auto& bucket = by_hash[hash[c]];
      int32_t cls = -1;
      for (int32_t k : bucket) {
        const uint32_t rep = classes[k].cells[0];
        if (classes[k].n_cv == n && std::memcmp(d.cv_parent + d.cv_off[rep], d.cv_parent + d.cv_off[c], 4 * (size_t)n) == 0) { cls = k; break; }
      }
      if (cls < 0) {
        cls = (int32_t)classes.size();
        classes.emplace_back();
        classes[cls].n_cv = n;
        bucket.push_back(cls);
      }
      classes[cls].cells.push_back((uint32_t)c);
    }
    for (size_t k = 0; k < classes.size(); ++k) {
      ClassInfo& K = classes[k];
      K.grouped = K.cells.size() >= P.group_min_cells;
      if (K.grouped) {
        // a group's state record (V, synaptic g, gates), two coefficient buffers and instance tables
        // must fit in shared memory - twice per SM at least; cells with very many point mechanisms
        // (the paper's 10,000-synapse ring cell) are laid out as units instead
        uint32_t mx_hh = 0, mx_syn = 0, mx_cl = 0;
        for (uint32_t c : K.cells) {
          mx_hh = std::max(mx_hh, cell_hh[c]);
          if (d.syn_off) mx_syn = std::max(mx_syn, (uint32_t)std::min<int64_t>(d.syn_off[c + 1] - d.syn_off[c], 1 << 24));
          mx_cl = std::max(mx_cl, (uint32_t)std::min<int64_t>(clamp_off[c + 1] - clamp_off[c], 1 << 24));
        }
        const GConstOff co = gconst_offsets(K.n_cv, mx_hh, mx_syn, mx_cl, H.syn_uniform);
        GroupCaps caps;
        caps.slot_cap = K.n_cv;
        caps.state_bytes = 8 * gstate_offsets(K.n_cv, mx_hh, mx_syn).total;
        caps.tail_bytes = co.total - co.hh_gna;
        caps.class_bytes = 64 + 40 * K.n_cv;               // upper bound: one segment per control volume
        caps.buf_rows = std::max(K.n_cv, mx_hh + mx_syn + mx_cl);
        if (group_smem_plan(caps).bytes > P.group_max_smem) K.grouped = false;
      }
      if (!K.grouped) continue;
      for (size_t i = 0; i < K.cells.size(); i += kG) {
        GroupCounts G;
        G.cls = (uint32_t)k;
        G.n_cell = (uint32_t)std::min<size_t>(kG, K.cells.size() - i);
        G.cell_begin = (int64_t)group_cells.size();
        for (uint32_t j = 0; j < G.n_cell; ++j) { group_cells.push_back(K.cells[i + j]); cell_class[K.cells[i + j]] = (int32_t)k; }
        groups.push_back(G);
      }
    }
    parallel_for((int64_t)classes.size(), [&](int64_t k) {
      if (classes[k].grouped) build_class(d.cv_parent + d.cv_off[classes[k].cells[0]], classes[k].n_cv, classes[k]);
    });
  }
  const int64_t ngc = (int64_t)group_cells.size();
  H.n_groups = (int64_t)groups.size();
  H.n_group_cells = ngc;
  // internal cell order: group cells, forest cells (big first), block-unit cells
  std::vector<uint32_t> forest_cells, block_cells, point_cells;
  for (int64_t c = 0; c < nc; ++c) {
    if (cell_class[c] >= 0) continue;
    if (d.cell_kind && d.cell_kind[c] != 0) { point_cells.push_back((uint32_t)c); continue; }
    uint64_t n_cv, n_syn, n_cl;
    cell_counts(c, n_cv, n_syn, n_cl);
    const bool fits = n_cv <= P.forest_max_cv && n_syn < P.forest_max_syn &&
                      forest_need(n_cv, cell_nbr[c], cell_hh[c], n_syn, n_cl, 1, kForestMaxWarps, cell_lvl[c]) <= forest_class_budget(kForestClasses - 1);
    (fits ? forest_cells : block_cells).push_back((uint32_t)c);
  }
  auto bigger = [&](uint32_t x, uint32_t y) { return d.cv_off[x + 1] - d.cv_off[x] > d.cv_off[y + 1] - d.cv_off[y]; };
  std::stable_sort(forest_cells.begin(), forest_cells.end(), bigger);
  std::stable_sort(block_cells.begin(), block_cells.end(), bigger);
  H.cell_order = group_cells;
  H.cell_order.insert(H.cell_order.end(), forest_cells.begin(), forest_cells.end());
  H.cell_order.insert(H.cell_order.end(), block_cells.begin(), block_cells.end());
  H.cell_order.insert(H.cell_order.end(), point_cells.begin(), point_cells.end());   // LIF cells and spike sources come last
  H.n_pcells = (int64_t)point_cells.size();
  H.pc_first = nc - H.n_pcells;
  H.cell_internal.resize(nc);
  for (int64_t i = 0; i < nc; ++i) H.cell_internal[H.cell_order[i]] = (uint32_t)i;
  // partition into units: forests (several small cells share one as long as it fits the smallest launch class),
  // then one block unit per remaining cell
  std::vector<int64_t> unit_begin;
  {
    uint64_t cv = 0, br = 0, hh = 0, syn = 0, cl = 0, cells = 0;
    uint32_t lv = 0;
    uint64_t forest_cv = P.forest_cv;
    if (P.forest_cv_auto) {                // few control volumes in all: more, smaller forests (measured on the paper's ring cell,
      uint64_t total = 0;                  // 2.6e5 CVs: forests of 256 / 384 / 512 / 1,024 CVs 0.033 / 0.0225 / 0.0227 / 0.027 ms per step)
      for (uint32_t c : forest_cells) total += (uint64_t)(d.cv_off[c + 1] - d.cv_off[c]);
      forest_cv = std::min<uint64_t>(P.forest_cv, std::max<uint64_t>(384, total / (4 * 148)));
    }
    for (int64_t i = 0; i < (int64_t)forest_cells.size(); ++i) {
      uint64_t n_cv, n_syn, n_cl;
      cell_counts(forest_cells[i], n_cv, n_syn, n_cl);
      const uint64_t n_hh = cell_hh[forest_cells[i]], n_br = cell_nbr[forest_cells[i]];
      if (cells == 0 || cells >= kForestMaxCells || cv + n_cv > forest_cv ||
          forest_need(cv + n_cv + 1, br + n_br, hh + n_hh, syn + n_syn, cl + n_cl, cells + 1, kForestWarps, std::max(lv, cell_lvl[forest_cells[i]])) > forest_class_budget(0)) {
        unit_begin.push_back(ngc + i); cv = br = hh = syn = cl = cells = 0; lv = 0;
      }
      lv = std::max(lv, cell_lvl[forest_cells[i]]);
      cv += n_cv; br += n_br; hh += n_hh; syn += n_syn; cl += n_cl; ++cells;
    }
    H.n_forests = (int64_t)unit_begin.size();
    for (int64_t i = 0; i < (int64_t)block_cells.size(); ++i) unit_begin.push_back(ngc + (int64_t)forest_cells.size() + i);
    unit_begin.push_back(nc - H.n_pcells);
  }
  H.n_units = (int64_t)unit_begin.size() - 1;
  H.units.resize(H.n_units);
  std::vector<uint32_t> unit_cells(H.n_units);
  for (int64_t u = 0; u < H.n_units; ++u) unit_cells[u] = (uint32_t)(unit_begin[u + 1] - unit_begin[u]);
  unit_begin.pop_back();
  // pass 1: counts and topo records
  std::vector<std::vector<uint8_t>> topo(H.n_units);
  std::atomic<int> too_many(0);
  parallel_for(H.n_units, [&](int64_t u) {
    UnitBuilder B{d, P, H, clamp_off, clamp_idx, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, false};
    B.forest = u < H.n_forests;
    H.units[u] = B.run(unit_begin[u], unit_cells[u], &topo[u], nullptr, nullptr);
    H.units[u].topo_bytes = (uint32_t)topo[u].size();
    if (B.forest) {
      // a forest beyond launch class 0 (one large cell) is swept by twice the warps (forest_layout.h)
      const UnitCounts& uc = H.units[u];
      ForestCaps fc;
      fc.state_bytes = uc.state_bytes; fc.topo_bytes = uc.topo_bytes; fc.n_branch = uc.n_lane; fc.n_spec = uc.n_hh + uc.n_syn + uc.n_clamp; fc.n_cell = uc.n_cell;
      if (forest_smem_plan(fc).bytes > forest_class_budget(0)) {
        UnitBuilder B2{d, P, H, clamp_off, clamp_idx, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, false};
        B2.forest = true; B2.n_warp = kForestWarpsBig;
        H.units[u] = B2.run(unit_begin[u], unit_cells[u], &topo[u], nullptr, nullptr);
        H.units[u].topo_bytes = (uint32_t)topo[u].size();
        H.units[u].n_warp = kForestWarpsBig;
        if (B2.bad) too_many.store(1);
      } else {
        H.units[u].n_warp = kForestWarps;
      }
    }
    if (u >= H.n_forests) H.units[u].flags |= UNIT_BLOCK;
    if (H.units[u].n_level > 60000 || H.units[u].n_slot > 0x3FFFFFFFu) too_many.store(1);
    if (B.bad) too_many.store(1);
  });
  if (too_many.load()) { err = "a cell is too deep or too large for the unit layout"; return ARB_E_INVALID; }
  // forests are launched by shared-memory need (forest_layout.h): order them by launch class, the class with
  // the largest forests first, and inside a class by size (the hardware deals CTAs in index order)
  {
    auto need_of = [&](const UnitCounts& uc) {
      ForestCaps fc;
      fc.state_bytes = uc.state_bytes; fc.topo_bytes = uc.topo_bytes; fc.n_branch = uc.n_lane; fc.n_spec = uc.n_hh + uc.n_syn + uc.n_clamp; fc.n_cell = uc.n_cell;
      return forest_smem_plan(fc).bytes;
    };
    auto class_of = [&](const UnitCounts& uc) {
      const uint32_t need = need_of(uc);
      for (int k = 0; k < kForestClasses; ++k) if (need <= forest_class_budget(k)) return k;
      return kForestClasses;               // does not fit (decided above with exact counts: cannot happen)
    };
    std::vector<int64_t> perm(H.n_forests);
    for (int64_t u = 0; u < H.n_forests; ++u) perm[u] = u;
    std::vector<int> cls(H.n_forests);
    for (int64_t u = 0; u < H.n_forests; ++u) {
      cls[u] = class_of(H.units[u]);
      if (cls[u] >= kForestClasses) { err = "a forest does not fit in shared memory"; return ARB_E_INVALID; }
    }
    std::stable_sort(perm.begin(), perm.end(), [&](int64_t x, int64_t y) {
      if (cls[x] != cls[y]) return cls[x] > cls[y];
      return H.units[x].n_cv > H.units[y].n_cv;
    });
    std::vector<UnitCounts> units2(H.units);
    std::vector<std::vector<uint8_t>> topo2(H.n_forests);
    std::vector<int64_t> begin2(unit_begin);
    std::vector<uint32_t> cells2(unit_cells);
    for (int64_t i = 0; i < H.n_forests; ++i) {
      units2[i] = H.units[perm[i]]; topo2[i].swap(topo[perm[i]]); begin2[i] = unit_begin[perm[i]]; cells2[i] = unit_cells[perm[i]];
    }
    for (int64_t i = 0; i < H.n_forests; ++i) topo[i].swap(topo2[i]);
    H.units.swap(units2); unit_begin.swap(begin2); unit_cells.swap(cells2);
    for (int k = 0; k < kForestClasses; ++k) { H.fcls[k].first = 0; H.fcls[k].count = 0; H.fcls[k].n_warp = k == 0 ? kForestWarps : kForestWarpsBig; }
    for (int k = 0; k < kForestClasses; ++k) H.fcls[k].plan = forest_smem_plan(ForestCaps{0, 0, 0, 0, 0});
    for (int64_t i = 0; i < H.n_forests; ++i) {
      const UnitCounts& uc = H.units[i];
      const int k = class_of(uc);
      if (H.fcls[k].count++ == 0) H.fcls[k].first = i;
      ForestCaps fc;
      fc.state_bytes = uc.state_bytes; fc.topo_bytes = uc.topo_bytes; fc.n_branch = uc.n_lane; fc.n_spec = uc.n_hh + uc.n_syn + uc.n_clamp; fc.n_cell = uc.n_cell;
      const ForestSmemPlan P = forest_smem_plan(fc);
      if (P.bytes > H.fcls[k].plan.bytes) H.fcls[k].plan = P;   // the launch reserves the largest need of the class
    }
  }
  // groups: row counts, then placement (groups first in every pool)
  parallel_for(H.n_groups, [&](int64_t g) {
    GroupCounts& G = groups[g];
    G.disjoint = true;
    std::vector<uint8_t> kind;
    for (uint32_t lc = 0; lc < G.n_cell; ++lc) {
      const uint32_t c = group_cells[G.cell_begin + lc];
      {                                   // does any control volume of the cell carry two kinds of point mechanism?
        const int64_t a0 = d.cv_off[c];
        kind.assign((size_t)(d.cv_off[c + 1] - a0), 0);
        if (d.hh_gnabar)
          for (size_t i = 0; i < kind.size(); ++i)
            if (d.hh_gnabar[a0 + i] != 0.0 || d.hh_gkbar[a0 + i] != 0.0 || d.hh_gl[a0 + i] != 0.0) kind[i] |= 1;
        if (d.syn_off)
          for (int64_t q = d.syn_off[c]; q < d.syn_off[c + 1]; ++q) kind[d.syn_cv[q]] |= 2;
        for (int64_t q = clamp_off[c]; q < clamp_off[c + 1]; ++q) kind[d.clamp_cv[clamp_idx[q]]] |= 4;
        for (uint8_t k : kind) if (k & (k - 1)) G.disjoint = false;
      }
      G.n_hh_rows = std::max(G.n_hh_rows, cell_hh[c]);
      if (d.syn_off) G.n_syn_rows = std::max(G.n_syn_rows, (uint32_t)(d.syn_off[c + 1] - d.syn_off[c]));
      G.n_cl_rows = std::max(G.n_cl_rows, (uint32_t)(clamp_off[c + 1] - clamp_off[c]));
    }
  });
  for (auto& K : classes)
    if (K.grouped) {
      K.topo_off = H.topo_bytes;
      H.topo_bytes += (int64_t)K.record.size();
      H.n_classes++;
      H.g_seg_cap = std::max(H.g_seg_cap, K.n_seg);
      H.gcaps.class_bytes = std::max(H.gcaps.class_bytes, (uint32_t)K.record.size());
    }
  H.gdescs.resize(H.n_groups);
  for (int64_t g = 0; g < H.n_groups; ++g) {
    GroupCounts& G = groups[g];
    const ClassInfo& K = classes[G.cls];
    GroupDesc& D = H.gdescs[g];
    D.n_cv = K.n_cv; D.n_cell = G.n_cell; D.n_hh_rows = G.n_hh_rows; D.n_syn_rows = G.n_syn_rows; D.n_cl_rows = G.n_cl_rows; D.flags = G.disjoint ? GROUP_POINT_DISJOINT : 0u;
    D.class_off = K.topo_off;
    D.cell_base = G.cell_begin;
    const GConstOff co = gconst_offsets(K.n_cv, G.n_hh_rows, G.n_syn_rows, G.n_cl_rows, H.syn_uniform);
    const GStateOff so = gstate_offsets(K.n_cv, G.n_hh_rows, G.n_syn_rows);
    D.const_off = H.fast_bytes;   H.fast_bytes += co.total;
    D.state_base = H.state_doubles; H.state_doubles += so.total;
    H.gcaps.state_bytes = std::max(H.gcaps.state_bytes, 8 * so.total);
    H.gcaps.tail_bytes = std::max(H.gcaps.tail_bytes, co.total - co.hh_gna);
    D.gen_base = H.gen_doubles;   H.gen_doubles += ggen_offsets(K.n_cv, G.n_syn_rows).total;
    G.hh_base = H.n_hh;
    for (uint32_t lc = 0; lc < G.n_cell; ++lc) H.n_hh += cell_hh[group_cells[G.cell_begin + lc]];
    H.gcaps.slot_cap = std::max(H.gcaps.slot_cap, K.n_cv);
    H.gcaps.buf_rows = std::max(H.gcaps.buf_rows, std::max(K.n_seg, G.n_hh_rows + G.n_syn_rows + G.n_cl_rows));
  }
  // placement; tree structures are deduplicated by content
  std::unordered_map<uint64_t, std::vector<int64_t>> seen;   // hash -> units that own a stored record
  std::vector<int64_t> topo_owner(H.n_units, -1);
  for (int64_t u = 0; u < H.n_units; ++u) {
    UnitCounts& uc = H.units[u];
    uc.fast_off = H.fast_bytes;     H.fast_bytes += align_up(uc.fast_bytes, 128);
    uc.state_base = H.state_doubles; H.state_doubles += align_up(uc.state_bytes, 128) / 8;
    uc.gen_base = H.gen_doubles;    H.gen_doubles += gen_offsets(uc.n_slot, uc.n_syn).total;
    uc.lane_base = H.n_lanes;       H.n_lanes += uc.n_lane;
    uc.hh_base = H.n_hh;            H.n_hh += uc.n_hh;
    const uint64_t h = fnv1a(topo[u].data(), topo[u].size());
    auto& bucket = seen[h];
    int64_t owner = -1;
    for (int64_t v : bucket)
      if (topo[v].size() == topo[u].size() && std::memcmp(topo[v].data(), topo[u].data(), topo[u].size()) == 0) { owner = v; break; }
    if (owner < 0) {
      bucket.push_back(u);
      uc.topo_off = H.topo_bytes;
      H.topo_bytes += (int64_t)align_up((uint32_t)topo[u].size(), 128);
      H.topo_records++;
      topo_owner[u] = u;
    } else {
      uc.topo_off = H.units[owner].topo_off;
      std::vector<uint8_t>().swap(topo[u]);
    }
    const uint32_t n_spec = uc.n_hh + uc.n_syn + uc.n_clamp;
    if (uc.flags & UNIT_FOREST) {
      uc.scratch_base = H.scratch_doubles;
      H.scratch_doubles += fscratch_offsets(uc.n_slot, uc.n_lane).total;
    } else if (uc.flags & UNIT_BLOCK) {
      // contrib | dcontrib | xI | fgen | invdgen | run heads of the synapse list (uint32 count, then indices)
      uc.scratch_base = H.scratch_doubles;
      H.scratch_doubles += 2 * (int64_t)align_up(uc.n_lane, 2) + align_up(n_spec, 2) + 2 * (int64_t)uc.n_slot +
                           align_up(uc.n_slot / 2 + 2, 2);
      H.block_lane_cap = std::max(H.block_lane_cap, uc.n_lane);
    }
  }
  // point cells: a record each (V | runtime | t_last | t_ref_end | cursor), then one (unused) conductance slot per event
  // target, so that events on them sort like everybody else's
  H.pc_state_base = H.state_doubles;
  {
    int64_t targets = 0;
    for (uint32_t c : point_cells) {
      targets += d.syn_off ? d.syn_off[c + 1] - d.syn_off[c] : 0;
      if (d.cell_kind[c] == 2) H.n_sched += d.src_off[c + 1] - d.src_off[c];
    }
    H.state_doubles += align_up((uint32_t)std::min<int64_t>(kPcDoubles * H.n_pcells + targets, 0x7FFFFFF0), 16);
  }
  H.n_lazy = runs.n_lazy; H.n_runs = runs.n_runs;
  H.lazy_base = H.state_doubles;
  H.state_doubles += (3 * H.n_lazy + 15) / 16 * 16;
  H.n_syn_inst = H.n_syn;
  if (H.state_doubles >= (int64_t)0xFFFFFFF0u) { err = "state pool exceeds 2^32 doubles"; return ARB_E_INVALID; }
  // delays
  H.min_delay = std::numeric_limits<double>::infinity();
  H.max_delay = 0;
  for (int64_t k = 0; k < d.n_conn; ++k) { H.min_delay = std::min(H.min_delay, d.conn_delay[k]); H.max_delay = std::max(H.max_delay, d.conn_delay[k]); }
  if (!fill) { H.n_syn = n_syn_orig; return ARB_OK; }

  // pass 2: fill
  H.fast.assign(H.fast_bytes, 0);
  H.state.assign(H.state_doubles, 0.0);
  H.gen.assign(H.gen_doubles, 0.0);
  H.topo.assign(H.topo_bytes, 0);
  H.descs.resize(H.n_units);
  H.cell_rt_idx.resize(nc);
  H.cv_state_idx.resize(H.n_cv);
  H.syn_state_idx.resize(H.n_syn);
  H.hh_m_idx.resize(H.n_hh); H.hh_stride.resize(H.n_hh); H.hh_cv.resize(H.n_hh);
  for (const auto& K : classes)
    if (K.grouped) std::memcpy(H.topo.data() + K.topo_off, K.record.data(), K.record.size());
  parallel_for(H.n_groups, [&](int64_t g) {
    const GroupCounts& G = groups[g];
    const ClassInfo& K = classes[G.cls];
    const GroupDesc& D = H.gdescs[g];
    const uint32_t n = K.n_cv;
    const GConstOff co = gconst_offsets(n, G.n_hh_rows, G.n_syn_rows, G.n_cl_rows, H.syn_uniform);
    const GStateOff so = gstate_offsets(n, G.n_hh_rows, G.n_syn_rows);
    const GGenOff go = ggen_offsets(n, G.n_syn_rows);
    uint8_t* cb = H.fast.data() + D.const_off;
    double* st = H.state.data() + D.state_base;
    double* gen = H.gen.data() + D.gen_base;
    double* invd = (double*)(cb + co.invd);
    double* a = (double*)(cb + co.a);
    double* hh_gna = (double*)(cb + co.hh_gna); double* hh_gk = (double*)(cb + co.hh_gk); double* hh_gl = (double*)(cb + co.hh_gl);
    double* syn_e = (double*)(cb + co.syn_e);
    double* cl_t0 = (double*)(cb + co.cl_t0); double* cl_t1 = (double*)(cb + co.cl_t1); double* cl_amp = (double*)(cb + co.cl_amp);
    uint16_t* hh_slot = (uint16_t*)(cb + co.hh_slot); uint16_t* syn_slot = (uint16_t*)(cb + co.syn_slot);
    uint16_t* cl_slot = (uint16_t*)(cb + co.cl_slot); uint16_t* det_slot = (uint16_t*)(cb + co.det_slot);
    for (uint32_t e = 0; e < kG * G.n_hh_rows; ++e) hh_slot[e] = kNoSlot16;
    for (uint32_t e = 0; e < kG * G.n_syn_rows; ++e) syn_slot[e] = kNoSlot16;
    for (uint32_t e = 0; e < kG * G.n_cl_rows; ++e) cl_slot[e] = kNoSlot16;
    int64_t hh_pos = G.hh_base;
    struct Item { uint32_t slot; int64_t id; };
    std::vector<Item> items;
    auto by_slot = [](const Item& x, const Item& y) { return x.slot != y.slot ? x.slot < y.slot : x.id < y.id; };
    for (uint32_t lc = 0; lc < (uint32_t)kG; ++lc) {
      double* rt = st + so.rt + kRtDoubles * lc;
      rt[0] = std::numeric_limits<double>::infinity();
      rt[1] = 0.0;
      if (lc >= G.n_cell) {
        // padding lane: an isolated, inert "cell" (V stays where it is, no instances, detector unarmed)
        for (uint32_t s2 = 0; s2 < n; ++s2) {
          const uint32_t e = gpos(s2, lc);
          gen[go.C + e] = 1.0; st[so.v + e] = -65.0; invd[e] = 1.0; a[e] = 1.0;
        }
        det_slot[lc] = 0;
        rt[2] = 0.0;
        continue;
      }
      const int64_t orig = group_cells[G.cell_begin + lc];
      const int64_t a0 = d.cv_off[orig];
      const int32_t* par = d.cv_parent + a0;
      std::vector<double> S(n, 0.0);
      for (uint32_t i = 1; i < n; ++i) S[i] = 1.0 / d.cv_raxial[a0 + i];
      for (uint32_t i = 1; i < n; ++i) S[par[i]] += 1.0 / d.cv_raxial[a0 + i];   // ascending child order
      items.clear();
      for (uint32_t i = 0; i < n; ++i) {
        const uint32_t e = gpos(K.cv_slot[i], lc);
        const double area = d.cv_area[a0 + i];
        gen[go.C + e] = d.cv_cm[a0 + i] * area * 1e-5;                 // nF
        gen[go.S + e] = S[i];                                          // uS
        gen[go.sig + e] = i ? 1.0 / d.cv_raxial[a0 + i] : 0.0;         // uS
        const double Gp = d.pas_g ? d.pas_g[a0 + i] * area * 1e-2 : 0.0;  // uS
        gen[go.G + e] = Gp;
        gen[go.b + e] = d.pas_g ? Gp * d.pas_e[a0 + i] : 0.0;          // nA
        st[so.v + e] = d.cv_vinit ? d.cv_vinit[a0 + i] : -65.0;
        H.cv_state_idx[a0 + i] = (uint32_t)(D.state_base + so.v + e);
        if (d.hh_gnabar && (d.hh_gnabar[a0 + i] != 0.0 || d.hh_gkbar[a0 + i] != 0.0 || d.hh_gl[a0 + i] != 0.0)) items.push_back({K.cv_slot[i], (int64_t)i});
      }
      std::sort(items.begin(), items.end(), by_slot);
      for (uint32_t j = 0; j < items.size(); ++j) {
        const uint32_t e = j * kG + lc;
        const int64_t gi = a0 + items[j].id;
        const double sc = d.cv_area[gi] * 1e-2;
        hh_gna[e] = d.hh_gnabar[gi] * sc; hh_gk[e] = d.hh_gkbar[gi] * sc; hh_gl[e] = d.hh_gl[gi] * sc;
        hh_slot[e] = (uint16_t)items[j].slot;
        H.hh_m_idx[hh_pos] = (uint32_t)(D.state_base + so.m + e);
        H.hh_stride[hh_pos] = so.h - so.m;
        H.hh_cv[hh_pos] = (uint32_t)gi;
        ++hh_pos;
      }
      items.clear();
      if (d.syn_off)
        for (int64_t q = d.syn_off[orig]; q < d.syn_off[orig + 1]; ++q) items.push_back({K.cv_slot[d.syn_cv[q]], q});
      std::sort(items.begin(), items.end(), by_slot);
      for (uint32_t j = 0; j < items.size(); ++j) {
        const uint32_t e = j * kG + lc;
        syn_slot[e] = (uint16_t)items[j].slot;
        if (!H.syn_uniform) syn_e[e] = d.syn_e[items[j].id];
        gen[go.syn_tau + e] = d.syn_tau[items[j].id];
        H.syn_state_idx[items[j].id] = (uint32_t)(D.state_base + so.g + e);
      }
      items.clear();
      for (int64_t q = clamp_off[orig]; q < clamp_off[orig + 1]; ++q) items.push_back({K.cv_slot[d.clamp_cv[clamp_idx[q]]], clamp_idx[q]});
      std::sort(items.begin(), items.end(), by_slot);
      for (uint32_t j = 0; j < items.size(); ++j) {
        const uint32_t e = j * kG + lc;
        cl_slot[e] = (uint16_t)items[j].slot;
        cl_t0[e] = d.clamp_t0[items[j].id]; cl_t1[e] = d.clamp_t1[items[j].id]; cl_amp[e] = d.clamp_amp[items[j].id];
      }
      det_slot[lc] = (uint16_t)K.cv_slot[d.det_cv ? d.det_cv[orig] : 0];
      rt[2] = 1.0;                                                     // detector armed (reading R10)
      H.cell_rt_idx[G.cell_begin + lc] = (uint32_t)(D.state_base + so.rt + kRtDoubles * lc);
    }
    // padding rows of syn_tau must stay finite for exp(-delta / tau)
    for (uint32_t e = 0; e < kG * G.n_syn_rows; ++e) if (syn_slot[e] == kNoSlot16) gen[go.syn_tau + e] = 1.0;
  });
  for (int64_t u = 0; u < H.n_units; ++u) {
    if (topo_owner[u] == u) std::memcpy(H.topo.data() + H.units[u].topo_off, topo[u].data(), topo[u].size());
    UnitDesc& ud = H.descs[u];
    ud.fast_off = H.units[u].fast_off; ud.state_base = H.units[u].state_base;
    ud.fast_bytes = H.units[u].fast_bytes; ud.state_bytes = H.units[u].state_bytes;
    const bool is_forest = (H.units[u].flags & UNIT_FOREST) != 0;
    ud.topo_off16 = is_forest ? (uint32_t)(H.units[u].topo_off / 16) : 0u;
    ud.topo_bytes = is_forest ? H.units[u].topo_bytes : 0u;
  }
  std::vector<std::vector<uint8_t>>().swap(topo);
  parallel_for(H.n_units, [&](int64_t u) {
    UnitBuilder B{d, P, H, clamp_off, clamp_idx, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, {}, false};
    B.forest = u < H.n_forests;
    UnitCounts placed = H.units[u];
    if (B.forest) B.n_warp = placed.n_warp;
    B.run(unit_begin[u], unit_cells[u], nullptr, &placed, &H);
  });
  // point cells
  H.pc_kind.resize(H.n_pcells); H.pc_par.assign(6 * (size_t)H.n_pcells, 0.0); H.pc_cv.resize(H.n_pcells);
  H.pc_src_off.assign((size_t)H.n_pcells + 1, 0);
  {
    int64_t gpos = H.pc_state_base + kPcDoubles * H.n_pcells;
    for (int64_t i = 0; i < H.n_pcells; ++i) {
      const int64_t c = point_cells[i];
      const int64_t cv = d.cv_off[c];
      double* st = H.state.data() + H.pc_state_base + kPcDoubles * i;
      st[0] = d.cv_vinit ? d.cv_vinit[cv] : -65.0;
      st[1] = std::numeric_limits<double>::infinity(); st[2] = 0.0; st[3] = 1.0;
      st[4] = 0.0; st[5] = -std::numeric_limits<double>::infinity(); st[6] = 0.0;
      H.cv_state_idx[cv] = (uint32_t)(H.pc_state_base + kPcDoubles * i);
      H.cell_rt_idx[H.pc_first + i] = (uint32_t)(H.pc_state_base + kPcDoubles * i + 1);
      H.pc_kind[i] = d.cell_kind[c];
      H.pc_cv[i] = (uint32_t)cv;
      const double par[6] = {d.lif_tau_m[c], d.lif_v_th[c], d.lif_c_m[c], d.lif_e_l[c], d.lif_e_r[c], d.lif_t_ref[c]};
      std::memcpy(H.pc_par.data() + 6 * i, par, sizeof par);
      if (d.syn_off)
        for (int64_t q = d.syn_off[c]; q < d.syn_off[c + 1]; ++q) H.syn_state_idx[q] = (uint32_t)gpos++;
      const int64_t ns = d.cell_kind[c] == 2 ? d.src_off[c + 1] - d.src_off[c] : 0;
      H.pc_src_off[i + 1] = H.pc_src_off[i] + (uint32_t)ns;
      for (int64_t q = 0; q < ns; ++q) H.pc_src_time.push_back(d.src_time[d.src_off[c] + q]);
    }
  }
  // state index of every ORIGINAL synapse: its instance, or its lazy record when its cell keeps run sums
  if (H.n_lazy > 0) {
    std::vector<uint32_t> final_idx((size_t)n_syn_orig);
    H.lazy_run.resize(H.n_lazy);
    double* lz = H.state.data() + H.lazy_base;
    for (int64_t s = 0; s < n_syn_orig; ++s) {
      const uint32_t inst = H.syn_state_idx[runs.map[s]];
      if (runs.lid[s] < 0) { final_idx[s] = inst; continue; }
      const int64_t l = runs.lid[s];
      final_idx[s] = (uint32_t)(H.lazy_base + l);
      H.lazy_run[l] = inst;
      lz[l] = 0.0; lz[H.n_lazy + l] = 0.0; lz[2 * H.n_lazy + l] = d_in.syn_tau[s];   // g_j, time of last touch, tau
    }
    H.run_off.clear(); H.run_gidx.clear();
    for (int64_t l = 0; l < H.n_lazy; ++l)
      if (l == 0 || runs.run_of_lazy[l] != runs.run_of_lazy[l - 1]) { H.run_off.push_back((uint32_t)l); H.run_gidx.push_back(H.lazy_run[l]); }
    H.run_off.push_back((uint32_t)H.n_lazy);
    H.syn_state_idx.swap(final_idx);
  }
  H.n_syn = n_syn_orig;
  // connections grouped by caller's source cell, ascending k inside a group
  H.conn_off.assign(H.n_src + 1, 0);             // by GLOBAL source id when the model is a shard
  for (int64_t k = 0; k < d.n_conn; ++k) H.conn_off[d.conn_src[k] + 1]++;
  for (int64_t c = 0; c < H.n_src; ++c) H.conn_off[c + 1] += H.conn_off[c];
  H.conn_dst.resize(d.n_conn); H.conn_gidx.resize(d.n_conn); H.conn_delay.resize(d.n_conn); H.conn_w.resize(d.n_conn);
  {
    std::vector<uint32_t> cur(H.conn_off.begin(), H.conn_off.end() - 1);
    for (int64_t k = 0; k < d.n_conn; ++k) {
      uint32_t p = cur[d.conn_src[k]]++;
      H.conn_dst[p] = H.cell_internal[d.conn_dst[k]];
      H.conn_gidx[p] = H.syn_state_idx[d_in.syn_off[d.conn_dst[k]] + d.conn_syn[k]];
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
      H.ext_gidx[p] = H.syn_state_idx[d_in.syn_off[d.ext_cell[k]] + d.ext_syn[k]];
      H.ext_w[p] = d.ext_weight[k];
    }
  }
  return ARB_OK;
}

}  // namespace arbb
