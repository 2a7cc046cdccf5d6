// transfer.cpp -- host side of the re-mesh step: the plan that moves the state of one
// tree onto another.  "This involves iterating over all cells in the updated tree and checking if corresponding LB data
// exists at the same location in the previous tree.  If a match is found, populations are directly copied; otherwise,
// they are recomputed using conservative coalescence (for cell coarsening) or uniform explosion (for cell refinement)."
//
// Rule per stored cell (level l, position (x, y)) of the new tree, ghost and boundary cells included:
//   1. the old tree stores a cell at (l, x, y): copy;
//   2. else the nearest stored ancestor (l+k, x >> k, y >> k): uniform explosion, Eq. 5, 7 (its state, all directions);
//   3. else the mean over the children (l-1, 2x+a, 2y+b) that can be evaluated by this same rule restricted to
//      1. and 3. (coalescence, Eq. 4, 6, all directions; children inside solids do not exist): recursively, so a
//      cell is the area-weighted mean of the old leaves it covers;
//   a NEUMANN cell takes the plan of its source cell (it replicates that cell's complete update, S13).
// The result is a flat list of (old level, old index, weight) per new cell; the device kernel of lbm_api.cu sums it.
#include <algorithm>
#include <cstdint>
#include <new>
#include <utility>
#include <vector>

#include "grid.hpp"

namespace lbm {

namespace {

constexpr int OFF = 1 << 20;      // boundary layers have negative coordinates

inline uint64_t pos_key(int x, int y) { return ((uint64_t)(uint32_t)(y + OFF) << 32) | (uint32_t)(x + OFF); }

struct Lookup {
  std::vector<std::pair<uint64_t, int32_t>> v;
  void build(const HostLevel& L) {
    v.resize((size_t)L.n);
    for (int64_t c = 0; c < L.n; ++c) v[(size_t)c] = {pos_key(L.ix[c], L.iy[c]), (int32_t)c};
    std::sort(v.begin(), v.end());
  }
  int32_t find(int x, int y) const {
    const uint64_t k = pos_key(x, y);
    auto it = std::lower_bound(v.begin(), v.end(), std::make_pair(k, (int32_t)-1));
    return (it != v.end() && it->first == k) ? it->second : -1;
  }
};

struct Walker {
  const std::vector<Lookup>& look;
  int depth;
  // rule 1 + 3: appends the entries of (l, x, y) scaled by w; false if nothing of the old tree lies there
  bool down(int l, int x, int y, double w, std::vector<TransferEntry>& out) const {
    if (l <= depth) {
      const int32_t s = look[(size_t)l].find(x, y);
      if (s >= 0) { out.push_back({s, l, w}); return true; }
    }
    if (l == 0) return false;
    const size_t mark = out.size();
    int nf = 0;
    std::vector<TransferEntry> child[4];
    for (int k = 0; k < 4; ++k)
      if (down(l - 1, 2 * x + (k & 1), 2 * y + (k >> 1), 1.0, child[k])) ++nf;
    if (nf == 0) { out.resize(mark); return false; }
    for (int k = 0; k < 4; ++k)
      for (const TransferEntry& e : child[k]) out.push_back({e.index, e.level, w * e.weight / (double)nf});
    return true;
  }
};

}  // namespace

int build_transfer_plan(const HostGrid& src, const HostGrid& dst, TransferPlan* plan) try {
  if (src.lat.Q != dst.lat.Q) return LBM_EINVAL;
  if (((int64_t)src.cfg.nx_coarse << src.depth) != ((int64_t)dst.cfg.nx_coarse << dst.depth) ||
      ((int64_t)src.cfg.ny_coarse << src.depth) != ((int64_t)dst.cfg.ny_coarse << dst.depth))
    return LBM_EINVAL;
  std::vector<Lookup> look((size_t)src.depth + 1);
  for (int l = 0; l <= src.depth; ++l) look[(size_t)l].build(src.lv[(size_t)l]);
  const Walker wk{look, src.depth};
  plan->off.assign((size_t)dst.depth + 1, std::vector<int64_t>());
  plan->entry.assign((size_t)dst.depth + 1, std::vector<TransferEntry>());
  for (int l = 0; l <= dst.depth; ++l) {
    const HostLevel& L = dst.lv[(size_t)l];
    std::vector<int64_t>& off = plan->off[(size_t)l];
    std::vector<TransferEntry>& ent = plan->entry[(size_t)l];
    off.assign((size_t)L.n + 1, 0);
    for (int64_t c = 0; c < L.n; ++c) {
      // a Neumann cell follows its source cell (an in-box cell, stored before it: its plan is complete already)
      if (L.type[c] == LBM_NEUMANN) {
        const int64_t s = L.aux[c];
        if (s < 0 || s >= c) return LBM_EMESH;
        for (int64_t k = off[(size_t)s]; k < off[(size_t)s + 1]; ++k) { const TransferEntry e = ent[(size_t)k]; ent.push_back(e); }
        off[(size_t)c + 1] = (int64_t)ent.size();
        continue;
      }
      const int x = L.ix[c], y = L.iy[c];
      bool found = false;
      if (l <= src.depth) {
        const int32_t s = look[(size_t)l].find(x, y);
        if (s >= 0) { ent.push_back({s, l, 1.0}); found = true; }
      }
      for (int k = 1; !found && l + k <= src.depth; ++k) {          // rule 2: nearest stored ancestor (floor division)
        const int32_t s = look[(size_t)(l + k)].find(x >> k, y >> k);
        if (s >= 0) { ent.push_back({s, l + k, 1.0}); found = true; }
      }
      if (!found) found = wk.down(l, x, y, 1.0, ent);               // rule 3
      if (!found) return LBM_EMESH;                                  // the old tree has no data there (geometry changed)
      off[(size_t)c + 1] = (int64_t)ent.size();
    }
  }
  return LBM_OK;
} catch (const std::bad_alloc&) {
  return LBM_ENOMEM;
}

}  // namespace lbm
