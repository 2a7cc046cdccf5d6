// grid_builder.cpp -- host grid builder of the product path.
//
// Emits, per level, the Morton-ordered cell tables, the int32 neighbour list (direction-major, the
// layout the sweep kernel reads), the ghost lists of every interface and the cell types
// (paper Sec. 4.3-4.4, Sec. 3.2; concrete rules: DESIGN.md Sec. 5-6).
//
// Technique: every level keeps dense bitmaps over the Z-curve of its bounding power-of-two square,
// one 64-bit word per 8x8-cell tile.  Because the storage order of in-box cells IS the Z-curve
// (x in the even bits), the storage index of a cell is
//     base[tile] + popcount(mask[tile] & bits_below(cell)),
// so membership tests and neighbour searches are two loads and a popcount, with no sort and no tree
// walk.  Loops over cells run on all host cores.
#include "grid.hpp"

#include <algorithm>
#include <cmath>
#include <atomic>
#include <cstring>
#include <new>
#include <thread>

namespace lbm {

// ------------------------------------------------------------------ lattices (Table 4)
bool make_lattice(int Q, Lattice* L) {
  struct Group { int a, b; double w; };
  static const Group g9[] = {{0, 0, 4.0 / 9.0}, {1, 0, 1.0 / 9.0}, {1, 1, 1.0 / 36.0}};
  static const Group g13[] = {{0, 0, 3.0 / 8.0}, {1, 0, 1.0 / 12.0}, {1, 1, 1.0 / 16.0}, {2, 0, 1.0 / 96.0}};
  static const Group g21[] = {{0, 0, 91.0 / 324.0}, {1, 0, 1.0 / 12.0}, {1, 1, 2.0 / 27.0}, {2, 0, 7.0 / 360.0},
                              {2, 2, 1.0 / 432.0}, {3, 0, 1.0 / 1620.0}};
  static const Group g37[] = {{0, 0, 0.233150669132352}, {1, 0, 0.107306091542219}, {1, 1, 0.057667859888794},
                              {2, 0, 0.014208216158450}, {2, 1, 0.005353049000513}, {2, 2, 0.001011937592673},
                              {3, 0, 0.000245301027757}, {3, 1, 0.000283414252994}};
  const Group* groups = nullptr;
  int ngroups = 0;
  switch (Q) {
    case 9: groups = g9; ngroups = 3; L->cs2 = 1.0 / 3.0; break;
    case 13: groups = g13; ngroups = 4; L->cs2 = 0.5; break;
    case 21: groups = g21; ngroups = 6; L->cs2 = 2.0 / 3.0; break;
    case 37: groups = g37; ngroups = 8; L->cs2 = 0.697953322019683; break;
    default: return false;
  }
  int n = 0, reach = 0;
  auto put = [&](int x, int y, double w) { L->cx[n] = x; L->cy[n] = y; L->w[n] = w; ++n; };
  for (int gi = 0; gi < ngroups; ++gi) {
    const Group& g = groups[gi];
    const int a = g.a, b = g.b;
    reach = std::max(reach, std::max(a, b));
    if (a == 0) {
      put(0, 0, g.w);
    } else if (b == 0) {                      // (a,0): counter-clockwise from +x
      put(a, 0, g.w); put(0, a, g.w); put(-a, 0, g.w); put(0, -a, g.w);
    } else if (a == b) {                      // (a,a)
      put(a, a, g.w); put(-a, a, g.w); put(-a, -a, g.w); put(a, -a, g.w);
    } else {                                  // (a,b), a > b > 0
      put(a, b, g.w); put(b, a, g.w); put(-b, a, g.w); put(-a, b, g.w);
      put(-a, -b, g.w); put(-b, -a, g.w); put(b, -a, g.w); put(a, -b, g.w);
    }
  }
  L->Q = n; L->W = reach;
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j)
      if (L->cx[j] == -L->cx[i] && L->cy[j] == -L->cy[i]) L->opp[i] = j;
  return n == Q;
}

namespace {

// ------------------------------------------------------------------ Z-curve helpers
inline uint64_t spread_bits(uint32_t v) {
  uint64_t x = v;
  x = (x | (x << 16)) & 0x0000FFFF0000FFFFull;
  x = (x | (x << 8)) & 0x00FF00FF00FF00FFull;
  x = (x | (x << 4)) & 0x0F0F0F0F0F0F0F0Full;
  x = (x | (x << 2)) & 0x3333333333333333ull;
  x = (x | (x << 1)) & 0x5555555555555555ull;
  return x;
}
inline uint32_t gather_bits(uint64_t x) {
  x &= 0x5555555555555555ull;
  x = (x | (x >> 1)) & 0x3333333333333333ull;
  x = (x | (x >> 2)) & 0x0F0F0F0F0F0F0F0Full;
  x = (x | (x >> 4)) & 0x00FF00FF00FF00FFull;
  x = (x | (x >> 8)) & 0x0000FFFF0000FFFFull;
  x = (x | (x >> 16)) & 0x00000000FFFFFFFFull;
  return (uint32_t)x;
}
inline uint64_t zkey(int ix, int iy) { return spread_bits((uint32_t)ix) | (spread_bits((uint32_t)iy) << 1); }

template <class F>
void parallel_for(int64_t n, F&& body) {
  unsigned nt = std::thread::hardware_concurrency();
  if (nt == 0) nt = 1;
  if (nt > 32) nt = 32;
  if (n < 1 << 15 || nt == 1) { body((int64_t)0, n); return; }
  std::vector<std::thread> th;
  const int64_t chunk = (n + nt - 1) / nt;
  for (unsigned t = 0; t < nt; ++t) {
    const int64_t lo = (int64_t)t * chunk, hi = std::min(n, lo + chunk);
    if (lo >= hi) break;
    th.emplace_back([&body, lo, hi]() { body(lo, hi); });
  }
  for (auto& t : th) t.join();
}

// Bitmap over the Z-curve of a (2^bits)^2 square; one word per 8x8 tile.
struct ZBitmap {
  std::vector<uint64_t> word;
  void init(int bits) { word.assign((size_t)1 << (2 * bits - 6), 0ull); }
  bool empty() const { return word.empty(); }
  void set(uint64_t key) { word[key >> 6] |= 1ull << (key & 63); }
  void clear(uint64_t key) { word[key >> 6] &= ~(1ull << (key & 63)); }
  bool test(uint64_t key) const { return (word[key >> 6] >> (key & 63)) & 1ull; }
};

// Bitmap + exclusive prefix counts = the directory (ix,iy) -> storage index.
struct ZDirectory {
  ZBitmap bm;
  std::vector<int32_t> base;
  int64_t count = 0;
  void finish() {
    base.resize(bm.word.size());
    int64_t run = 0;
    for (size_t t = 0; t < bm.word.size(); ++t) { base[t] = (int32_t)run; run += __builtin_popcountll(bm.word[t]); }
    count = run;
  }
  int32_t find(uint64_t key) const {
    const uint64_t w = bm.word[key >> 6], b = key & 63;
    if (!((w >> b) & 1ull)) return -1;
    return base[key >> 6] + __builtin_popcountll(w & ((1ull << b) - 1ull));
  }
};

inline bool boundary_cell_kind(int kind) {
  return kind == LBM_BC_DIRICHLET_EQ || kind == LBM_BC_DIRICHLET_EQ_RHO_EXTRAP || kind == LBM_BC_NEUMANN;
}

struct BuildLevel {
  int nx = 0, ny = 0, bits = 3;
  ZBitmap split, solid;
  ZDirectory cells;                       // in-box stored cells
  bool in_box(int x, int y) const { return x >= 0 && y >= 0 && x < nx && y < ny; }
};

// periodic wrap of one coordinate; false if it stays outside
inline bool wrap(int& t, int n, bool periodic) {
  if (t >= 0 && t < n) return true;
  if (!periodic) return false;
  t %= n;
  if (t < 0) t += n;
  return true;
}

}  // namespace

int build_grid(const lbm_config& cfg, const int64_t* split_off, const int32_t* split_xy,
               const int64_t* solid_off, const int32_t* solid_xy, HostGrid* out) try {
  HostGrid& G = *out;
  G.cfg = cfg;
  if (!make_lattice(cfg.lattice, &G.lat)) return LBM_EINVAL;
  const Lattice& lat = G.lat;
  const int d = cfg.depth, Q = lat.Q, W = lat.W;
  if (d < 0 || d > 20 || d >= LBM_MAX_LEVELS || cfg.nx_coarse < 1 || cfg.ny_coarse < 1) return LBM_EINVAL;
  for (int s = 0; s < 4; ++s)
    if (cfg.bc[s] < LBM_BC_PERIODIC || cfg.bc[s] > LBM_BC_NEUMANN) return LBM_EINVAL;
  const bool perx = cfg.bc[0] == LBM_BC_PERIODIC, pery = cfg.bc[2] == LBM_BC_PERIODIC;
  if (perx != (cfg.bc[1] == LBM_BC_PERIODIC) || pery != (cfg.bc[3] == LBM_BC_PERIODIC)) return LBM_EINVAL;
  if (((int64_t)cfg.nx_coarse << d) > (1 << 24) || ((int64_t)cfg.ny_coarse << d) > (1 << 24)) return LBM_EINVAL;
  G.depth = d;
  G.lv.assign((size_t)d + 1, HostLevel());
  std::vector<BuildLevel> B((size_t)d + 1);
  std::atomic<int> err{LBM_OK};

  // ---- split / solid bitmaps; a split cell must lie in the box and have a split parent
  for (int l = d; l >= 0; --l) {
    BuildLevel& b = B[l];
    b.nx = cfg.nx_coarse << (d - l);
    b.ny = cfg.ny_coarse << (d - l);
    if (l == d) {
      while ((1 << b.bits) < std::max(b.nx, b.ny)) ++b.bits;
      if (b.bits + d > 16) return LBM_EINVAL;              // bitmaps are dense over the bounding square
    } else {
      b.bits = B[l + 1].bits + 1;                          // children of key k are keys 4k..4k+3
    }
    const int64_t ns = split_off ? split_off[l + 1] - split_off[l] : 0;
    const int64_t nz = solid_off ? solid_off[l + 1] - solid_off[l] : 0;
    if (ns < 0 || nz < 0) return LBM_EINVAL;
    if (l == 0 && ns != 0) return LBM_EMESH;
    b.split.init(b.bits);
    b.solid.init(b.bits);
    for (int64_t k = 0; k < ns; ++k) {
      const int x = split_xy[2 * (split_off[l] + k)], y = split_xy[2 * (split_off[l] + k) + 1];
      if (!b.in_box(x, y)) return LBM_EMESH;
      if (l < d && !B[l + 1].split.test(zkey(x >> 1, y >> 1))) return LBM_EMESH;
      b.split.set(zkey(x, y));
    }
    for (int64_t k = 0; k < nz; ++k) {
      const int x = solid_xy[2 * (solid_off[l] + k)], y = solid_xy[2 * (solid_off[l] + k) + 1];
      if (b.in_box(x, y)) b.solid.set(zkey(x, y));      // positions outside the box are never looked up
    }
  }

  // ---- top-down: leaves, fine ghosts, coarse-ghost band
  for (int l = d; l >= 0; --l) {
    BuildLevel& b = B[l];
    HostLevel& L = G.lv[l];
    L.nx = b.nx; L.ny = b.ny;
    b.cells.bm.init(b.bits);
    ZBitmap& bm = b.cells.bm;
    // (1) leaves: cells that exist on this level and are neither split nor solid
    if (l == d) {
      for (int y = 0; y < b.ny; ++y)
        for (int x = 0; x < b.nx; ++x) bm.set(zkey(x, y));
    } else {
      // the four children of a split parent are the four consecutive keys 4k..4k+3
      const ZBitmap& ps = B[l + 1].split;
      parallel_for((int64_t)ps.word.size(), [&](int64_t lo, int64_t hi) {
        for (int64_t t = lo; t < hi; ++t) {
          uint64_t w = ps.word[t];
          while (w) {
            const int bit = __builtin_ctzll(w);
            w &= w - 1;
            const uint64_t ck = (((uint64_t)t << 6) | (uint64_t)bit) << 2;   // 4 children share one word
            bm.word[ck >> 6] |= 0xFull << (ck & 63);
          }
        }
      });
    }
    parallel_for((int64_t)bm.word.size(), [&](int64_t lo, int64_t hi) {
      for (int64_t t = lo; t < hi; ++t) bm.word[t] &= ~(b.split.word[t] | b.solid.word[t]);
    });
    // (3) fine ghosts = children of the coarse ghosts of level l+1, solid children not created
    std::vector<uint64_t> fg_keys;
    if (l < d) {
      const HostLevel& C = G.lv[l + 1];
      for (int64_t t = 0; t < C.n_inbox; ++t) {
        if (C.type[t] != LBM_COARSE_GHOST) continue;
        for (int ch = 0; ch < 4; ++ch) {
          const uint64_t k = zkey(2 * C.ix[t] + (ch & 1), 2 * C.iy[t] + (ch >> 1));
          if (b.solid.test(k)) continue;
          if (bm.test(k)) return LBM_EMESH;
          bm.set(k);
          fg_keys.push_back(k);
        }
      }
    }
    b.cells.finish();
    if (b.cells.count >= (int64_t)0x7FFFFFF0) return LBM_EINVAL;   // int32 storage indices
    const int64_t n_in = b.cells.count;
    L.n_inbox = n_in;
    L.n_fine_ghost = (int64_t)fg_keys.size();
    L.type.assign((size_t)n_in, (uint8_t)LBM_FLUID);
    L.ix.resize((size_t)n_in);
    L.iy.resize((size_t)n_in);
    for (uint64_t k : fg_keys) L.type[b.cells.find(k)] = LBM_FINE_GHOST;
    // coordinates in storage order: decode the set bits of every tile
    parallel_for((int64_t)bm.word.size(), [&](int64_t lo, int64_t hi) {
      for (int64_t t = lo; t < hi; ++t) {
        uint64_t w = bm.word[t];
        int32_t r = b.cells.base[t];
        while (w) {
          const uint64_t key = ((uint64_t)t << 6) | (uint64_t)__builtin_ctzll(w);
          w &= w - 1;
          L.ix[r] = (int32_t)gather_bits(key);
          L.iy[r] = (int32_t)gather_bits(key >> 1);
          ++r;
        }
      }
    });
    // (2) coarse-ghost band: stored cells within Chebyshev distance W of a split cell (reading S4)
    if (l >= 1) {
      uint8_t* type = L.type.data();
      parallel_for((int64_t)b.split.word.size(), [&](int64_t lo, int64_t hi) {
        for (int64_t t = lo; t < hi; ++t) {
          uint64_t w = b.split.word[t];
          while (w) {
            const uint64_t key = ((uint64_t)t << 6) | (uint64_t)__builtin_ctzll(w);
            w &= w - 1;
            const int sx = (int)gather_bits(key), sy = (int)gather_bits(key >> 1);
            for (int dy = -W; dy <= W; ++dy)
              for (int dx = -W; dx <= W; ++dx) {
                int tx = sx + dx, ty = sy + dy;
                if (!wrap(tx, b.nx, perx) || !wrap(ty, b.ny, pery)) continue;
                const int32_t c = b.cells.find(zkey(tx, ty));
                if (c < 0) continue;
                const uint8_t cur = __atomic_load_n(&type[c], __ATOMIC_RELAXED);
                if (cur == LBM_FINE_GHOST) { err.store(LBM_EMESH); continue; }   // interfaces too close
                if (cur != LBM_COARSE_GHOST) __atomic_store_n(&type[c], (uint8_t)LBM_COARSE_GHOST, __ATOMIC_RELAXED);
              }
          }
        }
      });
      if (err.load()) return err.load();
    }
  }

  // ---- boundary cells, neighbour lists
  for (int l = d; l >= 0; --l) {
    BuildLevel& b = B[l];
    HostLevel& L = G.lv[l];
    const int64_t n_in = L.n_inbox;
    // (5) W layers of boundary cells outside DIRICHLET / NEUMANN sides, generated by (iy, ix)
    bool anyb = false;
    for (int s = 0; s < 4; ++s) anyb = anyb || boundary_cell_kind(cfg.bc[s]);
    const int64_t bw = (int64_t)b.nx + 2 * W;          // boundary cells are looked up by (iy+W)*bw + ix+W
    std::vector<int64_t> bkey;
    if (anyb) {
      auto visit = [&](int x, int y) -> int {
        const int ox = x < 0 ? 0 : (x >= b.nx ? 1 : -1);
        const int oy = y < 0 ? 2 : (y >= b.ny ? 3 : -1);
        if (ox >= 0 && !boundary_cell_kind(cfg.bc[ox])) return LBM_OK;
        if (oy >= 0 && !boundary_cell_kind(cfg.bc[oy])) return LBM_OK;
        const int sx = std::min(std::max(x, 0), b.nx - 1), sy = std::min(std::max(y, 0), b.ny - 1);
        const int32_t s = b.cells.find(zkey(sx, sy));
        if (s < 0) return LBM_OK;                       // source not stored on this level
        if (L.type[s] != LBM_FLUID) return LBM_EMESH;   // an interface touches the boundary
        const int sd = oy >= 0 ? oy : ox;
        L.ix.push_back(x); L.iy.push_back(y);
        L.type.push_back(cfg.bc[sd] == LBM_BC_NEUMANN ? LBM_NEUMANN : LBM_DIRICHLET);
        bkey.push_back((int64_t)(y + W) * bw + (x + W));
        return LBM_OK;
      };
      for (int y = -W; y < b.ny + W; ++y) {
        if (y >= 0 && y < b.ny) {
          for (int x = -W; x < 0; ++x) { int rc = visit(x, y); if (rc) return rc; }
          for (int x = b.nx; x < b.nx + W; ++x) { int rc = visit(x, y); if (rc) return rc; }
        } else {
          for (int x = -W; x < b.nx + W; ++x) { int rc = visit(x, y); if (rc) return rc; }
        }
      }
    }
    L.n = (int64_t)L.ix.size();
    if (L.n >= (int64_t)0x7FFFFFF0) return LBM_EINVAL;
    const int64_t n = L.n;
    L.aux.assign((size_t)n, -1);
    L.side.assign((size_t)n, 0);
    L.nbr.assign((size_t)(n * (Q - 1)), LBM_LINK_NONE);
    auto find_boundary = [&](int x, int y) -> int32_t {
      const int64_t k = (int64_t)(y + W) * bw + (x + W);
      auto it = std::lower_bound(bkey.begin(), bkey.end(), k);
      if (it == bkey.end() || *it != k) return -1;
      return (int32_t)(n_in + (it - bkey.begin()));
    };
    // (7) row of an in-box cell: pull source of direction i is the cell at x - xi_i (Eq. 31)
    parallel_for(n_in, [&](int64_t lo, int64_t hi) {
      for (int64_t c = lo; c < hi; ++c) {
        const int type = L.type[c];
        for (int i = 1; i < Q; ++i) {
          int tx = L.ix[c] - lat.cx[i], ty = L.iy[c] - lat.cy[i];
          const bool inx = wrap(tx, b.nx, perx), iny = wrap(ty, b.ny, pery);
          int32_t link = LBM_LINK_NONE;
          if (inx && iny) {
            const uint64_t k = zkey(tx, ty);
            const int32_t s = b.cells.find(k);
            if (s >= 0) link = s;
            else if (b.solid.test(k)) link = LBM_LINK_WALL;          // bounce-back on solids
            else {
              if (type == LBM_FLUID) err.store(LBM_EMESH);           // no ghost band between two levels
              if (type == LBM_COARSE_GHOST && !b.split.test(k)) err.store(LBM_EMESH);
            }
          } else {
            const int ox = inx ? -1 : (tx < 0 ? 0 : 1);
            const int oy = iny ? -1 : (ty < 0 ? 2 : 3);
            const int sides[2] = {oy >= 0 ? oy : ox, (oy >= 0 && ox >= 0) ? ox : -1};
            for (int p = 0; p < 2 && sides[p] >= 0; ++p) {
              const int kind = cfg.bc[sides[p]];
              if (kind == LBM_BC_WALL) { link = LBM_LINK_WALL; break; }
              if (kind == LBM_BC_MOVING_WALL || kind == LBM_BC_INFLOW_VBB) { link = LBM_LINK_VBB0 - sides[p]; break; }
              if (boundary_cell_kind(kind)) {
                const int32_t s = find_boundary(tx, ty);
                if (s >= 0) { link = s; break; }
              }
            }
            if (link == LBM_LINK_NONE && type != LBM_FINE_GHOST) err.store(LBM_EMESH);
          }
          L.nbr[(size_t)(i - 1) * n + c] = link;
        }
      }
    });
    if (err.load()) return err.load();
    // boundary cells: a NEUMANN cell replicates its source's row (reading S13); a DIRICHLET cell has no links
    for (int64_t c = n_in; c < n; ++c) {
      const int x = L.ix[c], y = L.iy[c];
      const int sx = std::min(std::max(x, 0), b.nx - 1), sy = std::min(std::max(y, 0), b.ny - 1);
      const int32_t s = b.cells.find(zkey(sx, sy));
      L.aux[c] = s;
      const int ox = x < 0 ? 0 : (x >= b.nx ? 1 : -1);
      const int oy = y < 0 ? 2 : (y >= b.ny ? 3 : -1);
      L.side[c] = (uint8_t)(oy >= 0 ? oy : ox);
      if (L.type[c] == LBM_NEUMANN)
        for (int i = 1; i < Q; ++i) L.nbr[(size_t)(i - 1) * n + c] = L.nbr[(size_t)(i - 1) * n + s];
    }
  }

  // ---- (8) ghost lists, in storage order of the coarse level
  for (int l = 1; l <= d; ++l) {
    HostLevel& L = G.lv[l];
    const BuildLevel& f = B[l - 1];
    for (int64_t c = 0; c < L.n_inbox; ++c) {
      if (L.type[c] != LBM_COARSE_GHOST) continue;
      L.aux[c] = (int32_t)L.g_coarse.size();
      L.g_coarse.push_back((int32_t)c);
      int nchild = 0;
      for (int ch = 0; ch < 4; ++ch) {
        const int32_t s = f.cells.find(zkey(2 * L.ix[c] + (ch & 1), 2 * L.iy[c] + (ch >> 1)));
        L.g_child.push_back(s);
        nchild += s >= 0;
      }
      uint64_t m = 0;
      for (int i = 1; i < Q; ++i)
        if (L.nbr[(size_t)(i - 1) * L.n + c] == LBM_LINK_NONE) m |= 1ull << i;
      L.g_mask.push_back(m);
      if (m && nchild == 0) return LBM_EMESH;
    }
    L.ng = (int64_t)L.g_coarse.size();
  }
  // ---- sponge coefficient of Eq. 11 (reading S24) at the cell centres ((ix+1/2)h, (iy+1/2)h), h = 2^l
  if (cfg.sponge_sigma_max > 0.0)
    for (int l = 0; l <= d; ++l) {
      HostLevel& L = G.lv[l];
      const double h = (double)((int64_t)1 << l);
      std::vector<double> sg((size_t)L.n, 0.0);
      bool any = false;
      for (int64_t c = 0; c < L.n; ++c) {
        const double dx = (L.ix[c] + 0.5) * h - cfg.sponge_x0, dy = (L.iy[c] + 0.5) * h - cfg.sponge_y0;
        const double r = std::sqrt(dx * dx + dy * dy);
        double v = 0.0;
        if (r >= cfg.sponge_r1) v = cfg.sponge_sigma_max;
        else if (r >= cfg.sponge_r0) v = cfg.sponge_sigma_max * (r - cfg.sponge_r0) / (cfg.sponge_r1 - cfg.sponge_r0);
        sg[(size_t)c] = v;
        any = any || v > 0.0;
      }
      if (any) L.sigma.swap(sg);
    }

  // ---- (9) regular bricks: an aligned 8x8 tile whose 64 cells are stored (hence consecutive along the Z-curve), all
  // FLUID, and whose every list entry equals base[tile of the source] + Z-position of the
  // source inside that tile.  Each candidate is VERIFIED against the list built above, entry by entry, so the
  // compressed addressing can never disagree with the neighbour list it replaces on the device.
  G.brick_tab.assign((size_t)(Q - 1) * 64, 0);
  for (int i = 1; i < Q; ++i)
    for (int m = 0; m < 64; ++m) {
      const int x = (int)gather_bits((uint64_t)m), y = (int)gather_bits((uint64_t)m >> 1);
      const int sx = x - lat.cx[i], sy = y - lat.cy[i];
      const int kx = sx < 0 ? 0 : (sx > 7 ? 2 : 1), ky = sy < 0 ? 0 : (sy > 7 ? 2 : 1);
      G.brick_tab[(size_t)(i - 1) * 64 + m] = (uint16_t)(((kx + 3 * ky) << 6) | (int)zkey(sx & 7, sy & 7));
    }
  for (int l = 0; l <= d; ++l) {
    HostLevel& L = G.lv[l];
    const BuildLevel& b = B[l];
    const int64_t n = L.n;
    const size_t ntile = b.cells.bm.word.size();
    const int tnx = b.nx / 8, tny = b.ny / 8;            // whole tiles inside the box
    std::vector<int32_t> cand(ntile * 9, -1);
    std::vector<uint8_t> isbrick(ntile, 0);
    parallel_for((int64_t)ntile, [&](int64_t lo, int64_t hi) {
      for (int64_t t = lo; t < hi; ++t) {
        if (b.cells.bm.word[t] != ~0ull) continue;
        const int32_t base = b.cells.base[t];
        bool ok = true;
        for (int m = 0; m < 64 && ok; ++m)
          ok = L.type[(size_t)base + m] == LBM_FLUID && (L.sigma.empty() || L.sigma[(size_t)base + m] == 0.0);   // sponge cells use the list path
        if (!ok) continue;
        const int tx = (int)gather_bits((uint64_t)t), ty = (int)gather_bits((uint64_t)t >> 1);
        int32_t* nb = &cand[(size_t)t * 9];
        for (int k = 0; k < 9; ++k) {
          int ux = tx + k % 3 - 1, uy = ty + k / 3 - 1;
          if (ux < 0 || ux >= tnx) { if (!perx || b.nx % 8 != 0) continue; ux = (ux + tnx) % tnx; }
          if (uy < 0 || uy >= tny) { if (!pery || b.ny % 8 != 0) continue; uy = (uy + tny) % tny; }
          const uint64_t u = zkey(ux, uy);
          if (u < ntile && b.cells.bm.word[u] == ~0ull) nb[k] = b.cells.base[u];
        }
        for (int i = 1; i < Q && ok; ++i)
          for (int m = 0; m < 64; ++m) {
            const uint16_t e = G.brick_tab[(size_t)(i - 1) * 64 + m];
            const int32_t tb = nb[e >> 6];
            if (tb < 0 || L.nbr[(size_t)(i - 1) * n + base + m] != tb + (e & 63)) { ok = false; break; }
          }
        isbrick[t] = ok ? 1 : 0;
      }
    });
    std::vector<uint8_t> covered((size_t)n, 0);
    for (size_t t = 0; t < ntile; ++t) {
      if (!isbrick[t]) continue;
      L.brick_nb.insert(L.brick_nb.end(), &cand[t * 9], &cand[t * 9] + 9);
      std::fill(covered.begin() + b.cells.base[t], covered.begin() + b.cells.base[t] + 64, (uint8_t)1);
    }
    L.nbrick = (int64_t)(L.brick_nb.size() / 9);
    L.irr.reserve((size_t)(n - 64 * L.nbrick));
    for (int64_t c = 0; c < n; ++c)
      if (!covered[(size_t)c]) L.irr.push_back((int32_t)c);
  }

  // Eq. 3 (reading S3): tau_l - 1/2 = (tau_0 - 1/2) / 2^l
  for (int l = 0; l <= d; ++l) G.lv[l].tau = 0.5 + (cfg.tau0 - 0.5) / (double)((int64_t)1 << l);
  return LBM_OK;
} catch (const std::bad_alloc&) {
  return LBM_ENOMEM;
}

}  // namespace lbm
