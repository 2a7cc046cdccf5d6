// grid.hpp -- host-side mesh tables of the product path (a11 of SURVEY.md Sec. 8(a)).
// Built by grid_builder.cpp from the quadtree's internal nodes; consumed by lbm_api.cu.
#pragma once
#include <cstdint>
#include <vector>

#include "../../include/lbm.h"

namespace lbm {

struct Lattice {
  int Q = 0, W = 0;
  double cs2 = 0.0;
  int cx[LBM_QMAX], cy[LBM_QMAX], opp[LBM_QMAX];
  double w[LBM_QMAX];
};
// Table 4 in the canonical direction order of DESIGN.md Sec. 2; false if Q is not a known lattice.
bool make_lattice(int Q, Lattice* L);

struct HostLevel {
  int nx = 0, ny = 0;
  int64_t n = 0, n_inbox = 0, n_fine_ghost = 0;
  std::vector<int32_t> ix, iy, aux;
  std::vector<uint8_t> type;          // LBM_FLUID ... LBM_DIRICHLET
  std::vector<uint8_t> side;          // boundary cells: side whose kind they carry (0 elsewhere)
  std::vector<int32_t> nbr;           // direction-major: nbr[(i-1)*n + cell], i = 1..Q-1 (device layout)
  int64_t ng = 0;
  std::vector<int32_t> g_coarse, g_child;   // g_child: 4 per ghost
  std::vector<uint64_t> g_mask;
  double tau = 0.0;
  // regular bricks (compressed addressing of the CUDA path): aligned 8x8 tiles of FLUID cells whose
  // every link is reproduced by tile arithmetic.  brick_nb[9*b + k]: storage index of the first cell of the tile at
  // offset (k%3-1, k/3-1) (k = 4: the brick itself).  irr: the cells outside bricks, ascending.
  std::vector<double> sigma;          // sponge coefficient per stored cell (Eq. 11); empty when no cell of the level has one
  int64_t nbrick = 0;
  std::vector<int32_t> brick_nb;
  std::vector<int32_t> irr;
};

struct HostGrid {
  lbm_config cfg;
  Lattice lat;
  int depth = 0;
  std::vector<HostLevel> lv;
  // brick_tab[(i-1)*64 + m] = (k << 6) | off: the pull source of direction i of the cell at Z-position m of a brick
  // is cell `off` (Z-position) of the tile k of brick_nb.
  std::vector<uint16_t> brick_tab;
};

// Returns LBM_OK, LBM_EINVAL, LBM_EMESH or LBM_ENOMEM.
int build_grid(const lbm_config& cfg, const int64_t* split_off, const int32_t* split_xy,
               const int64_t* solid_off, const int32_t* solid_xy, HostGrid* out);

}  // namespace lbm
